"""B200-native batched action-expert denoise loop (ROSA's inter-robot batched System-1 path).

``cases`` (seeded inputs) imports without the CUDA library; ``binding`` loads
``librosa.so`` and fails loudly if it is missing.  Nothing here imports ``oracle/``.
"""
__all__ = ["cases", "binding", "build"]
