"""ctypes binding of librosa.so — same names as include/rosa.h and include/rosa_debug.h, argument marshalling only.

PyTorch is used by callers for device memory and streams; this module only reads
``tensor.data_ptr()``.  Every step of the path runs inside the library's CUDA kernels.
There is no fallback: a missing library raises ImportError-like ``RosaError`` at load time.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "librosa.so")

ROSA_OK, ROSA_ERR_INVALID_ARG, ROSA_ERR_UNBOUND_ROBOT = 0, -1, -2
ROSA_ERR_CAPACITY, ROSA_ERR_CUDA, ROSA_ERR_UNSUPPORTED = -3, -4, -5
ROSA_F32, ROSA_BF16 = 0, 1

EXPORTS = ("rosa_expert_create", "rosa_expert_destroy", "rosa_prefix_kv_bind", "rosa_prefix_kv_unbind", "rosa_prefix_kv_produce",
           "rosa_denoise_batch", "rosa_denoise_batch_ex", "rosa_denoise_batch_host",
           "rosa_linear_noalloc", "rosa_last_error", "rosa_version")
ROSA_NOALLOC_MAX_ELEMS = 1 << 20
# include/rosa_debug.h: measurement and unit-test hooks
DEBUG_EXPORTS = ("rosa_profile_batch", "rosa_kernel_class_name", "rosa_last_launch_count", "rosa_kernel_family",
                 "rosa_debug_graph_captures", "rosa_debug_gemm", "rosa_debug_attn_plan")
ROSA_KC_COUNT = 11
EPI_STORE_F32, EPI_BIAS_F32, EPI_RESID = 0, 2, 4


class RosaError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"librosa status {status}: {msg}")
        self.status = status


class rosa_expert_config_t(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("layers", "d_model", "n_q_heads", "n_kv_heads", "head_dim", "ffn",
                                         "horizon", "action_dim", "max_robots", "max_batch",
                                         "max_prefix_len", "max_steps")] + \
               [(n, C.c_float) for n in ("rope_base", "rms_eps", "time_min_period", "time_max_period")] + \
               [("time_conditioning", C.c_int32)]


_GLOBAL = ("w_in", "b_in", "w_t1", "b_t1", "w_t2", "b_t2", "w_out", "b_out", "g_final")
_LAYER = ("g_attn", "wq", "wk", "wv", "wo", "g_mlp", "w_gate", "w_up", "w_down")
_LAYER_ADA = ("w_mod_attn", "b_mod_attn", "w_mod_mlp", "b_mod_mlp")      # time_conditioning == 1 only
_GLOBAL_ADA = ("w_mod_final", "b_mod_final")


class rosa_weights_t(C.Structure):
    _fields_ = [("dtype", C.c_int), ("on_device", C.c_int32)] + [(n, C.c_void_p) for n in _GLOBAL] + \
               [(n, C.POINTER(C.c_void_p)) for n in _LAYER] + [(n, C.POINTER(C.c_void_p)) for n in _LAYER_ADA] + \
               [(n, C.c_void_p) for n in _GLOBAL_ADA]


_lib = None


def load():
    """dlopen librosa.so (built in-tree by ``build.py``); loud failure if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RosaError(ROSA_ERR_CUDA, f"{LIB_PATH} not built: run `python -m paper_2607_01088_b200.build` "
                                       "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.rosa_expert_create.argtypes = [C.POINTER(rosa_expert_config_t), C.POINTER(rosa_weights_t), C.POINTER(vp)]
    lib.rosa_expert_destroy.argtypes = [vp]
    lib.rosa_prefix_kv_bind.argtypes = [vp, i32, C.POINTER(vp), C.POINTER(vp), i32, C.c_int]
    lib.rosa_prefix_kv_unbind.argtypes = [vp, i32]
    lib.rosa_prefix_kv_produce.argtypes = [vp, i32, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), i32, C.POINTER(vp), C.POINTER(vp), vp]
    lib.rosa_denoise_batch.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    lib.rosa_denoise_batch_ex.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.rosa_denoise_batch_host.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.rosa_last_launch_count.argtypes = [vp, C.POINTER(i64)]
    lib.rosa_kernel_family.argtypes = [vp, C.POINTER(i32)]
    lib.rosa_linear_noalloc.argtypes = [i32, i32, i32, i32, i32, vp, vp, vp, vp, vp]
    lib.rosa_debug_graph_captures.argtypes = [vp, C.POINTER(i64)]
    lib.rosa_debug_gemm.argtypes = [i32, i32, i32, i32, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.rosa_debug_attn_plan.argtypes = [i32, i32, vp, i32, vp, vp, i32]
    lib.rosa_debug_attn_plan.restype = i32
    lib.rosa_profile_batch.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.rosa_kernel_class_name.argtypes = [i32]
    lib.rosa_kernel_class_name.restype = C.c_char_p
    lib.rosa_last_error.restype = C.c_char_p
    lib.rosa_version.restype = i32
    for n in EXPORTS + DEBUG_EXPORTS:
        if n not in ("rosa_last_error", "rosa_version", "rosa_kernel_class_name", "rosa_debug_attn_plan"):
            getattr(lib, n).restype = C.c_int
    _lib = lib
    return lib


def _check(st: int):
    if st != ROSA_OK:
        raise RosaError(st, load().rosa_last_error().decode())


def _ptr(t) -> int:
    """Address of a torch tensor / numpy array / int (None -> NULL)."""
    if t is None:
        return 0
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _host(a, dtype) -> Optional[np.ndarray]:
    return None if a is None else np.ascontiguousarray(a, dtype=dtype)


def _stream_handle(stream) -> int:
    if stream is None:
        return 0
    return stream if isinstance(stream, int) else stream.cuda_stream


class Expert:
    """Opaque ``rosa_expert_t*`` plus the Python references that keep borrowed buffers alive."""

    def __init__(self, handle: int, cfg: rosa_expert_config_t):
        self.handle = handle
        self.cfg = cfg
        self._keep: Dict[int, tuple] = {}

    def __del__(self):
        try:
            if self.handle:
                rosa_expert_destroy(self)
        except Exception:
            pass


def rosa_expert_create(cfg: dict, weights: Dict[str, object], *, max_robots: int, max_batch: int,
                       max_prefix_len: int, max_steps: int = 16) -> Expert:
    """``cfg``: ExpertConfig fields; ``weights``: name -> float32 numpy array (or list per layer).
    Host float32 pointers are handed to the library, which converts and repacks them itself."""
    lib = load()
    c = rosa_expert_config_t()
    for k in ("layers", "d_model", "n_q_heads", "n_kv_heads", "head_dim", "ffn", "horizon", "action_dim"):
        setattr(c, k, int(cfg[k]))
    c.max_robots, c.max_batch, c.max_prefix_len, c.max_steps = max_robots, max_batch, max_prefix_len, max_steps
    c.rope_base, c.rms_eps = float(cfg["rope_base"]), float(cfg["rms_eps"])
    c.time_min_period, c.time_max_period = float(cfg["time_min_period"]), float(cfg["time_max_period"])
    c.time_conditioning = int(cfg.get("time_conditioning", 0))
    ada = c.time_conditioning == 1
    w = rosa_weights_t()
    w.dtype, w.on_device = ROSA_F32, 0
    keep = []
    for n in _GLOBAL + (_GLOBAL_ADA if ada else ()):
        a = np.ascontiguousarray(weights[n], dtype=np.float32)
        keep.append(a)
        setattr(w, n, a.ctypes.data)
    for n in _LAYER + (_LAYER_ADA if ada else ()):
        arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in weights[n]]
        keep.append(arrs)
        pa = (C.c_void_p * len(arrs))(*[a.ctypes.data for a in arrs])
        keep.append(pa)
        setattr(w, n, pa)
    out = C.c_void_p()
    _check(lib.rosa_expert_create(C.byref(c), C.byref(w), C.byref(out)))
    return Expert(out.value, c)


def rosa_expert_destroy(e: Expert):
    h, e.handle = e.handle, 0
    e._keep.clear()
    if h:
        _check(load().rosa_expert_destroy(h))


def rosa_prefix_kv_bind(e: Expert, robot: int, k_layers: Sequence, v_layers: Sequence, length: int,
                        dtype: int = ROSA_BF16):
    """k_layers/v_layers: per-layer device tensors (or raw device addresses) [len, n_kv, hd]."""
    n = e.cfg.layers
    ka = (C.c_void_p * n)(*[_ptr(t) for t in k_layers]) if length > 0 else None
    va = (C.c_void_p * n)(*[_ptr(t) for t in v_layers]) if length > 0 else None
    _check(load().rosa_prefix_kv_bind(e.handle, robot, ka, va, length, dtype))
    e._keep[robot] = (list(k_layers), list(v_layers))


def rosa_prefix_kv_produce(e: Expert, d_prefix: int, hidden_layers: Sequence, wk_layers: Sequence, wv_layers: Sequence,
                           length: int, k_out_layers: Sequence, v_out_layers: Sequence, stream=None):
    """Per-layer device tensors (or raw device addresses), all bf16: hidden [len, d_prefix], wk / wv [n_kv*hd, d_prefix],
    outputs [len, n_kv, hd]."""
    n = e.cfg.layers
    arr = lambda ts: (C.c_void_p * n)(*[_ptr(t) for t in ts])
    _check(load().rosa_prefix_kv_produce(e.handle, d_prefix, arr(hidden_layers), arr(wk_layers), arr(wv_layers), length,
                                         arr(k_out_layers), arr(v_out_layers), _stream_handle(stream)))


def rosa_prefix_kv_unbind(e: Expert, robot: int):
    _check(load().rosa_prefix_kv_unbind(e.handle, robot))
    e._keep.pop(robot, None)


def rosa_denoise_batch(e: Expert, robot_ids, noise, t_start, n_steps, out_actions, stream=None):
    ids = _host(robot_ids, np.int32)
    t0, ns = _host(t_start, np.float32), _host(n_steps, np.int32)
    _check(load().rosa_denoise_batch(e.handle, len(ids), _ptr(ids), _ptr(noise), _ptr(t0), _ptr(ns),
                                     _ptr(out_actions), _stream_handle(stream)))


def rosa_denoise_batch_ex(e: Expert, robot_ids, noise, t_start, dt, n_steps, out_actions,
                          out_velocity=None, stream=None):
    ids = _host(robot_ids, np.int32)
    t0, d, ns = _host(t_start, np.float32), _host(dt, np.float32), _host(n_steps, np.int32)
    _check(load().rosa_denoise_batch_ex(e.handle, len(ids), _ptr(ids), _ptr(noise), _ptr(t0), _ptr(d), _ptr(ns),
                                        _ptr(out_actions), _ptr(out_velocity), _stream_handle(stream)))


def rosa_denoise_batch_host(e: Expert, robot_ids, noise_host, t_start, dt, n_steps, out_actions_host, stream=None):
    """noise_host / out_actions_host: host float32 buffers (numpy arrays or pinned torch CPU tensors)."""
    ids = _host(robot_ids, np.int32)
    t0, d, ns = _host(t_start, np.float32), _host(dt, np.float32), _host(n_steps, np.int32)
    _check(load().rosa_denoise_batch_host(e.handle, len(ids), _ptr(ids), _ptr(noise_host), _ptr(t0), _ptr(d),
                                          _ptr(ns), _ptr(out_actions_host), _stream_handle(stream)))


def rosa_linear_noalloc(M: int, N: int, K: int, A16, W16, C_f32, *, epi: int = EPI_STORE_F32, fp16: int = 0, bias=None,
                        stream=None):
    """C = epi(A W^T) through the allocation-free entry point (static device scratch, M * N <= ROSA_NOALLOC_MAX_ELEMS)."""
    _check(load().rosa_linear_noalloc(epi, fp16, M, N, K, _ptr(A16), _ptr(W16), _ptr(bias), _ptr(C_f32), _stream_handle(stream)))


def rosa_profile_batch(e: Expert, robot_ids, noise, t_start, dt, n_steps, out_actions, stream=None):
    """Returns {kernel class name: (milliseconds, launches)} for one un-graphed, event-timed call."""
    ids = _host(robot_ids, np.int32)
    t0, d, ns = _host(t_start, np.float32), _host(dt, np.float32), _host(n_steps, np.int32)
    ms = np.zeros(ROSA_KC_COUNT, dtype=np.float32)
    nl = np.zeros(ROSA_KC_COUNT, dtype=np.int32)
    _check(load().rosa_profile_batch(e.handle, len(ids), _ptr(ids), _ptr(noise), _ptr(t0), _ptr(d), _ptr(ns),
                                     _ptr(out_actions), _stream_handle(stream), _ptr(ms), _ptr(nl)))
    return {rosa_kernel_class_name(c): (float(ms[c]), int(nl[c])) for c in range(ROSA_KC_COUNT)}


def rosa_kernel_class_name(cls: int) -> str:
    return load().rosa_kernel_class_name(cls).decode()


def rosa_last_launch_count(e: Expert) -> int:
    n = C.c_int64()
    _check(load().rosa_last_launch_count(e.handle, C.byref(n)))
    return n.value


def rosa_kernel_family(e: Expert) -> int:
    n = C.c_int32()
    _check(load().rosa_kernel_family(e.handle, C.byref(n)))
    return n.value


def rosa_debug_graph_captures(e: Expert) -> int:
    n = C.c_int64()
    _check(load().rosa_debug_graph_captures(e.handle, C.byref(n)))
    return n.value


def rosa_debug_gemm(family: int, M: int, N: int, K: int, A16, W16, C_f32, *, epi: int = EPI_STORE_F32, pair: int = -1,
                    bn: int = 0, fp16: int = 0, bias=None, h16=None, ssq=None, stream=None):
    _check(load().rosa_debug_gemm(family, epi, pair, bn, fp16, M, N, K, _ptr(A16), _ptr(W16), _ptr(C_f32), _ptr(bias),
                                  _ptr(h16), _ptr(ssq), _stream_handle(stream)))


def rosa_debug_attn_plan(horizon: int, lens, n_cta: int):
    """Host logic of the attention work split (no device): returns (offs [n_cta + 1], segs [n, 6] int32 with columns
    robot, tile, kb0, kb1, n_part, part0)."""
    ln = np.ascontiguousarray(lens, dtype=np.int32)
    cap = int(ln.shape[0]) * ((int(horizon) + 15) // 16) + 4 * int(n_cta)
    offs = np.zeros(n_cta + 1, dtype=np.int32)
    segs = np.zeros((cap, 8), dtype=np.int32)
    n = load().rosa_debug_attn_plan(int(horizon), int(ln.shape[0]), _ptr(ln), int(n_cta), _ptr(offs), _ptr(segs), cap)
    if n < 0:
        raise RosaError(n, rosa_last_error())
    return offs, segs[:n, :6].copy()


def rosa_last_error() -> str:
    return load().rosa_last_error().decode()


def rosa_version() -> int:
    return load().rosa_version()
