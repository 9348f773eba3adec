"""Seeded synthetic inputs for the batched action-expert denoise loop.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library (through the
tests and ``bench.py``).  It holds none of the method's arithmetic: it only draws random
tensors in a fixed, documented order and (for the bf16 configurations) rounds them to
bf16 so both sides see bit-identical operand values (reading R12/R13).

Workload recipe = BASELINE.json ``configs`` 0..4 (stand-ins for the paper's replayed
Franka observations through GR00T N1.6 / pi0.5, which are not public):
weights and biases N(0, 0.02), RMSNorm gains 1, prefix K/V and initial noise N(0, 1).

Draw order (one ``numpy.random.Generator(PCG64(seed))``, float32 ``standard_normal``):
  1. prefix lengths (integers, both bounds inclusive) when the config draws them
  2. global weights in struct order: w_in, w_t1, w_t2, w_out
  3. per layer l = 0..layers-1: wq, wk, wv, wo, w_gate, w_up, w_down
  4. biases: b_in, b_t1, b_t2, b_out
  5. per robot i: per layer l: K then V, each [L_i, n_kv, head_dim]
  6. noise [B, H, A]
  7. config 3 only: per-robot start-time index
Adaptive-norm variant (``time_conditioning=1``, reading R25): w_t1 is [d, d], and after
step 4 a third generator ``PCG64([seed, 0x5eed])`` draws, per layer, w_mod_attn, w_mod_mlp [3d, d], then
w_mod_final, then the biases b_mod_* [3d] in the same order, all N(0, 0.02), with +1 added to the gate
third of every b_mod so the blocks contribute (a zero-mean gate would switch them off).
"""
from __future__ import annotations

from dataclasses import dataclass, field, asdict
from typing import Dict, List, Optional

import numpy as np


@dataclass(frozen=True)
class ExpertConfig:
    layers: int
    d_model: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    ffn: int
    horizon: int
    action_dim: int
    rope_base: float = 10000.0
    rms_eps: float = 1e-6
    time_min_period: float = 4e-3
    time_max_period: float = 4.0
    time_conditioning: int = 0       # 0: time concatenated into the embedding MLP (pi0-style); 1: adaptive RMSNorm (pi0.5-style, R25)

    def as_dict(self) -> dict:
        return asdict(self)


TINY = ExpertConfig(layers=2, d_model=128, n_q_heads=4, n_kv_heads=1, head_dim=32,
                    ffn=512, horizon=8, action_dim=7)
PI0 = ExpertConfig(layers=18, d_model=1024, n_q_heads=8, n_kv_heads=1, head_dim=256,
                   ffn=4096, horizon=50, action_dim=32)

GLOBAL_WEIGHTS = ("w_in", "w_t1", "w_t2", "w_out")
LAYER_WEIGHTS = ("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down")
BIASES = ("b_in", "b_t1", "b_t2", "b_out")


def weight_shapes(c: ExpertConfig) -> Dict[str, tuple]:
    """[out_features, in_features] row-major for every matrix (reading R10)."""
    d, a, f = c.d_model, c.action_dim, c.ffn
    nq, nkv, hd = c.n_q_heads, c.n_kv_heads, c.head_dim
    ada = {"w_mod": (3 * d, d), "b_mod": (3 * d,)} if c.time_conditioning == 1 else {}   # per norm: 2 per layer + final
    return {
        **ada,
        "w_in": (d, a), "w_t1": (d, d if c.time_conditioning == 1 else 2 * d), "w_t2": (d, d), "w_out": (a, d),
        "wq": (nq * hd, d), "wk": (nkv * hd, d), "wv": (nkv * hd, d), "wo": (d, nq * hd),
        "w_gate": (f, d), "w_up": (f, d), "w_down": (d, f),
        "b_in": (d,), "b_t1": (d,), "b_t2": (d,), "b_out": (a,),
    }


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even float32 -> bf16 bit pattern (uint16). Input preparation only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    bias = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + bias) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def round_bf16(x: np.ndarray) -> np.ndarray:
    """float32 values that are exactly representable in bf16 (RNE)."""
    return bf16_bits_to_f32(f32_to_bf16_bits(x))


@dataclass
class Case:
    name: str
    seed: int
    cfg: ExpertConfig
    bf16: bool                       # True: every weight / prefix value is bf16-representable
    weights: Dict[str, object]       # name -> float32 array, or list of per-layer arrays
    prefix_lens: np.ndarray          # int32 [B]
    prefix_k: List[np.ndarray]       # per robot [layers, L_i, n_kv, head_dim]; uint16 bf16 bits if bf16 else float32
    prefix_v: List[np.ndarray]
    noise: np.ndarray                # float32 [B, H, A]
    t_start: np.ndarray              # float32 [B]
    dt: np.ndarray                   # float32 [B]
    n_steps: np.ndarray              # int32 [B]
    notes: dict = field(default_factory=dict)

    @property
    def batch(self) -> int:
        return int(self.prefix_lens.shape[0])

    def prefix_f32(self, i: int):
        """Prefix K, V of robot i as float32 [layers, L_i, n_kv, head_dim]."""
        if self.bf16:
            return bf16_bits_to_f32(self.prefix_k[i]), bf16_bits_to_f32(self.prefix_v[i])
        return self.prefix_k[i], self.prefix_v[i]

    def cu_seqlens(self) -> np.ndarray:
        out = np.zeros(self.batch + 1, dtype=np.int64)
        np.cumsum(self.prefix_lens, out=out[1:])
        return out

    def subset(self, idx) -> "Case":
        """The same case restricted to robots ``idx`` (robots are independent units)."""
        idx = list(idx)
        return Case(self.name + "-sub", self.seed, self.cfg, self.bf16, self.weights,
                    self.prefix_lens[idx].copy(), [self.prefix_k[i] for i in idx],
                    [self.prefix_v[i] for i in idx], self.noise[idx].copy(),
                    self.t_start[idx].copy(), self.dt[idx].copy(), self.n_steps[idx].copy(),
                    dict(self.notes))


def _normal(rng: np.random.Generator, shape, scale: float = 1.0) -> np.ndarray:
    x = rng.standard_normal(size=shape, dtype=np.float32)
    if scale != 1.0:
        x *= np.float32(scale)
    return x


def build_case(name: str, seed: int, cfg: ExpertConfig, *, bf16: bool,
               prefix_lens=None, draw_lens=None, batch: Optional[int] = None,
               n_steps: int = 10, cfg3_mix: bool = False, with_prefix: bool = True,
               robot_stream: int = 0) -> Case:
    """Draw one case in the documented order.  ``draw_lens=(lo, hi)`` draws B integer
    lengths uniformly with both bounds inclusive (reading R14).

    ``robot_stream`` != 0 (bench.py, ranks > 0 of a multi-GPU run: same replicated weights,
    different robots) draws everything per-robot (lengths, K/V, noise, start times) from a
    second generator ``PCG64([seed, robot_stream])`` instead of the main one."""
    rng = np.random.Generator(np.random.PCG64(seed))
    rrng = rng if robot_stream == 0 else np.random.Generator(np.random.PCG64([seed, robot_stream]))
    if draw_lens is not None:
        lo, hi = draw_lens
        lens = rng.integers(lo, hi, size=batch, endpoint=True).astype(np.int32)   # keeps the weight stream aligned
        if robot_stream != 0:
            lens = rrng.integers(lo, hi, size=batch, endpoint=True).astype(np.int32)
    else:
        lens = np.asarray(prefix_lens, dtype=np.int32)
    B = int(lens.shape[0])
    shp = weight_shapes(cfg)
    rnd = round_bf16 if bf16 else (lambda a: a)

    w: Dict[str, object] = {}
    for k in GLOBAL_WEIGHTS:
        w[k] = rnd(_normal(rng, shp[k], 0.02))
    for k in LAYER_WEIGHTS:
        w[k] = [None] * cfg.layers
    for l in range(cfg.layers):
        for k in LAYER_WEIGHTS:
            w[k][l] = rnd(_normal(rng, shp[k], 0.02))
    for k in BIASES:
        w[k] = rnd(_normal(rng, shp[k], 0.02))
    ones = np.ones(cfg.d_model, dtype=np.float32)
    w["g_final"] = ones.copy()
    w["g_attn"] = [ones.copy() for _ in range(cfg.layers)]
    w["g_mlp"] = [ones.copy() for _ in range(cfg.layers)]
    if cfg.time_conditioning == 1:
        mrng = np.random.Generator(np.random.PCG64([seed, 0x5eed]))
        w["w_mod_attn"], w["w_mod_mlp"] = [None] * cfg.layers, [None] * cfg.layers
        for l in range(cfg.layers):
            w["w_mod_attn"][l] = rnd(_normal(mrng, shp["w_mod"], 0.02))
            w["w_mod_mlp"][l] = rnd(_normal(mrng, shp["w_mod"], 0.02))
        w["w_mod_final"] = rnd(_normal(mrng, shp["w_mod"], 0.02))

        def mod_bias():
            b = _normal(mrng, shp["b_mod"], 0.02)
            b[2 * cfg.d_model:] += np.float32(1.0)
            return rnd(b)
        w["b_mod_attn"], w["b_mod_mlp"] = [None] * cfg.layers, [None] * cfg.layers
        for l in range(cfg.layers):
            w["b_mod_attn"][l] = mod_bias()
            w["b_mod_mlp"][l] = mod_bias()
        w["b_mod_final"] = mod_bias()

    pk, pv = [], []
    if with_prefix:
        for i in range(B):
            L = int(lens[i])
            k_i = np.empty((cfg.layers, L, cfg.n_kv_heads, cfg.head_dim),
                           dtype=np.uint16 if bf16 else np.float32)
            v_i = np.empty_like(k_i)
            for l in range(cfg.layers):
                kk = _normal(rrng, (L, cfg.n_kv_heads, cfg.head_dim))
                vv = _normal(rrng, (L, cfg.n_kv_heads, cfg.head_dim))
                k_i[l] = f32_to_bf16_bits(kk) if bf16 else kk
                v_i[l] = f32_to_bf16_bits(vv) if bf16 else vv
            pk.append(k_i)
            pv.append(v_i)
    noise = _normal(rrng, (B, cfg.horizon, cfg.action_dim))

    if cfg3_mix:
        # reading R15: t_i uniform over {1.0, 0.9, ..., 0.1}; remaining steps n_i = round(10 t_i); dt_i = -0.1
        m = rrng.integers(1, 10, size=B, endpoint=True).astype(np.int32)
        t0 = (m.astype(np.float32) / np.float32(10.0)).astype(np.float32)
        ns = m.copy()
        dt = np.full(B, -0.1, dtype=np.float32)
    else:
        t0 = np.ones(B, dtype=np.float32)
        ns = np.full(B, n_steps, dtype=np.int32)
        dt = (-t0 / ns.astype(np.float32)).astype(np.float32)
    return Case(name, seed, cfg, bf16, w, lens, pk, pv, noise, t0, dt, ns)


def make_case(config: int, *, batch: Optional[int] = None, with_prefix: bool = True,
              robot_stream: int = 0, time_conditioning: int = 0) -> Case:
    """BASELINE.json ``configs[config]``.  ``batch`` selects the B of the config-4 sweep.
    ``time_conditioning=1`` (configs 1-4): the same workload on the adaptive-norm variant of the expert (R25)."""
    kw = dict(with_prefix=with_prefix, robot_stream=robot_stream)
    if time_conditioning:
        from dataclasses import replace
        pi0 = replace(PI0, time_conditioning=1)
        spec = {1: dict(prefix_lens=[816] * 8), 2: dict(draw_lens=(600, 1000), batch=batch or 64),
                3: dict(draw_lens=(400, 1200), batch=batch or 256, cfg3_mix=True),
                4: dict(prefix_lens=[816] * (batch or 64))}[config]
        return build_case(f"cfg{config}-adarms", config, pi0, bf16=True, **spec, **kw)
    if config == 0:
        return build_case("cfg0-tiny", 0, TINY, bf16=False, prefix_lens=[48, 64], n_steps=4, **kw)
    if config == 1:
        return build_case("cfg1-pi0-b8", 1, PI0, bf16=True, prefix_lens=[816] * 8, **kw)
    if config == 2:
        return build_case("cfg2-fleet-b64", 2, PI0, bf16=True, draw_lens=(600, 1000),
                          batch=batch or 64, **kw)
    if config == 3:
        return build_case("cfg3-contbatch-b256", 3, PI0, bf16=True, draw_lens=(400, 1200),
                          batch=batch or 256, cfg3_mix=True, **kw)
    if config == 4:
        b = batch or 64
        return build_case(f"cfg4-sweep-b{b}", 4, PI0, bf16=True, prefix_lens=[816] * b, **kw)
    raise ValueError(f"unknown config {config}")


def make_adarms_case(scale: str = "tiny", *, batch: int = 2, layers: Optional[int] = None, seed: int = 5) -> Case:
    """Adaptive-norm variant (reading R25) on the tiny fp32 shapes or on pi0-scale bf16 shapes with fewer
    layers (the oracle's time grows with layers x batch; kernels are exercised from 2 layers on)."""
    from dataclasses import replace
    if scale == "tiny":
        cfg = replace(TINY, time_conditioning=1, layers=layers or TINY.layers)
        return build_case("adarms-tiny", seed, cfg, bf16=False, prefix_lens=[48, 64][:batch] if batch <= 2 else [48 + 5 * i for i in range(batch)], n_steps=4)
    cfg = replace(PI0, time_conditioning=1, layers=layers or 3)
    return build_case(f"adarms-pi0-l{cfg.layers}-b{batch}", seed, cfg, bf16=True, draw_lens=(300, 500), batch=batch, n_steps=4)


SWEEP_BATCHES = (1, 2, 4, 8, 16, 32, 64, 128, 256, 512)
