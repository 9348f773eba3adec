"""CPU ORACLE for the batched action-expert denoise loop.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this file.  It shares no code with the CUDA library
(``paper_2607_01088_b200/csrc``) and never imports it; the product path never routes here.

What it computes: the paper (ROSA) batches System-1
action-model inference across robots but treats the model as a black box, so the model is
the pi0-style flow-matching action expert that BASELINE.json ``north_star``/``configs``
spell out, completed by readings R1..R19 of DESIGN.md (= SURVEY.md section 8(c)).  The
oracle follows that algorithm step by step in fp64 (numpy); ``numpy.matmul`` is the only
library primitive used.  No blocking, fusion or reordering beyond the definition.

Pins (tests/test_oracle_pins.py): brute-force fp64 attention loops, closed forms (constant
velocity, zero output projection, uniform attention, RoPE shift invariance, norm scale
invariance), step composition, batch/permutation invariance, and torch fp64 library
routines as an independent third opinion.  The adaptive-norm variant (reading R25) is pinned by
its reductions: zero modulation with unit gate equals the pinned blocks on the same normed input,
zero gate is the identity, a hand-written per-element loop, and torch fp64.  The numeric output
of a *trained* model is "parity unpinned": no trained weights or published tensors exist.
"""
from __future__ import annotations

import math
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

F = np.float64


# ----------------------------------------------------------------------------- pieces
def sinusoidal_time_embedding(t: np.ndarray, d: int, p_min: float, p_max: float, dtype=F) -> np.ndarray:
    """tau(t) in R^d for each robot (BASELINE.json cfg0 "sinusoidal(128)"; reading R3).

    period_j = p_min * (p_max/p_min)^(j/(d/2-1)), j < d/2;
    tau = [sin(2 pi t / period_j)]_j || [cos(2 pi t / period_j)]_j.
    """
    half = d // 2
    j = np.arange(half, dtype=dtype)
    frac = j / dtype(max(half - 1, 1))
    period = dtype(p_min) * (dtype(p_max) / dtype(p_min)) ** frac
    ang = (dtype(2.0) * dtype(math.pi)) * np.asarray(t, dtype=dtype)[:, None] / period[None, :]
    return np.concatenate([np.sin(ang), np.cos(ang)], axis=1)


def swish(z: np.ndarray) -> np.ndarray:
    """swish(z) = z / (1 + e^-z)  (BASELINE.json cfg0 "2-layer swish MLP")."""
    return z / (1.0 + np.exp(-z))


def gelu_tanh(z: np.ndarray) -> np.ndarray:
    """GeGLU gate activation, tanh form (reading R6): 0.5 z (1 + tanh(sqrt(2/pi)(z + 0.044715 z^3)))."""
    c = math.sqrt(2.0 / math.pi)
    return 0.5 * z * (1.0 + np.tanh(c * (z + 0.044715 * z * z * z)))


def rmsnorm(x: np.ndarray, g: np.ndarray, eps: float) -> np.ndarray:
    """y = x * rsqrt(mean(x^2) + eps) * g over the last axis (reading R5)."""
    ms = np.mean(x * x, axis=-1, keepdims=True)
    return x / np.sqrt(ms + eps) * g


def rope(x: np.ndarray, pos: np.ndarray, base: float) -> np.ndarray:
    """Rotary embedding, half-split pairs (reading R7).

    x: [T, heads, hd]; pos: [T].  theta_c = base^(-2c/hd), c < hd/2; phi = pos * theta_c;
    (x_c, x_{c+hd/2}) -> (x_c cos phi - x_{c+hd/2} sin phi, x_{c+hd/2} cos phi + x_c sin phi).
    """
    hd = x.shape[-1]
    half = hd // 2
    c = np.arange(half, dtype=x.dtype)
    theta = x.dtype.type(base) ** (-2.0 * c / hd)
    phi = np.asarray(pos, dtype=x.dtype)[:, None] * theta[None, :]        # [T, half]
    cos, sin = np.cos(phi)[:, None, :], np.sin(phi)[:, None, :]
    x1, x2 = x[..., :half], x[..., half:]
    return np.concatenate([x1 * cos - x2 * sin, x2 * cos + x1 * sin], axis=-1)


def attention_robot(q: np.ndarray, k_all: np.ndarray, v_all: np.ndarray) -> np.ndarray:
    """Grouped-query softmax attention of one robot, full visibility (readings R8, R9).

    q: [H, n_q, hd]; k_all, v_all: [L+H, n_kv, hd] = [prefix ; own action tokens].
    Query head a uses KV head a // (n_q / n_kv).  Scale 1/sqrt(hd); no mask.
    Returns o: [H, n_q, hd].
    """
    H, n_q, hd = q.shape
    n_kv = k_all.shape[1]
    group = n_q // n_kv
    o = np.empty_like(q)
    for a in range(n_q):
        g = a // group
        s = (q[:, a, :] @ k_all[:, g, :].T) / math.sqrt(hd)               # [H, L+H]
        s = s - np.max(s, axis=1, keepdims=True)
        p = np.exp(s)
        p = p / np.sum(p, axis=1, keepdims=True)
        o[:, a, :] = p @ v_all[:, g, :]
    return o


# ----------------------------------------------------------------------------- model
def _as(w, dtype):
    return np.asarray(w, dtype=dtype)


def embed(cfg, W: Dict, x: np.ndarray, t: np.ndarray, dtype=F) -> np.ndarray:
    """Steps 1-3 of the algorithm; x: [B, H, A], t: [B] -> h: [B, H, d].

    a = x W_in^T + b_in;  u = [tau(t) ; a] (reading R2: time half first);
    h = W_2 swish(W_1 u + b_1) + b_2.
    """
    B, H, _ = x.shape
    d = cfg.d_model
    a = x @ _as(W["w_in"], dtype).T + _as(W["b_in"], dtype)               # [B, H, d]
    tau = sinusoidal_time_embedding(t, d, cfg.time_min_period, cfg.time_max_period, dtype)
    u = np.concatenate([np.broadcast_to(tau[:, None, :], (B, H, d)), a], axis=2)  # [B, H, 2d]
    z = swish(u @ _as(W["w_t1"], dtype).T + _as(W["b_t1"], dtype))
    return z @ _as(W["w_t2"], dtype).T + _as(W["b_t2"], dtype)


def attention_sublayer(cfg, W: Dict, l: int, n1: np.ndarray, prefix_k: Sequence[np.ndarray],
                       prefix_v: Sequence[np.ndarray], dtype=F) -> np.ndarray:
    """Attention half of a block, from the normed input n1 [B, H, d] to the W_o output [B, H, d]
    (step 4 of SURVEY 8(c)).  prefix_k[i], prefix_v[i]: [L_i, n_kv, hd] of THIS layer for robot i."""
    B, H, d = n1.shape
    nq, nkv, hd = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    q = (n1 @ _as(W["wq"][l], dtype).T).reshape(B, H, nq, hd)
    k = (n1 @ _as(W["wk"][l], dtype).T).reshape(B, H, nkv, hd)
    v = (n1 @ _as(W["wv"][l], dtype).T).reshape(B, H, nkv, hd)
    o = np.empty((B, H, nq, hd), dtype=dtype)
    for i in range(B):
        L = prefix_k[i].shape[0]
        pos = L + np.arange(H)                                            # reading R7: per-robot positions
        q_i = rope(q[i], pos, cfg.rope_base)
        k_i = rope(k[i], pos, cfg.rope_base)
        k_all = np.concatenate([_as(prefix_k[i], dtype), k_i], axis=0)    # prefix K is stored rotated
        v_all = np.concatenate([_as(prefix_v[i], dtype), v[i]], axis=0)
        o[i] = attention_robot(q_i, k_all, v_all)
    return o.reshape(B, H, nq * hd) @ _as(W["wo"][l], dtype).T


def mlp_sublayer(cfg, W: Dict, l: int, n2: np.ndarray, dtype=F) -> np.ndarray:
    """GeGLU MLP half of a block, from the normed input n2 to the W_down output (reading R6)."""
    m = gelu_tanh(n2 @ _as(W["w_gate"][l], dtype).T) * (n2 @ _as(W["w_up"][l], dtype).T)
    return m @ _as(W["w_down"][l], dtype).T


def layer(cfg, W: Dict, l: int, h: np.ndarray, prefix_k: Sequence[np.ndarray],
          prefix_v: Sequence[np.ndarray], dtype=F) -> np.ndarray:
    """One pre-norm transformer block (step 4 of SURVEY 8(c)); h: [B, H, d]."""
    n1 = rmsnorm(h, _as(W["g_attn"][l], dtype), cfg.rms_eps)
    h = h + attention_sublayer(cfg, W, l, n1, prefix_k, prefix_v, dtype)
    n2 = rmsnorm(h, _as(W["g_mlp"][l], dtype), cfg.rms_eps)
    return h + mlp_sublayer(cfg, W, l, n2, dtype)


# ----------------------------------------------------------------------------- adaptive-norm variant
# SURVEY.md 8(f) item 4 / PAPER.md:438: the paper also evaluates pi0.5, whose action expert takes the
# flow-matching time through adaptive RMSNorm instead of the concatenated time MLP.  DESIGN.md reading
# R25 fixes the form (cfg.time_conditioning == 1):
#   cond   = swish(W_t2 swish(W_t1 tau(t) + b_t1) + b_t2)  in R^d       (W_t1 is [d, d] here)
#   h0     = W_in x + b_in                                               (no time in the token embedding)
#   every norm n:  (scale, shift, gate) = W_mod^n cond + b_mod^n  in R^{3d}, split in that order,
#                  y = h rsqrt(mean(h^2) + eps) (1 + scale) + shift     (no learned gain),
#                  h <- h + gate * sublayer(y);  the final norm uses scale and shift only.
def time_condition(cfg, W: Dict, t: np.ndarray, dtype=F) -> np.ndarray:
    """cond [B, d] of the adaptive-norm variant (reading R25)."""
    tau = sinusoidal_time_embedding(t, cfg.d_model, cfg.time_min_period, cfg.time_max_period, dtype)
    z = swish(tau @ _as(W["w_t1"], dtype).T + _as(W["b_t1"], dtype))
    return swish(z @ _as(W["w_t2"], dtype).T + _as(W["b_t2"], dtype))


def adarms(h: np.ndarray, cond: np.ndarray, w_mod: np.ndarray, b_mod: np.ndarray, eps: float):
    """Adaptive RMSNorm (reading R25): h [B, H, d], cond [B, d] -> (y [B, H, d], gate [B, 1, d])."""
    d = h.shape[-1]
    mod = cond @ w_mod.T + b_mod                                          # [B, 3d]
    scale, shift, gate = mod[:, None, :d], mod[:, None, d:2 * d], mod[:, None, 2 * d:]
    ms = np.mean(h * h, axis=-1, keepdims=True)
    return h / np.sqrt(ms + eps) * (1.0 + scale) + shift, gate


def velocity_adarms(cfg, W: Dict, x: np.ndarray, t: np.ndarray, prefix_k: Sequence[np.ndarray],
                    prefix_v: Sequence[np.ndarray], dtype=F) -> np.ndarray:
    """v(x, t) of the adaptive-norm variant.  prefix_k[i]: [layers, L_i, n_kv, hd]."""
    cond = time_condition(cfg, W, t, dtype)
    h = x @ _as(W["w_in"], dtype).T + _as(W["b_in"], dtype)
    for l in range(cfg.layers):
        y, gate = adarms(h, cond, _as(W["w_mod_attn"][l], dtype), _as(W["b_mod_attn"][l], dtype), cfg.rms_eps)
        h = h + gate * attention_sublayer(cfg, W, l, y, [pk[l] for pk in prefix_k], [pv[l] for pv in prefix_v], dtype)
        y, gate = adarms(h, cond, _as(W["w_mod_mlp"][l], dtype), _as(W["b_mod_mlp"][l], dtype), cfg.rms_eps)
        h = h + gate * mlp_sublayer(cfg, W, l, y, dtype)
    y, _ = adarms(h, cond, _as(W["w_mod_final"], dtype), _as(W["b_mod_final"], dtype), cfg.rms_eps)
    return y @ _as(W["w_out"], dtype).T + _as(W["b_out"], dtype)


def velocity(cfg, W: Dict, x: np.ndarray, t: np.ndarray, prefix_k: Sequence[np.ndarray],
             prefix_v: Sequence[np.ndarray], dtype=F) -> np.ndarray:
    """v(x, t) for a batch of robots (steps 1-5).  prefix_k[i]: [layers, L_i, n_kv, hd]."""
    if getattr(cfg, "time_conditioning", 0) == 1:
        return velocity_adarms(cfg, W, x, t, prefix_k, prefix_v, dtype)
    h = embed(cfg, W, x, t, dtype)
    for l in range(cfg.layers):
        h = layer(cfg, W, l, h, [pk[l] for pk in prefix_k], [pv[l] for pv in prefix_v], dtype)
    n = rmsnorm(h, _as(W["g_final"], dtype), cfg.rms_eps)
    return n @ _as(W["w_out"], dtype).T + _as(W["b_out"], dtype)


def denoise_batch(cfg, W: Dict, prefix_k: Sequence[np.ndarray], prefix_v: Sequence[np.ndarray],
                  noise: np.ndarray, t_start: np.ndarray, dt: np.ndarray, n_steps: np.ndarray,
                  return_velocity: bool = False, dtype=F
                  ) -> Tuple[np.ndarray, Optional[List[np.ndarray]]]:
    """The whole call (steps 1-6, readings R1, R15, R16).

    Robot i is integrated for n_steps[i] Euler steps x <- x + dt_i v(x, t_k), with
    t_k = t_start[i] + k dt_i (by multiplication); the call runs max_i n_steps[i]
    iterations; a robot with k >= n_steps[i] is left untouched.
    Returns x [B, H, A] and, if asked, the list over k of v_k [B, H, A] (rows of inactive
    robots are zero).
    """
    x = np.array(noise, dtype=dtype, copy=True)
    t0 = np.asarray(t_start, dtype=dtype)
    dts = np.asarray(dt, dtype=dtype)
    ns = np.asarray(n_steps, dtype=np.int64)
    vel: List[np.ndarray] = []
    for k in range(int(ns.max()) if ns.size else 0):
        act = np.nonzero(ns > k)[0]
        t_k = t0[act] + k * dts[act]
        v = velocity(cfg, W, x[act], t_k, [prefix_k[i] for i in act], [prefix_v[i] for i in act], dtype)
        x[act] = x[act] + dts[act][:, None, None] * v
        if return_velocity:
            full = np.zeros_like(x)
            full[act] = v
            vel.append(full)
    return x, (vel if return_velocity else None)


def prefix_kv(cfg, hidden: np.ndarray, w_pk: np.ndarray, w_pv: np.ndarray, dtype=F):
    """The step before the loop (the VLM backbone processes the observation; SURVEY 8(f) item 4;
    reading R29 of DESIGN.md): one layer's prefix K/V of a robot from the backbone's NORMALISED hidden states of its
    L prefix tokens,  K = RoPE(n W_pk^T, positions 0..L-1)  ("K pre-rotated", BASELINE.json configs[1]; R7),
    V = n W_pv^T.   hidden [L, d_p]; w_pk, w_pv [n_kv * hd, d_p]  ->  K, V [L, n_kv, hd].
    (The backbone that produces `hidden` is out of scope: its weights are not public.)"""
    n = np.asarray(hidden, dtype=dtype)
    L = n.shape[0]
    k = (n @ _as(w_pk, dtype).T).reshape(L, cfg.n_kv_heads, cfg.head_dim)
    v = (n @ _as(w_pv, dtype).T).reshape(L, cfg.n_kv_heads, cfg.head_dim)
    return rope(k, np.arange(L), cfg.rope_base), v


def denoise_case(case, robots: Optional[Sequence[int]] = None, return_velocity: bool = False, dtype=F):
    """Run ``denoise_batch`` on a ``cases.Case`` (optionally only some robots — exact,
    because robots are independent units)."""
    idx = list(range(case.batch)) if robots is None else list(robots)
    pk, pv = [], []
    for i in idx:
        k_i, v_i = case.prefix_f32(i)
        pk.append(k_i)
        pv.append(v_i)
    return denoise_batch(case.cfg, case.weights, pk, pv, case.noise[idx], case.t_start[idx],
                         case.dt[idx], case.n_steps[idx], return_velocity, dtype)
