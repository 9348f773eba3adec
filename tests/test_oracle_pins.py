"""Pins for the CPU oracle (oracle/rosa_oracle.py) against things OTHER than itself:
scalar brute force written from the definitions, closed forms, invariants and torch fp64
library routines.  Pin numbers P1..P13 follow DESIGN.md / SURVEY.md section 8(c).
CPU only (``-m "not gpu"``)."""
import math

import numpy as np
import pytest
import torch

from oracle import rosa_oracle as O
from paper_2607_01088_b200 import cases

MICRO = cases.ExpertConfig(layers=2, d_model=16, n_q_heads=4, n_kv_heads=2, head_dim=8,
                           ffn=24, horizon=3, action_dim=3)


def micro_case(seed=11, lens=(5, 7), cfg=MICRO, random_gains=True, n_steps=3):
    c = cases.build_case("micro", seed, cfg, bf16=False, prefix_lens=list(lens), n_steps=n_steps)
    if random_gains:
        rng = np.random.default_rng(seed + 1000)
        c.weights["g_final"] = rng.uniform(0.5, 1.5, cfg.d_model).astype(np.float32)
        c.weights["g_attn"] = [rng.uniform(0.5, 1.5, cfg.d_model).astype(np.float32) for _ in range(cfg.layers)]
        c.weights["g_mlp"] = [rng.uniform(0.5, 1.5, cfg.d_model).astype(np.float32) for _ in range(cfg.layers)]
        # larger weights so softmax is not flat and every nonlinearity is exercised
        for k in cases.GLOBAL_WEIGHTS + cases.BIASES:
            c.weights[k] = (c.weights[k] * 12).astype(np.float32)
        for k in cases.LAYER_WEIGHTS:
            c.weights[k] = [(w * 12).astype(np.float32) for w in c.weights[k]]
    return c


# ------------------------------------------------------------------ scalar brute force (P1)
def _dot(a, b):
    s = 0.0
    for p, q in zip(a, b):
        s += float(p) * float(q)
    return s


def _matvec(Wm, x, b=None):
    return [_dot(Wm[o], x) + (float(b[o]) if b is not None else 0.0) for o in range(len(Wm))]


def _rms(x, g, eps):
    ms = sum(v * v for v in x) / len(x)
    r = 1.0 / math.sqrt(ms + eps)
    return [v * r * float(gg) for v, gg in zip(x, g)]


def _rope_vec(x, pos, base):
    hd = len(x)
    half = hd // 2
    y = [0.0] * hd
    for c in range(half):
        phi = pos * base ** (-2.0 * c / hd)
        y[c] = x[c] * math.cos(phi) - x[c + half] * math.sin(phi)
        y[c + half] = x[c + half] * math.cos(phi) + x[c] * math.sin(phi)
    return y


def _brute_attention_rows(cfg, W, l, n1, pk, pv):
    """W_o output rows of one robot's attention sublayer from its normed rows n1 [H][d] (scalar loops)."""
    H = cfg.horizon
    nq, nkv, hd = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    L = pk.shape[1]
    q, k, v = [], [], []
    for j in range(H):
        qj = _matvec(W["wq"][l], n1[j])
        kj = _matvec(W["wk"][l], n1[j])
        vj = _matvec(W["wv"][l], n1[j])
        q.append([_rope_vec(qj[a * hd:(a + 1) * hd], L + j, cfg.rope_base) for a in range(nq)])
        k.append([_rope_vec(kj[g * hd:(g + 1) * hd], L + j, cfg.rope_base) for g in range(nkv)])
        v.append([vj[g * hd:(g + 1) * hd] for g in range(nkv)])
    rows = []
    for j in range(H):
        o = []
        for a in range(nq):
            g = a // (nq // nkv)
            keys = [list(map(float, pk[l, s, g])) for s in range(L)] + [k[jj][g] for jj in range(H)]
            vals = [list(map(float, pv[l, s, g])) for s in range(L)] + [v[jj][g] for jj in range(H)]
            sc = [_dot(q[j][a], kk) / math.sqrt(hd) for kk in keys]
            e = [math.exp(s) for s in sc]            # plain definition, no max subtraction
            den = sum(e)
            o += [sum(e[s] * vals[s][c] for s in range(L + H)) / den for c in range(hd)]
        rows.append(_matvec(W["wo"][l], o))
    return rows


def _brute_mlp_row(W, l, n2):
    gt = _matvec(W["w_gate"][l], n2)
    up = _matvec(W["w_up"][l], n2)
    m = [0.5 * a_ * (1 + math.tanh(math.sqrt(2 / math.pi) * (a_ + 0.044715 * a_ ** 3))) * b_
         for a_, b_ in zip(gt, up)]
    return _matvec(W["w_down"][l], m)


def brute_velocity_robot(cfg, W, x, t, pk, pv):
    """v(x, t) of ONE robot with scalar loops only (math module), straight from the definitions."""
    d, H, A = cfg.d_model, cfg.horizon, cfg.action_dim
    nq, nkv, hd = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    L = pk.shape[1]
    half = d // 2
    tau = [0.0] * d
    for j in range(half):
        period = cfg.time_min_period * (cfg.time_max_period / cfg.time_min_period) ** (j / (half - 1))
        tau[j] = math.sin(2 * math.pi * t / period)
        tau[half + j] = math.cos(2 * math.pi * t / period)
    h = []
    for j in range(H):
        a = _matvec(W["w_in"], x[j], W["b_in"])
        u = tau + a
        z = _matvec(W["w_t1"], u, W["b_t1"])
        z = [v / (1.0 + math.exp(-v)) for v in z]
        h.append(_matvec(W["w_t2"], z, W["b_t2"]))
    for l in range(cfg.layers):
        proj = _brute_attention_rows(cfg, W, l, [_rms(h[j], W["g_attn"][l], cfg.rms_eps) for j in range(H)], pk, pv)
        for j in range(H):
            h[j] = [p + r for p, r in zip(h[j], proj[j])]
        for j in range(H):
            proj_j = _brute_mlp_row(W, l, _rms(h[j], W["g_mlp"][l], cfg.rms_eps))
            h[j] = [p + r for p, r in zip(h[j], proj_j)]
    out = []
    for j in range(H):
        n = _rms(h[j], W["g_final"], cfg.rms_eps)
        out.append(_matvec(W["w_out"], n, W["b_out"]))
    return np.array(out)


def test_p1_bruteforce_velocity_and_denoise():
    c = micro_case()
    ts = np.array([0.7, 0.3])
    pk = [c.prefix_k[i] for i in range(2)]
    pv = [c.prefix_v[i] for i in range(2)]
    v = O.velocity(c.cfg, c.weights, c.noise.astype(np.float64), ts, pk, pv)
    for i in range(2):
        vb = brute_velocity_robot(c.cfg, c.weights, c.noise[i].astype(np.float64), float(ts[i]), pk[i], pv[i])
        assert np.abs(vb).max() > 1e-2
        np.testing.assert_allclose(v[i], vb, rtol=0, atol=1e-11)
    # and the Euler loop around it (3 steps, per-robot dt)
    x, vel = O.denoise_case(c, return_velocity=True)
    for i in range(2):
        xb = c.noise[i].astype(np.float64)
        for k in range(int(c.n_steps[i])):
            tk = float(c.t_start[i]) + k * float(c.dt[i])
            vb = brute_velocity_robot(c.cfg, c.weights, xb, tk, pk[i], pv[i])
            np.testing.assert_allclose(vel[k][i], vb, rtol=0, atol=1e-10)
            xb = xb + float(c.dt[i]) * vb
        np.testing.assert_allclose(x[i], xb, rtol=0, atol=1e-10)


def test_p1_softmax_not_flat_in_micro_case():
    """The brute-force pin is only meaningful if attention weights are far from uniform."""
    c = micro_case()
    cfg = c.cfg
    h = O.embed(cfg, c.weights, c.noise.astype(np.float64), np.array([0.7, 0.3]))
    n1 = O.rmsnorm(h, c.weights["g_attn"][0].astype(np.float64), cfg.rms_eps)
    q = (n1 @ c.weights["wq"][0].astype(np.float64).T).reshape(2, cfg.horizon, cfg.n_q_heads, cfg.head_dim)
    s = q[0][:, 0, :] @ c.prefix_k[0][0][:, 0, :].astype(np.float64).T / math.sqrt(cfg.head_dim)
    assert s.std() > 0.5


# ------------------------------------------------------------------ P10 library routines
def test_p10_torch_library_routines():
    rng = np.random.default_rng(5)
    z = rng.standard_normal((7, 33)) * 3
    zt = torch.from_numpy(z)
    np.testing.assert_allclose(O.gelu_tanh(z), torch.nn.functional.gelu(zt, approximate="tanh").numpy(), atol=1e-14)
    np.testing.assert_allclose(O.swish(z), torch.nn.functional.silu(zt).numpy(), atol=1e-14)
    g = rng.uniform(0.5, 1.5, 33)
    ref = torch.nn.functional.rms_norm(zt, (33,), torch.from_numpy(g), eps=1e-6).numpy()
    np.testing.assert_allclose(O.rmsnorm(z, g, 1e-6), ref, atol=1e-14)
    # attention: n_q=4, n_kv=2 (GQA contiguous groups, R9), H=5 queries, 11 keys
    q = rng.standard_normal((5, 4, 8)); k = rng.standard_normal((11, 2, 8)); v = rng.standard_normal((11, 2, 8))
    o = O.attention_robot(q, k, v)
    qt = torch.from_numpy(q).permute(1, 0, 2)[None]
    kt = torch.from_numpy(k).permute(1, 0, 2).repeat_interleave(2, dim=0)[None]
    vt = torch.from_numpy(v).permute(1, 0, 2).repeat_interleave(2, dim=0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt)[0].permute(1, 0, 2).numpy()
    np.testing.assert_allclose(o, ref, atol=1e-13)


def test_gelu_tanh_close_to_erf_gelu():
    z = np.linspace(-6, 6, 1001)
    erf = 0.5 * z * (1 + np.vectorize(math.erf)(z / math.sqrt(2)))
    assert np.abs(O.gelu_tanh(z) - erf).max() < 1e-3      # R6: forms differ by < 1e-3 abs


# ------------------------------------------------------------------ closed forms of the pieces
def test_time_embedding_closed_form():
    d = 128
    tau = O.sinusoidal_time_embedding(np.array([1.0, 0.5, 0.0]), d, 4e-3, 4.0)
    half = d // 2
    # slowest channel: period 4.0 -> angle = pi/2 * t ... at t=1 sin=1, cos=0
    assert abs(tau[0, half - 1] - 1.0) < 1e-12 and abs(tau[0, d - 1]) < 1e-12
    assert abs(tau[1, half - 1] - math.sin(math.pi / 4)) < 1e-12
    # fastest channel: period 4e-3 -> 250 full turns at t=1
    assert abs(tau[0, 0]) < 1e-9 and abs(tau[0, half] - 1.0) < 1e-9
    # t = 0: sin half 0, cos half 1
    assert np.all(tau[2, :half] == 0) and np.all(tau[2, half:] == 1)
    # geometric period ladder
    j = 10
    period = 4e-3 * (1000.0) ** (j / (half - 1))
    assert abs(tau[1, j] - math.sin(2 * math.pi * 0.5 / period)) < 1e-10


def test_rope_closed_forms():
    rng = np.random.default_rng(3)
    x = rng.standard_normal((4, 2, 8))
    np.testing.assert_array_equal(O.rope(x, np.zeros(4), 10000.0), x)           # pos 0 = identity
    y = O.rope(x, np.array([3, 17, 100, 865]), 10000.0)
    np.testing.assert_allclose(np.linalg.norm(y, axis=-1), np.linalg.norm(x, axis=-1), rtol=1e-13)
    # hd = 2 is a plain 2-D rotation by pos (theta_0 = 1)
    v = np.array([[[1.0, 0.0]]])
    np.testing.assert_allclose(O.rope(v, np.array([math.pi / 2]), 10000.0)[0, 0], [0.0, 1.0], atol=1e-15)
    # pair (c, c+hd/2) rotates by pos * base^(-2c/hd): check channel c=1 of hd=8 at pos=5
    e = np.zeros((1, 1, 8)); e[0, 0, 1] = 1.0
    r = O.rope(e, np.array([5.0]), 10000.0)[0, 0]
    phi = 5.0 * 10000.0 ** (-2.0 / 8.0)
    np.testing.assert_allclose([r[1], r[5]], [math.cos(phi), math.sin(phi)], atol=1e-15)
    assert np.count_nonzero(r) == 2
    # relative-position property: <rope(q, m), rope(k, n)> depends on m - n only
    q = rng.standard_normal((1, 1, 8)); k = rng.standard_normal((1, 1, 8))
    a = np.sum(O.rope(q, np.array([9.0]), 1e4) * O.rope(k, np.array([4.0]), 1e4))
    b = np.sum(O.rope(q, np.array([109.0]), 1e4) * O.rope(k, np.array([104.0]), 1e4))
    assert abs(a - b) < 1e-12


# ------------------------------------------------------------------ invariants of the whole call
def _run(c, **kw):
    return O.denoise_case(c, **kw)


def test_p2_batch_invariance_and_p3_permutation():
    c = micro_case(lens=(5, 7, 0, 9), seed=21)          # includes L = 0 (self-attention only, R8)
    x, _ = _run(c)
    for i in range(c.batch):
        xi, _ = _run(c, robots=[i])
        np.testing.assert_allclose(xi[0], x[i], rtol=0, atol=1e-13)
    perm = [2, 0, 3, 1]
    xp, _ = _run(c, robots=perm)
    np.testing.assert_allclose(xp, x[perm], rtol=0, atol=1e-13)


def test_p4_zero_output_projection_leaves_x_unchanged():
    c = micro_case()
    c.weights["w_out"] = np.zeros_like(c.weights["w_out"])
    c.weights["b_out"] = np.zeros_like(c.weights["b_out"])
    x, _ = _run(c)
    np.testing.assert_array_equal(x, c.noise.astype(np.float64))


def test_p5_constant_velocity_closed_form():
    c = micro_case(lens=(5, 7, 6), seed=31)
    c.weights["w_out"] = np.zeros_like(c.weights["w_out"])
    bo = c.weights["b_out"].astype(np.float64)
    c.t_start = np.array([1.0, 0.6, 0.3], dtype=np.float32)
    c.n_steps = np.array([4, 3, 1], dtype=np.int32)
    c.dt = (-c.t_start / c.n_steps).astype(np.float32)
    x, vel = _run(c, return_velocity=True)
    assert len(vel) == 4
    for i in range(3):
        # x_n = x0 + n dt c  (= x0 - t0 c up to the fp32 rounding of dt)
        want = c.noise[i].astype(np.float64) + int(c.n_steps[i]) * float(c.dt[i]) * bo[None, :]
        np.testing.assert_allclose(x[i], want, rtol=0, atol=1e-14)
        np.testing.assert_allclose(want, c.noise[i] - float(c.t_start[i]) * bo[None, :], atol=1e-7)
    # R16: a finished robot is untouched and reports zero velocity afterwards
    assert np.all(vel[3][2] == 0) and np.all(vel[1][2] == 0) and np.all(vel[0][2] == bo)


def test_p6_step_composition():
    c = micro_case(n_steps=10, seed=41)
    x_full, _ = _run(c)
    a = c.subset([0, 1]); a.n_steps[:] = 4
    x_a, _ = _run(a)
    b = c.subset([0, 1]); b.noise = x_a.astype(np.float32)   # (fp32 hand-over as through the API)
    # exact hand-over in fp64 instead, to keep the comparison at rounding level:
    pk = [b.prefix_k[i] for i in range(2)]; pv = [b.prefix_v[i] for i in range(2)]
    t_mid = c.t_start.astype(np.float64) + 4 * c.dt.astype(np.float64)
    x_b, _ = O.denoise_batch(b.cfg, b.weights, pk, pv, x_a, t_mid, c.dt, np.array([6, 6]))
    np.testing.assert_allclose(x_b, x_full, rtol=0, atol=1e-12)


def test_p7_uniform_attention_special_case():
    """W_q = 0 -> all logits 0 -> o = mean over the L_i + H rows of [V ; v] (softmax
    denominator counts exactly L_i + H keys)."""
    c = micro_case(lens=(5, 7))
    cfg = c.cfg
    l = 0
    W = c.weights
    W["wq"][l] = np.zeros_like(W["wq"][l])
    h = np.random.default_rng(0).standard_normal((2, cfg.horizon, cfg.d_model))
    pk = [c.prefix_k[i][l] for i in range(2)]; pv = [c.prefix_v[i][l] for i in range(2)]
    # isolate the attention branch: zero the MLP
    W["w_down"][l] = np.zeros_like(W["w_down"][l])
    out = O.layer(cfg, W, l, h, pk, pv)
    n1 = O.rmsnorm(h, W["g_attn"][l].astype(np.float64), cfg.rms_eps)
    v_own = (n1 @ W["wv"][l].astype(np.float64).T).reshape(2, cfg.horizon, cfg.n_kv_heads, cfg.head_dim)
    for i in range(2):
        mean_v = np.concatenate([pv[i].astype(np.float64), v_own[i]], axis=0).mean(axis=0)   # [n_kv, hd]
        o = np.repeat(mean_v, cfg.n_q_heads // cfg.n_kv_heads, axis=0).reshape(-1)           # [n_q*hd]
        want = h[i] + (o @ W["wo"][l].astype(np.float64).T)[None, :]
        np.testing.assert_allclose(out[i], want, rtol=0, atol=1e-13)


def test_p8_rope_shift_invariance():
    """Draw UNROTATED prefix K, rotate it at positions p..p+L-1 here, and place the action
    tokens at p+L+j: the layer output must not depend on p (q and k use the same R7
    convention).  p = 0 is ``layer()`` itself; p = 13 re-assembles the same block from the
    oracle's pieces with the shifted positions."""
    c = micro_case(lens=(6,), seed=51)
    cfg = c.cfg
    l = 1
    rng = np.random.default_rng(1)
    k_raw = rng.standard_normal((6, cfg.n_kv_heads, cfg.head_dim))
    v_pre = rng.standard_normal((6, cfg.n_kv_heads, cfg.head_dim))
    h = rng.standard_normal((1, cfg.horizon, cfg.d_model))
    outs = []
    for p in (0, 13):
        k_rot = O.rope(k_raw, p + np.arange(6), cfg.rope_base)
        if p == 0:
            outs.append(O.layer(cfg, c.weights, l, h, [k_rot], [v_pre]))
        else:
            # call the pieces with explicit positions, exactly as layer() does but at offset p
            W = c.weights
            n1 = O.rmsnorm(h, W["g_attn"][l].astype(np.float64), cfg.rms_eps)
            q = (n1 @ W["wq"][l].astype(np.float64).T).reshape(1, cfg.horizon, cfg.n_q_heads, cfg.head_dim)
            k = (n1 @ W["wk"][l].astype(np.float64).T).reshape(1, cfg.horizon, cfg.n_kv_heads, cfg.head_dim)
            v = (n1 @ W["wv"][l].astype(np.float64).T).reshape(1, cfg.horizon, cfg.n_kv_heads, cfg.head_dim)
            pos = p + 6 + np.arange(cfg.horizon)
            o = O.attention_robot(O.rope(q[0], pos, cfg.rope_base),
                                  np.concatenate([k_rot, O.rope(k[0], pos, cfg.rope_base)]),
                                  np.concatenate([v_pre, v[0]]))
            h2 = h + o.reshape(1, cfg.horizon, -1) @ W["wo"][l].astype(np.float64).T
            n2 = O.rmsnorm(h2, W["g_mlp"][l].astype(np.float64), cfg.rms_eps)
            m = O.gelu_tanh(n2 @ W["w_gate"][l].astype(np.float64).T) * (n2 @ W["w_up"][l].astype(np.float64).T)
            outs.append(h2 + m @ W["w_down"][l].astype(np.float64).T)
    np.testing.assert_allclose(outs[1], outs[0], rtol=0, atol=1e-11)


def test_p9_norm_scale_invariance():
    rng = np.random.default_rng(2)
    x = rng.standard_normal((5, 64)); g = rng.uniform(0.5, 1.5, 64)
    a = O.rmsnorm(x, g, 1e-6); b = O.rmsnorm(37.0 * x, g, 1e-6)
    np.testing.assert_allclose(a, b, rtol=1e-6)
    # unit gain: rows have unit RMS
    np.testing.assert_allclose(np.sqrt(np.mean(O.rmsnorm(x, np.ones(64), 0.0) ** 2, axis=1)), 1.0, rtol=1e-14)


def test_p11_single_step_linear_in_dt():
    c = micro_case(n_steps=1)
    x1, v1 = _run(c, return_velocity=True)
    c2 = micro_case(n_steps=1); c2.dt = (c2.dt / 2).astype(np.float32)
    x2, v2 = _run(c2, return_velocity=True)
    np.testing.assert_array_equal(v1[0], v2[0])
    s1 = (x1 - c.noise) / c.dt.astype(np.float64)[:, None, None]
    s2 = (x2 - c2.noise) / c2.dt.astype(np.float64)[:, None, None]
    np.testing.assert_allclose(s1, s2, atol=1e-12)
    np.testing.assert_allclose(s1, v1[0], atol=1e-12)


def test_time_concat_order_r2():
    """u = [tau ; a]: W_1[:, :d] multiplies the time half.  Zeroing W_1[:, :d] must remove
    all dependence on t; zeroing W_1[:, d:] must remove all dependence on x."""
    c = micro_case()
    cfg, W = c.cfg, c.weights
    d = cfg.d_model
    x = c.noise.astype(np.float64)
    Wa = dict(W); Wa["w_t1"] = W["w_t1"].copy(); Wa["w_t1"][:, :d] = 0
    np.testing.assert_array_equal(O.embed(cfg, Wa, x, np.array([0.2, 0.9])), O.embed(cfg, Wa, x, np.array([0.5, 0.1])))
    Wb = dict(W); Wb["w_t1"] = W["w_t1"].copy(); Wb["w_t1"][:, d:] = 0
    np.testing.assert_array_equal(O.embed(cfg, Wb, x, np.array([0.2, 0.9])), O.embed(cfg, Wb, 2 * x + 1, np.array([0.2, 0.9])))
    assert np.abs(O.embed(cfg, W, x, np.array([0.2, 0.9])) - O.embed(cfg, W, x, np.array([0.5, 0.1]))).max() > 1e-3


def test_cases_generator_contract():
    c0 = cases.make_case(0)
    assert c0.batch == 2 and list(c0.prefix_lens) == [48, 64] and list(c0.n_steps) == [4, 4]
    assert np.allclose(c0.dt, -0.25) and c0.prefix_k[0].shape == (2, 48, 1, 32)
    n_params = sum(int(np.prod(s)) * (c0.cfg.layers if k in cases.LAYER_WEIGHTS else 1)
                   for k, s in cases.weight_shapes(c0.cfg).items()) + (2 * c0.cfg.layers + 1) * c0.cfg.d_model
    assert n_params == 527111
    again = cases.make_case(0)
    np.testing.assert_array_equal(c0.noise, again.noise)
    np.testing.assert_array_equal(c0.weights["wq"][1], again.weights["wq"][1])
    # bf16 rounding helper: RNE, idempotent, exact on representable values
    x = np.array([1.0, 1.00390625, 1.005859375, -3.14159, 1e-20, 65504.0], dtype=np.float32)
    r = cases.round_bf16(x)
    np.testing.assert_array_equal(cases.round_bf16(r), r)
    assert r[0] == 1.0 and r[1] == 1.0 and r[2] == 1.0078125   # tie -> even; above tie -> up
    t = torch.from_numpy(x).to(torch.bfloat16).to(torch.float32).numpy()
    np.testing.assert_array_equal(r, t)
    c3 = cases.make_case(3, batch=16, with_prefix=False)
    assert set(np.round(c3.t_start * 10).astype(int)) <= set(range(1, 11))
    np.testing.assert_array_equal(c3.n_steps, np.round(c3.t_start * 10).astype(np.int32))
    assert c3.prefix_lens.min() >= 400 and c3.prefix_lens.max() <= 1200


# ------------------------------------------------------------------ adaptive-norm variant (reading R25)
MICRO_ADA = cases.ExpertConfig(layers=2, d_model=16, n_q_heads=4, n_kv_heads=2, head_dim=8,
                               ffn=24, horizon=3, action_dim=3, time_conditioning=1)


def micro_ada_case(seed=21, lens=(5, 7)):
    c = cases.build_case("micro-ada", seed, MICRO_ADA, bf16=False, prefix_lens=list(lens), n_steps=3)
    for k in cases.GLOBAL_WEIGHTS + cases.BIASES:
        c.weights[k] = (c.weights[k] * 12).astype(np.float32)
    for k in cases.LAYER_WEIGHTS + ("w_mod_attn", "w_mod_mlp"):
        c.weights[k] = [(w * 12).astype(np.float32) for w in c.weights[k]]
    c.weights["w_mod_final"] = (c.weights["w_mod_final"] * 12).astype(np.float32)
    return c


def brute_velocity_adarms_robot(cfg, W, x, t, pk, pv):
    """v(x, t) of ONE robot of the adaptive-norm variant, scalar loops only, from reading R25."""
    d, H = cfg.d_model, cfg.horizon
    half = d // 2
    tau = [0.0] * d
    for j in range(half):
        period = cfg.time_min_period * (cfg.time_max_period / cfg.time_min_period) ** (j / (half - 1))
        tau[j] = math.sin(2 * math.pi * t / period)
        tau[half + j] = math.cos(2 * math.pi * t / period)
    z = [v / (1.0 + math.exp(-v)) for v in _matvec(W["w_t1"], tau, W["b_t1"])]
    cond = [v / (1.0 + math.exp(-v)) for v in _matvec(W["w_t2"], z, W["b_t2"])]

    def ada(row, wm, bm):
        mod = _matvec(wm, cond, bm)                       # [scale | shift | gate]
        r = 1.0 / math.sqrt(sum(v * v for v in row) / d + cfg.rms_eps)
        return [row[c] * r * (1.0 + mod[c]) + mod[d + c] for c in range(d)], mod[2 * d:]

    h = [_matvec(W["w_in"], x[j], W["b_in"]) for j in range(H)]
    for l in range(cfg.layers):
        ys, gate = [], None
        for j in range(H):
            y, gate = ada(h[j], W["w_mod_attn"][l], W["b_mod_attn"][l])
            ys.append(y)
        proj = _brute_attention_rows(cfg, W, l, ys, pk, pv)
        for j in range(H):
            h[j] = [p + g * r for p, g, r in zip(h[j], gate, proj[j])]
        for j in range(H):
            y, gate = ada(h[j], W["w_mod_mlp"][l], W["b_mod_mlp"][l])
            h[j] = [p + g * r for p, g, r in zip(h[j], gate, _brute_mlp_row(W, l, y))]
    out = []
    for j in range(H):
        y, _ = ada(h[j], W["w_mod_final"], W["b_mod_final"])
        out.append(_matvec(W["w_out"], y, W["b_out"]))
    return np.array(out)


def test_adarms_bruteforce_velocity_and_denoise():
    c = micro_ada_case()
    ts = np.array([0.7, 0.3])
    pk = [c.prefix_k[i] for i in range(2)]
    pv = [c.prefix_v[i] for i in range(2)]
    v = O.velocity(c.cfg, c.weights, c.noise.astype(np.float64), ts, pk, pv)
    for i in range(2):
        vb = brute_velocity_adarms_robot(c.cfg, c.weights, c.noise[i].astype(np.float64), float(ts[i]), pk[i], pv[i])
        assert np.abs(vb).max() > 1e-2
        np.testing.assert_allclose(v[i], vb, rtol=0, atol=1e-11)
    x, vel = O.denoise_case(c, return_velocity=True)
    for i in range(2):
        xb = c.noise[i].astype(np.float64)
        for k in range(int(c.n_steps[i])):
            vb = brute_velocity_adarms_robot(c.cfg, c.weights, xb, float(c.t_start[i]) + k * float(c.dt[i]), pk[i], pv[i])
            np.testing.assert_allclose(vel[k][i], vb, rtol=0, atol=1e-10)
            xb = xb + float(c.dt[i]) * vb
        np.testing.assert_allclose(x[i], xb, rtol=0, atol=1e-10)
    # time really conditions the output, and through the modulation only
    v2 = O.velocity(c.cfg, c.weights, c.noise.astype(np.float64), ts[::-1].copy(), pk, pv)
    assert np.abs(v2 - v).max() > 1e-3


def _zero_mod(c, scale=0.0, shift=0.0, gate=1.0):
    d = c.cfg.d_model
    b = np.concatenate([np.full(d, scale), np.full(d, shift), np.full(d, gate)]).astype(np.float32)
    for k in ("w_mod_attn", "w_mod_mlp"):
        c.weights[k] = [np.zeros_like(w) for w in c.weights[k]]
    c.weights["w_mod_final"] = np.zeros_like(c.weights["w_mod_final"])
    c.weights["b_mod_attn"] = [b.copy() for _ in range(c.cfg.layers)]
    c.weights["b_mod_mlp"] = [b.copy() for _ in range(c.cfg.layers)]
    c.weights["b_mod_final"] = b.copy()
    return c


def test_adarms_reduces_to_plain_blocks_with_identity_modulation():
    """scale = shift = 0, gate = 1: the stack is the pinned pre-norm blocks (gains 1) on h0 = W_in x + b_in."""
    c = _zero_mod(micro_ada_case())
    W, cfg = c.weights, c.cfg
    x = c.noise.astype(np.float64)
    pk = [c.prefix_k[i] for i in range(2)]
    pv = [c.prefix_v[i] for i in range(2)]
    v = O.velocity(cfg, W, x, np.array([0.9, 0.2]), pk, pv)
    h = x @ W["w_in"].astype(np.float64).T + W["b_in"]
    for l in range(cfg.layers):
        h = O.layer(cfg, W, l, h, [p[l] for p in pk], [p[l] for p in pv])     # g_attn = g_mlp = 1 in the generator
    want = O.rmsnorm(h, np.ones(cfg.d_model), cfg.rms_eps) @ W["w_out"].astype(np.float64).T + W["b_out"]
    np.testing.assert_allclose(v, want, rtol=0, atol=1e-12)
    # ... and then the output does not depend on t at all
    v2 = O.velocity(cfg, W, x, np.array([0.1, 0.6]), pk, pv)
    np.testing.assert_allclose(v2, v, rtol=0, atol=1e-13)


def test_adarms_zero_gate_is_identity_and_shift_only_closed_form():
    c = _zero_mod(micro_ada_case(), gate=0.0)
    W, cfg = c.weights, c.cfg
    x = c.noise.astype(np.float64)
    pk = [c.prefix_k[i] for i in range(2)]
    pv = [c.prefix_v[i] for i in range(2)]
    v = O.velocity(cfg, W, x, np.array([0.9, 0.2]), pk, pv)
    h0 = x @ W["w_in"].astype(np.float64).T + W["b_in"]
    want = h0 / np.sqrt(np.mean(h0 * h0, axis=-1, keepdims=True) + cfg.rms_eps) @ W["w_out"].astype(np.float64).T + W["b_out"]
    np.testing.assert_allclose(v, want, rtol=0, atol=1e-12)
    # scale = -1 removes the token entirely: y = shift, so v = W_out (s 1) + b_out for every token
    c = _zero_mod(micro_ada_case(), scale=-1.0, shift=0.37, gate=0.0)
    v = O.velocity(c.cfg, c.weights, x, np.array([0.9, 0.2]), pk, pv)
    want_row = c.weights["w_out"].astype(np.float64) @ np.full(cfg.d_model, np.float64(np.float32(0.37))) + c.weights["b_out"]
    np.testing.assert_allclose(v, np.broadcast_to(want_row, v.shape), rtol=0, atol=1e-12)


def test_adarms_torch_third_opinion():
    c = micro_ada_case()
    W, cfg = c.weights, c.cfg
    d = cfg.d_model
    t = np.array([0.65, 0.15])
    cond = O.time_condition(cfg, W, t)
    tau = torch.from_numpy(O.sinusoidal_time_embedding(t, d, cfg.time_min_period, cfg.time_max_period))
    tl = lambda k: torch.from_numpy(W[k].astype(np.float64))
    z = torch.nn.functional.silu(torch.nn.functional.linear(tau, tl("w_t1"), tl("b_t1")))
    want = torch.nn.functional.silu(torch.nn.functional.linear(z, tl("w_t2"), tl("b_t2"))).numpy()
    np.testing.assert_allclose(cond, want, rtol=0, atol=1e-13)
    rng = np.random.default_rng(3)
    h = rng.standard_normal((2, cfg.horizon, d))
    wm, bm = W["w_mod_attn"][1].astype(np.float64), W["b_mod_attn"][1].astype(np.float64)
    y, gate = O.adarms(h, cond, wm, bm, cfg.rms_eps)
    mod = torch.nn.functional.linear(torch.from_numpy(cond), torch.from_numpy(wm), torch.from_numpy(bm))
    sc, sh, gt = mod.chunk(3, dim=-1)
    yt = torch.nn.functional.rms_norm(torch.from_numpy(h), (d,), eps=cfg.rms_eps) * (1 + sc[:, None]) + sh[:, None]
    np.testing.assert_allclose(y, yt.numpy(), rtol=0, atol=1e-13)
    np.testing.assert_allclose(gate[:, 0], gt.numpy(), rtol=0, atol=1e-15)


def test_adarms_batch_invariance_and_generator_contract():
    c = cases.make_adarms_case("tiny")
    assert c.cfg.time_conditioning == 1 and c.weights["w_t1"].shape == (128, 128)
    assert c.weights["w_mod_attn"][0].shape == (384, 128) and abs(float(c.weights["b_mod_mlp"][1][256:].mean()) - 1.0) < 0.01
    x, _ = O.denoise_case(c)
    for i in range(c.batch):
        xi, _ = O.denoise_case(c, robots=[i])
        np.testing.assert_allclose(xi[0], x[i], rtol=0, atol=1e-13)       # BLAS blocking differs with the batch
    # the modulation weights come from their own generator: the first draw of the main stream is the base one's
    base = cases.build_case("b", 5, cases.TINY, bf16=False, prefix_lens=[48, 64], n_steps=4)
    np.testing.assert_array_equal(base.weights["w_in"], c.weights["w_in"])


# ------------------------------------------------------------------ prefix K/V production (reading R29)
def test_prefix_kv_brute_force_and_closed_forms():
    """O.prefix_kv against a scalar loop written from the definition (math only): K[t, c] of head g pairs channel c
    with c + hd/2 and rotates by t * base^(-2c/hd); V is the plain projection.  Closed forms: token 0 is not rotated;
    with W_pk = identity the result is the rotation of the hidden state itself; rows keep their norm; and the K it
    produces is what P8 expects (an action-token query scores the same against it wherever the prefix starts)."""
    cfg = cases.TINY
    hd, nkv = cfg.head_dim, cfg.n_kv_heads
    rng = np.random.default_rng(61)
    L, dp = 5, 12
    n = rng.standard_normal((L, dp))
    wk = rng.standard_normal((nkv * hd, dp)) * 0.3
    wv = rng.standard_normal((nkv * hd, dp)) * 0.3
    K, V = O.prefix_kv(cfg, n, wk, wv)
    assert K.shape == V.shape == (L, nkv, hd)
    half = hd // 2
    for t in range(L):
        for g in range(nkv):
            proj_k = [sum(n[t, j] * wk[g * hd + c, j] for j in range(dp)) for c in range(hd)]
            proj_v = [sum(n[t, j] * wv[g * hd + c, j] for j in range(dp)) for c in range(hd)]
            for c in range(half):
                phi = t * cfg.rope_base ** (-2.0 * c / hd)
                lo = proj_k[c] * math.cos(phi) - proj_k[c + half] * math.sin(phi)
                hi = proj_k[c + half] * math.cos(phi) + proj_k[c] * math.sin(phi)
                assert abs(K[t, g, c] - lo) < 1e-12 and abs(K[t, g, c + half] - hi) < 1e-12
            for c in range(hd):
                assert abs(V[t, g, c] - proj_v[c]) < 1e-12
    np.testing.assert_allclose(K[0].ravel(), n[0] @ wk.T, rtol=1e-13)                       # position 0: no rotation
    np.testing.assert_allclose(np.linalg.norm(K, axis=-1), np.linalg.norm((n @ wk.T).reshape(L, nkv, hd), axis=-1), rtol=1e-13)
    eye = np.eye(nkv * hd)
    Ki, Vi = O.prefix_kv(cfg, n[:, :1].repeat(nkv * hd, axis=1) * 0 + rng.standard_normal((L, nkv * hd)), eye, eye)
    np.testing.assert_allclose(Ki, O.rope(Vi, np.arange(L), cfg.rope_base), rtol=1e-13)     # W = I: K is the rotated input, V the input
    # relative positions: <rope(q, L + j), K[t]> equals the unrotated <q, k_t> rotated by (L + j - t) only
    q = rng.standard_normal((1, nkv, hd))
    s1 = np.sum(O.rope(q, np.array([L + 2.0]), cfg.rope_base)[0] * K[3])
    k3 = (n[3] @ wk.T).reshape(1, nkv, hd)
    s2 = np.sum(O.rope(q, np.array([L + 2.0 - 3.0]), cfg.rope_base)[0] * k3[0])
    assert abs(s1 - s2) < 1e-12
