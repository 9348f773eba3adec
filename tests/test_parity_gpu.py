"""GPU parity: rosa_denoise_batch* (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json north_star (3):
final actions max-abs <= 2e-2 and rel-L2 <= 1e-2; per-step velocity rel-L2 <= 5e-3
(rel-L2 over the whole compared tensor, per Euler step for the velocity; reading R18).

Full-size cases (cfg2 B=64, cfg3 B=256, sweep B up to 512) run the WHOLE batch on the GPU in
the launch configuration bench.py times and compare a sample of robots with the oracle: robots
are independent units (pin P2), so the oracle's single-robot result is the exact expectation
for that robot's rows of the batched call."""
import numpy as np
import pytest
import torch

from oracle import rosa_oracle as O
from paper_2607_01088_b200 import binding as rosa
from paper_2607_01088_b200 import build as rosa_build
from paper_2607_01088_b200 import cases
from paper_2607_01088_b200.runner import DeviceFleet, LoadedCase, rel_l2

pytestmark = pytest.mark.gpu

TOL_ACT_ABS, TOL_ACT_REL, TOL_VEL_REL = 2e-2, 1e-2, 5e-3

# pi0 head geometry (8 q heads / 1 kv head / head_dim 256, H=50, A=32: the tcgen05 kernels) on a
# narrow 2-layer model, so the oracle finishes edge-case batches in seconds
MINI = cases.ExpertConfig(layers=2, d_model=256, n_q_heads=8, n_kv_heads=1, head_dim=256,
                          ffn=512, horizon=50, action_dim=32)


@pytest.fixture(scope="module", autouse=True)
def _built():
    rosa_build.build()
    rosa.load()


def compare(label, got_x, got_v, want_x, want_v):
    assert np.all(np.isfinite(got_x)), label
    err_abs = float(np.abs(got_x - want_x).max())
    err_rel = rel_l2(got_x, want_x)
    vel_rel = [rel_l2(got_v[k], want_v[k]) for k in range(len(want_v)) if np.any(want_v[k])]
    print(f"[{label}] actions max-abs {err_abs:.3e} rel-L2 {err_rel:.3e}; velocity rel-L2 max {max(vel_rel):.3e}")
    assert err_abs <= TOL_ACT_ABS, (label, err_abs)
    assert err_rel <= TOL_ACT_REL, (label, err_rel)
    assert max(vel_rel) <= TOL_VEL_REL, (label, vel_rel)


def check_against_oracle(case, lc, robots, label, sample=None):
    """Run `robots` as ONE batch on the GPU; oracle on `sample` (positions in `robots`, default all)."""
    got_x, got_v = lc.run(robots=robots, want_velocity=True)
    pos = list(range(len(robots))) if sample is None else list(sample)
    want_x, want_v = O.denoise_case(case, robots=[robots[p] for p in pos], return_velocity=True)
    compare(label, got_x[pos], [v[pos] for v in got_v[:len(want_v)]], want_x, want_v)
    return got_x, got_v


def test_cfg0_tiny_fp32():
    case = cases.make_case(0)
    lc = LoadedCase(case)
    assert rosa.rosa_kernel_family(lc.expert) == 0      # d=128 / head_dim 32: the shape-generic family
    check_against_oracle(case, lc, [0, 1], "cfg0")
    lc.close()


def test_cfg1_pi0_b8():
    case = cases.make_case(1)
    lc = LoadedCase(case)
    assert rosa.rosa_kernel_family(lc.expert) == 1
    check_against_oracle(case, lc, list(range(8)), "cfg1")
    lc.close()


def test_cfg2_fleet_b64_ragged_full():
    """The headline workload, ALL 64 robots against the oracle (full tensors on cfg0-3): every ragged
    prefix length, every attention work-list segment and every GEMM row block of the launch bench.py times."""
    case = cases.make_case(2)
    assert case.batch == 64 and case.prefix_lens.min() >= 600 and case.prefix_lens.max() <= 1000
    lc = LoadedCase(case)
    check_against_oracle(case, lc, list(range(64)), "cfg2-full")
    lc.close()


def test_cfg3_continuous_batching_b256_sampled():
    case = cases.make_case(3)
    assert case.batch == 256
    ns = case.n_steps
    # stratified over the remaining-step counts (three robots of each count that occurs: first, middle, last), plus
    # the first and last robots and the robots whose 50 token rows straddle a 256-row tile boundary after the
    # library's own ordering is unknown here, so simply every 16th robot as well: 40+ of the 256
    sample = {0, 255} | set(range(7, 256, 16))
    for n in np.unique(ns):
        idx = np.nonzero(ns == n)[0]
        sample |= {int(idx[0]), int(idx[len(idx) // 2]), int(idx[-1])}
    sample = sorted(sample)
    assert len(sample) >= 32
    lc = LoadedCase(case)
    got_x, got_v = check_against_oracle(case, lc, list(range(256)), "cfg3", sample=sample)
    # R16: velocity rows of a robot are zero once it is inactive
    for k in range(got_v.shape[0]):
        inactive = ns <= k
        assert not np.any(got_v[k][inactive])
    lc.close()


def test_cfg3_parity_variant_per_robot_dt():
    """R15 parity-only variant: n_i drawn independently of t_i, so dt_i truly differs per robot."""
    case = cases.build_case("cfg3-variant", 33, MINI, bf16=True, draw_lens=(40, 200), batch=12)
    rng = np.random.default_rng(5)
    case.n_steps = rng.integers(1, 7, size=12).astype(np.int32)
    case.t_start = (rng.integers(1, 11, size=12) / 10.0).astype(np.float32)
    case.dt = (-case.t_start / case.n_steps).astype(np.float32)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, list(range(12)), "cfg3-variant")
    lc.close()


@pytest.mark.parametrize("B,sample", [(1, [0]), (2, [0, 1]), (3, [0, 2]), (4, [1, 3]), (16, [0, 15]), (25, [3, 24]),
                                      (32, [7, 31]), (49, [11, 48]), (56, [30, 55]), (128, [0, 127])])
def test_cfg4_sweep_points(B, sample):
    """Every batch size of the sweep up to 128 (8 and 64 are cfg1 / cfg2's sizes), plus one B inside each range in
    which the residual GEMMs pick another N-tile width (21-30, 47-51, 52-61: gemm_tcgen05.cu resid_bn)."""
    case = cases.make_case(4, batch=B)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, list(range(B)), f"cfg4-B{B}", sample=sample)
    lc.close()


def test_cfg4_max_batch_512_property_and_sample():
    """B=512 (largest sweep point): batch invariance on the GPU for three robots, and one robot
    against the oracle (its prefix K/V is copied back from the seeded device generator)."""
    base = cases.make_case(4, batch=1, with_prefix=False)
    fl = DeviceFleet(base, [816] * 512, seed=4)
    B, cfg = 512, base.cfg
    ids = np.arange(B, dtype=np.int32)
    t0 = np.ones(B, dtype=np.float32)
    ns = np.full(B, 10, dtype=np.int32)
    dt = (-t0 / 10).astype(np.float32)
    out = torch.empty_like(fl.noise)
    rosa.rosa_denoise_batch_ex(fl.expert, ids, fl.noise, t0, dt, ns, out, None, None)
    torch.cuda.synchronize()
    big = out.cpu().numpy()
    pick = np.array([0, 255, 511], dtype=np.int32)
    small_out = torch.empty((3,) + tuple(fl.noise.shape[1:]), dtype=torch.float32, device=fl.noise.device)
    vel = torch.empty((10, 3) + tuple(fl.noise.shape[1:]), dtype=torch.float32, device=fl.noise.device)
    rosa.rosa_denoise_batch_ex(fl.expert, pick, fl.noise[pick.tolist()].contiguous(), t0[:3], dt[:3], ns[:3],
                               small_out, vel, None)
    torch.cuda.synchronize()
    small = small_out.cpu().numpy()
    # P2 on the GPU.  The RMSNorm statistics no longer depend on the tile width; what is left is the attention
    # work split: at B = 3 the planner cuts items between CTAs (a segment starts its own running maximum, so P is
    # rounded to bf16 against another reference, and the partial result is handed over in 16 bits), at B = 512 it
    # does not.  Measured 2.2e-3 over 18 layers x 10 steps here; 1e-3 holds wherever the plans agree (tests below).
    assert np.abs(big[pick] - small).max() <= 3e-3
    # robot 511 against the oracle
    row = cfg.n_kv_heads * cfg.head_dim
    sl = slice(511 * 816, 512 * 816)
    pk = np.stack([t[sl].float().cpu().numpy().reshape(816, cfg.n_kv_heads, cfg.head_dim) for t in fl.k])
    pv = np.stack([t[sl].float().cpu().numpy().reshape(816, cfg.n_kv_heads, cfg.head_dim) for t in fl.v])
    want_x, want_v = O.denoise_batch(cfg, base.weights, [pk], [pv], fl.noise[511:512].cpu().numpy(), t0[:1], dt[:1],
                                     ns[:1], return_velocity=True)
    compare("cfg4-B512-robot511", big[511:512], [vel[k, 2:3].cpu().numpy() for k in range(10)], want_x, want_v)
    assert row == 256
    fl.close()


def edge_case(lens, seed=21, n_steps=3):
    return cases.build_case("edge", seed, MINI, bf16=True, prefix_lens=list(lens), n_steps=n_steps)


def test_edge_prefix_lengths():
    """L = 0 (self-attention only, R8), 1, and lengths around the 64-key block boundary."""
    case = edge_case([0, 1, 63, 64, 65, 127, 128, 129, 200])
    lc = LoadedCase(case)
    check_against_oracle(case, lc, list(range(case.batch)), "edge-lens")
    lc.close()


def test_edge_one_block_segment_after_an_odd_block_count():
    """Attention work lists in which a one-block item (L = 0: the robot's own tokens only) follows a three-block item
    on EVERY CTA: the softmax warps split the key blocks by parity of the CTA-wide block count, so here the set that
    owns the thread issuing the bulk copies has no block in the second segment: the kernel then settles the staging
    tile ahead of the drain, behind a barrier of all eight warps, and that set's row sums are empty (0 at reference
    -inf).  The plan is checked on the host first so that the test keeps meaning what it says if the planner changes."""
    lens = [100] * 37 + [0] * 37            # 4 tiles per robot (H = 50): 148 + 148 items on 148 CTAs
    offs, segs = rosa.rosa_debug_attn_plan(MINI.horizon, lens, 148)
    special = 0
    for c in range(148):
        g = 0
        for i in range(offs[c], offs[c + 1]):
            n = int(segs[i][3] - segs[i][2])
            special += n == 1 and (g & 1) == 1
            g += n
    assert special >= 100, special
    case = edge_case(lens, seed=29, n_steps=2)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, list(range(case.batch)), "edge-one-block-after-odd", sample=[0, 17, 36, 37, 55, 73])
    lc.close()


def test_edge_single_step_and_single_robot():
    case = edge_case([100], n_steps=1)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, [0], "edge-1x1")
    lc.close()


def test_p2_batch_invariance_p3_permutation_and_aliasing():
    case = edge_case([70, 150, 33, 90, 64])
    lc = LoadedCase(case)
    full, _ = lc.run()
    want, _ = O.denoise_case(case)
    perm = [3, 0, 4, 2, 1]
    got_perm, _ = lc.run(robots=perm)
    assert np.abs(got_perm - full[perm]).max() <= 1e-3           # P3
    solo, _ = lc.run(robots=[2])
    assert np.abs(solo[0] - full[2]).max() <= 1e-3               # P2
    assert rel_l2(got_perm, want[perm]) <= TOL_ACT_REL
    # noise and out_actions may alias (rosa.h)
    buf = torch.from_numpy(case.noise.copy()).cuda()
    rosa.rosa_denoise_batch(lc.expert, np.arange(5, dtype=np.int32), buf, case.t_start, case.n_steps, buf)
    torch.cuda.synchronize()
    assert np.array_equal(buf.cpu().numpy(), full)               # P13 as well: bitwise equal to the first run
    lc.close()


def test_p13_determinism_bitwise():
    case = edge_case([300, 10, 77])
    lc = LoadedCase(case)
    a, va = lc.run(want_velocity=True)
    b, vb = lc.run(want_velocity=True)
    assert np.array_equal(a, b) and np.array_equal(va, vb)
    lc.close()


def test_p12_softmax_stress_online_rescaling():
    """Peaked softmax: three prefix keys per robot are scaled so that their logits have standard
    deviation ~4, ~8 and ~13 (the N(0,1) bulk has ~0.64), placed in increasing order along the
    key stream, so for many query rows the running maximum grows by more than 2^8 between key
    blocks and the lazy O-rescale path of the attention kernel runs.  (Larger scales exceed the
    velocity tolerance by construction: q is a bf16 operand, so a logit s carries an absolute
    error of about 1e-3 |s|, which softmax turns into a relative error of the same size.)"""
    case = edge_case([190, 260], seed=23, n_steps=2)
    for i in range(case.batch):
        k = cases.bf16_bits_to_f32(case.prefix_k[i]).copy()
        L = k.shape[1]
        for j, s in ((70, 6.0), (L // 2 + 40, 12.0), (L - 3, 20.0)):
            k[:, j] *= s
        case.prefix_k[i] = cases.f32_to_bf16_bits(k)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, [0, 1], "p12-softmax-stress")
    lc.close()


def test_p4_zero_output_projection_and_p5_constant_velocity():
    case = edge_case([50, 90])
    case.weights["w_out"] = np.zeros_like(case.weights["w_out"])
    case.weights["b_out"] = np.zeros_like(case.weights["b_out"])
    lc = LoadedCase(case)
    x, _ = lc.run()
    assert np.array_equal(x, case.noise)                          # P4: exactly unchanged
    lc.close()
    c = cases.round_bf16(np.linspace(-1, 1, MINI.action_dim).astype(np.float32))
    case.weights["b_out"] = c
    case.t_start = np.array([1.0, 0.5], dtype=np.float32)
    case.n_steps = np.array([4, 3], dtype=np.int32)
    case.dt = (-case.t_start / case.n_steps).astype(np.float32)
    lc = LoadedCase(case)
    x, _ = lc.run()
    want = case.noise - case.t_start[:, None, None] * c[None, None, :]   # x0 + n dt c = x0 - t0 c
    assert np.abs(x - want).max() <= 1e-5
    lc.close()


def test_p6_step_composition_via_ex():
    case = edge_case([120, 60], n_steps=10)
    lc = LoadedCase(case)
    full, _ = lc.run()
    ids = np.arange(2, dtype=np.int32)
    x = torch.from_numpy(case.noise).cuda()
    dt = np.full(2, -0.1, dtype=np.float32)
    rosa.rosa_denoise_batch_ex(lc.expert, ids, x, np.full(2, 1.0, np.float32), dt, np.full(2, 4, np.int32), x)
    rosa.rosa_denoise_batch_ex(lc.expert, ids, x, np.full(2, 0.6, np.float32), dt, np.full(2, 6, np.int32), x)
    torch.cuda.synchronize()
    # not bitwise: float32(0.6) != 1 + 4 * float32(-0.1) (3e-8 apart), which moves the highest time
    # frequency (2 pi / 4e-3) by 5e-5 rad and flips a few 16-bit operand roundings downstream
    assert np.abs(x.cpu().numpy() - full).max() <= 1e-3
    want, _ = O.denoise_case(case)
    assert rel_l2(x.cpu().numpy(), want) <= TOL_ACT_REL and np.abs(x.cpu().numpy() - want).max() <= TOL_ACT_ABS
    lc.close()


def test_rebind_unbind_and_error_codes():
    case = edge_case([40, 80, 120])
    lc = LoadedCase(case)
    e = lc.expert
    noise = torch.from_numpy(case.noise).cuda()
    out = torch.empty_like(noise)
    ns = case.n_steps

    def status(fn):
        with pytest.raises(rosa.RosaError) as ei:
            fn()
        return ei.value.status

    assert status(lambda: rosa.rosa_denoise_batch(e, [0, 0, 1], noise, None, ns, out)) == rosa.ROSA_ERR_INVALID_ARG
    assert status(lambda: rosa.rosa_denoise_batch(e, [0, 1, 7], noise, None, ns, out)) == rosa.ROSA_ERR_INVALID_ARG
    assert status(lambda: rosa.rosa_denoise_batch(e, [0, 1, 2], noise, None, [1, 0, 1], out)) == rosa.ROSA_ERR_INVALID_ARG
    assert status(lambda: rosa.rosa_denoise_batch(e, [0, 1, 2], noise, None, [1, 99, 1], out)) == rosa.ROSA_ERR_CAPACITY
    rosa.rosa_prefix_kv_unbind(e, 1)
    assert status(lambda: rosa.rosa_denoise_batch(e, [0, 1, 2], noise, None, ns, out)) == rosa.ROSA_ERR_UNBOUND_ROBOT
    k0 = [t for t in lc.kv_buffers[:MINI.layers]]
    assert status(lambda: rosa.rosa_prefix_kv_bind(e, 1, k0, k0, 10 ** 6)) == rosa.ROSA_ERR_CAPACITY
    # re-bind robot 1 to robot 0's prefix: its output must now equal robot 0's given the same noise
    row = MINI.n_kv_heads * MINI.head_dim
    kl, vl = lc.kv_buffers[:MINI.layers], lc.kv_buffers[MINI.layers:]
    rosa.rosa_prefix_kv_bind(e, 1, [t.data_ptr() for t in kl], [t.data_ptr() for t in vl], 40)
    n2 = torch.from_numpy(np.stack([case.noise[0], case.noise[0]])).cuda()
    o2 = torch.empty_like(n2)
    rosa.rosa_denoise_batch(e, [0, 1], n2, None, ns[:2], o2)
    torch.cuda.synchronize()
    o2 = o2.cpu().numpy()
    assert np.abs(o2[0] - o2[1]).max() <= 1e-3
    assert row == 256
    lc.close()


def _gemm_operands(M, N, K, fp16, seed):
    """Seeded operands that both formats represent exactly (bf16-rounded values inside the fp16 normal range)."""
    rng = np.random.default_rng(seed)
    a = cases.round_bf16(rng.standard_normal((M, K), dtype=np.float32))
    w = cases.round_bf16(rng.standard_normal((N, K), dtype=np.float32) * 0.05)
    w[np.abs(w) < 2.0 ** -14] = 0.0                      # below the fp16 normal range: not exact in fp16
    if fp16:
        A = torch.from_numpy(a.astype(np.float16).view(np.int16)).cuda()
        W = torch.from_numpy(w.astype(np.float16).view(np.int16)).cuda()
    else:
        A = torch.from_numpy(cases.f32_to_bf16_bits(a).view(np.int16)).cuda()
        W = torch.from_numpy(cases.f32_to_bf16_bits(w).view(np.int16)).cuda()
    return a, w, A, W


@pytest.mark.parametrize("M,N,K", [(1, 64, 64), (127, 128, 192), (129, 256, 1024), (400, 2560, 1024),
                                   (3200, 1024, 4096), (333, 8192, 1024), (3200, 1024, 2048)])
def test_tcgen05_gemm_unit(M, N, K):
    """C = A W^T through the tcgen05/TMA kernel the library picks, against numpy fp64 on the same bf16 operand values."""
    a, w, A, W = _gemm_operands(M, N, K, 0, M * 7 + N + K)
    C = torch.zeros((M, N), dtype=torch.float32, device="cuda")
    rosa.rosa_debug_gemm(1, M, N, K, A, W, C)
    torch.cuda.synchronize()
    want = a.astype(np.float64) @ w.astype(np.float64).T
    got = C.cpu().numpy()
    assert np.abs(got - want).max() <= 2e-5 * K ** 0.5 * 4 + 1e-6, np.abs(got - want).max()


PAIR_WIDTHS = (256, 224, 192, 160, 128, 96, 64)


@pytest.mark.parametrize("epi", [rosa.EPI_STORE_F32, rosa.EPI_BIAS_F32, rosa.EPI_RESID])
@pytest.mark.parametrize("pair,bn", [(1, b) for b in PAIR_WIDTHS] + [(0, 256), (0, 128), (0, 64)])
def test_tcgen05_gemm_every_width_and_epilogue(epi, pair, bn):
    """Every N-tile width of the CTA-pair kernel (and the three of the single-CTA kernel) x every fp32 epilogue of
    the path (plain store, + bias, + residual), against numpy fp64 on the same 16-bit operands: the fp32 result,
    the 16-bit copy of it (A operand of the next GEMM) and the per-32-column sums of squares (fused RMSNorm, a2).
    M has a ragged last row block; N = 1024, so the widths 224 / 192 / 160 / 96 end in a masked column tile."""
    M, N, K = (333 if pair else 100), 1024, 512
    fp16 = 1 if epi != rosa.EPI_STORE_F32 else 0          # the path's operand format (R19'); the plain store runs bf16
    a, w, A, W = _gemm_operands(M, N, K, fp16, 1000 + bn + 7 * epi + pair)
    rng = np.random.default_rng(bn + epi)
    c0 = rng.standard_normal((M, N), dtype=np.float32)
    bias = rng.standard_normal(N, dtype=np.float32)
    C = torch.from_numpy(c0.copy()).cuda()
    kw = {}
    if epi != rosa.EPI_STORE_F32:
        h16 = torch.zeros((M, N), dtype=torch.int16, device="cuda")
        ssq = torch.full((M, N // 32), -1.0, dtype=torch.float32, device="cuda")
        kw = dict(h16=h16, ssq=ssq, bias=torch.from_numpy(bias).cuda() if epi == rosa.EPI_BIAS_F32 else None)
    rosa.rosa_debug_gemm(1, M, N, K, A, W, C, epi=epi, pair=pair, bn=bn, fp16=fp16, **kw)
    torch.cuda.synchronize()
    want = a.astype(np.float64) @ w.astype(np.float64).T
    if epi == rosa.EPI_BIAS_F32:
        want = want + bias.astype(np.float64)
    if epi == rosa.EPI_RESID:
        want = want + c0.astype(np.float64)
    got = C.cpu().numpy()
    err = float(np.abs(got - want).max())
    print(f"[gemm pair={pair} bn={bn} epi={epi}] max-abs {err:.3e}")
    assert err <= 2e-5 * K ** 0.5 * 4 + 1e-6 + 4e-7 * np.abs(want).max(), err
    if epi != rosa.EPI_STORE_F32:
        got16 = h16.cpu().numpy().view(np.float16).astype(np.float32)
        assert np.array_equal(got16, got.astype(np.float16).astype(np.float32))        # RNE of the fp32 value written
        want_ssq = (got.astype(np.float64) ** 2).reshape(M, N // 32, 32).sum(-1)
        got_ssq = ssq.cpu().numpy()
        assert np.abs(got_ssq - want_ssq).max() <= 1e-5 * want_ssq.max()


def test_bf16_operand_mode_measured(monkeypatch):
    """Reading R19': with bf16 weight-GEMM operands (ROSA_GEMM_DTYPE=bf16) the final actions
    stay inside their tolerances, but the per-step velocity error is several times that of the default
    fp16 operands and does not meet 5e-3; the numbers are printed for profiles/r1_numerics.md."""
    case = cases.make_case(1)
    robots = list(range(8))
    want_x, want_v = O.denoise_case(case, robots=robots, return_velocity=True)
    res = {}
    for mode in ("fp16", "bf16"):
        monkeypatch.setenv("ROSA_GEMM_DTYPE", mode)
        lc = LoadedCase(case)
        got_x, got_v = lc.run(robots=robots, want_velocity=True)
        lc.close()
        res[mode] = (float(np.abs(got_x - want_x).max()), rel_l2(got_x, want_x),
                     max(rel_l2(got_v[k], want_v[k]) for k in range(len(want_v))))
        print(f"[cfg1 {mode} operands] actions max-abs {res[mode][0]:.3e} rel-L2 {res[mode][1]:.3e}; "
              f"velocity rel-L2 max {res[mode][2]:.3e}")
    assert res["bf16"][0] <= TOL_ACT_ABS and res["bf16"][1] <= TOL_ACT_REL
    assert res["fp16"][2] <= TOL_VEL_REL
    assert res["fp16"][2] < res["bf16"][2]


# ------------------------------------------------------------------ adaptive-norm variant (reading R25)
def test_adarms_variant_pi0_shapes():
    """pi0-scale widths (d 1024, F 4096, 8q/1kv x 256), 3 layers, ragged prefixes: CTA-pair GEMMs (M = 300)."""
    case = cases.make_adarms_case("pi0", batch=6, layers=3)
    assert case.cfg.time_conditioning == 1 and case.cfg.d_model == 1024
    lc = LoadedCase(case)
    assert rosa.rosa_kernel_family(lc.expert) == 1
    got_x, _ = check_against_oracle(case, lc, list(range(6)), "adarms-pi0-b6")
    again, _ = lc.run(robots=list(range(6)))
    assert np.array_equal(got_x, again)                                   # P13
    # M = 100 rows: the single-CTA GEMM kernels; batch invariance against the batched run (P2)
    sub, _ = check_against_oracle(case, lc, [4, 1], "adarms-pi0-b2")
    assert np.abs(sub - got_x[[4, 1]]).max() <= 1e-3
    one, _ = check_against_oracle(case, lc, [3], "adarms-pi0-b1")         # one robot: one row of cond / modulation
    assert np.abs(one[0] - got_x[3]).max() <= 1e-3
    lc.close()


def test_adarms_variant_mixed_steps_and_gate_wiring():
    """Narrow model, robots at different denoise stages (shrinking active set), then the closed forms."""
    from dataclasses import replace
    cfg = replace(MINI, time_conditioning=1)
    case = cases.build_case("adarms-mini-mix", 23, cfg, bf16=True, draw_lens=(0, 200), batch=5, cfg3_mix=True)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, list(range(5)), "adarms-mini-mix")
    lc.close()
    # zero gate: blocks are the identity, v = (h0 r)(1 + scale) + shift through W_out: oracle closed form pinned on CPU
    d = cfg.d_model
    for k in ("b_mod_attn", "b_mod_mlp"):
        case.weights[k] = [np.concatenate([b[:2 * d], np.zeros(d, np.float32)]) for b in case.weights[k]]
    for k in ("w_mod_attn", "w_mod_mlp"):
        case.weights[k] = [np.concatenate([w[:2 * d], np.zeros((d, d), np.float32)]) for w in case.weights[k]]
    lc = LoadedCase(case)
    got_x, got_v = lc.run(want_velocity=True)
    want_x, want_v = O.denoise_case(case, return_velocity=True)
    compare("adarms-zero-gate", got_x, got_v, want_x, want_v)
    lc.close()


def test_adarms_variant_needs_tcgen05_shapes():
    case = cases.make_adarms_case("tiny")
    with pytest.raises(rosa.RosaError) as ei:
        LoadedCase(case)
    assert ei.value.status == rosa.ROSA_ERR_UNSUPPORTED


def test_adarms_variant_full_depth_cfg1_sampled():
    """All 18 layers and 10 Euler steps of the cfg1 workload on the variant; oracle on two of the eight robots.

    Final actions: north_star tolerances.  Per-step velocity: 5e-3 holds when both sides evaluate v at the SAME x
    (each Euler step launched from the oracle's x_k: the arithmetic error of one velocity evaluation).  Along the
    free-running trajectory the variant's velocity is more sensitive to the accumulated difference in x than the
    base model's (x enters the residual stream through W_in alone, R25), so there the bound is 1e-2, stated here."""
    case = cases.make_case(1, time_conditioning=1)
    assert case.cfg.layers == 18 and case.batch == 8
    lc = LoadedCase(case)
    sample = [0, 5]
    got_x, got_v = lc.run(want_velocity=True)
    want_x, want_v = O.denoise_case(case, robots=sample, return_velocity=True)
    free = [rel_l2(got_v[k][sample], want_v[k]) for k in range(len(want_v))]
    print(f"[adarms-cfg1 free-running] actions max-abs {np.abs(got_x[sample] - want_x).max():.3e} rel-L2 "
          f"{rel_l2(got_x[sample], want_x):.3e}; velocity rel-L2 per step {[f'{v:.2e}' for v in free]}")
    assert np.abs(got_x[sample] - want_x).max() <= TOL_ACT_ABS and rel_l2(got_x[sample], want_x) <= TOL_ACT_REL
    assert free[0] <= TOL_VEL_REL and max(free) <= 1e-2
    # teacher-forced: step k from the oracle's x_k at t_k
    dev = lc.device
    ids = np.asarray(sample, dtype=np.int32)
    xk = case.noise[sample].astype(np.float64)
    forced = []
    for k in range(len(want_v)):
        x_in = torch.from_numpy(xk.astype(np.float32)).to(dev)
        out = torch.empty_like(x_in)
        vel = torch.empty((1,) + tuple(x_in.shape), dtype=torch.float32, device=dev)
        t_k = (case.t_start[sample] + k * case.dt[sample]).astype(np.float32)
        rosa.rosa_denoise_batch_ex(lc.expert, ids, x_in, t_k, case.dt[sample], np.ones(len(sample), np.int32), out, vel, None)
        torch.cuda.synchronize()
        forced.append(rel_l2(vel[0].cpu().numpy(), want_v[k]))
        xk = xk + case.dt[sample].astype(np.float64)[:, None, None] * want_v[k]
    print(f"[adarms-cfg1 same-x] velocity rel-L2 per step max {max(forced):.3e}")
    assert max(forced) <= TOL_VEL_REL, forced
    lc.close()


def test_soak_random_batch_compositions_are_reproducible():
    """~10 s of back-to-back calls with random batch sizes, robot subsets and per-robot step counts on the cfg2
    fleet (every call replays or captures a graph keyed by (batch, max steps)): each call is issued twice and must
    agree bitwise (P13: no order-dependent arithmetic, no race between the graph's kernels), stay finite, and robots
    that run all 10 steps must match their single-robot result (P2)."""
    import time
    case = cases.make_case(2)
    lc = LoadedCase(case)
    single = {r: lc.run(robots=[r])[0][0] for r in (0, 13, 63)}
    rng = np.random.default_rng(7)
    t_end, calls = time.time() + 10.0, 0
    while time.time() < t_end:
        b = int(rng.choice([1, 2, 3, 5, 8, 13, 21, 34, 50, 64]))
        idx = rng.permutation(64)[:b].astype(np.int32)
        ns = rng.integers(1, 11, size=b).astype(np.int32)
        tst = np.ones(b, np.float32)
        dt = (-tst / ns).astype(np.float32)
        noise = torch.from_numpy(case.noise[idx]).to(lc.device)
        o1, o2 = torch.empty_like(noise), torch.empty_like(noise)
        rosa.rosa_denoise_batch_ex(lc.expert, idx, noise, tst, dt, ns, o1, None, None)
        rosa.rosa_denoise_batch_ex(lc.expert, idx, noise, tst, dt, ns, o2, None, None)
        torch.cuda.synchronize()
        a = o1.cpu().numpy()
        assert np.all(np.isfinite(a)) and np.array_equal(a, o2.cpu().numpy()), (b, idx[:4], ns[:4])
        for j, r in enumerate(idx):
            if int(r) in single and ns[j] == 10:   # 3e-3: the attention work split differs between a lone robot and a batch
                assert np.abs(a[j] - single[int(r)]).max() <= 3e-3
        calls += 2
    print(f"[soak] {calls} calls, {rosa.rosa_debug_graph_captures(lc.expert)} graphs captured")
    assert calls >= 100
    lc.close()


def test_bucketed_graphs_no_capture_after_warmup():
    """Graphs are keyed by (batch bucket, max n_steps): after one call per key, 200 random (batch, n) pairs replay
    captured graphs only (no capture + instantiate on the request path), and a smaller batch run through its
    bucket's graph gives each robot the result of its own run."""
    case = edge_case([70, 150, 33, 90, 64, 200, 10, 129, 300, 17, 64, 65, 5], n_steps=3)
    lc = LoadedCase(case, max_steps=4)
    B = case.batch
    solo = {r: lc.run(robots=[r])[0][0] for r in (0, 7, 12)}
    noise_all = torch.from_numpy(case.noise).to(lc.device)

    def call(idx, ns):
        idx = np.asarray(idx, dtype=np.int32)
        ns = np.asarray(ns, dtype=np.int32)
        t0 = np.ones(len(idx), np.float32)
        out = torch.empty((len(idx),) + tuple(noise_all.shape[1:]), dtype=torch.float32, device=lc.device)
        rosa.rosa_denoise_batch_ex(lc.expert, idx, noise_all[idx.tolist()].contiguous(), t0, (-t0 / ns).astype(np.float32), ns, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    for bucket in (1, 2, 4, 8, 13):                     # warm-up: one call per (bucket, n)
        for n in (1, 2, 3, 4):
            call(list(range(bucket)), [n] * bucket)
    warm = rosa.rosa_debug_graph_captures(lc.expert)
    assert warm <= 5 * 4
    rng = np.random.default_rng(11)
    for _ in range(200):
        b = int(rng.integers(1, B + 1))
        idx = rng.permutation(B)[:b]
        ns = rng.integers(1, 5, size=b)
        out = call(idx, ns)
        assert np.all(np.isfinite(out))
        for j, r in enumerate(idx):
            if int(r) in solo and ns[j] == 3:
                assert np.abs(out[j] - solo[int(r)]).max() <= 1e-3
    assert rosa.rosa_debug_graph_captures(lc.expert) == warm
    lc.close()


def test_fp16_range_of_the_residual_stream():
    """The default operand format keeps a 16-bit fp16 copy of the UN-normalised residual h as the A operand of the
    QKV / gate-up GEMMs (R23); fp16 ends at 65504.  The library's contract (include/rosa.h): the copy
    SATURATES at +-65504, so an out-of-range residual gives finite, clipped results, never inf / NaN; with
    ROSA_GEMM_DTYPE=bf16 the operand has the range of fp32 and the same model stays within the bf16-mode accuracy.
    Here b_t2 (the bias of the embedding MLP's second layer, which enters h0 directly) is scaled so that |h| reaches
    ~1e5 on some channels while everything downstream is scale-invariant (RMSNorm)."""
    import os
    case = edge_case([40, 90], n_steps=2)
    b = case.weights["b_t2"].copy()
    b[::7] = cases.round_bf16(np.full_like(b[::7], 1.0e5))
    case.weights["b_t2"] = b
    want_x, want_v = O.denoise_case(case, return_velocity=True)
    lc = LoadedCase(case)
    got_x, got_v = lc.run(want_velocity=True)
    lc.close()
    assert np.all(np.isfinite(got_x)) and np.all(np.isfinite(got_v))          # saturated, not inf / NaN
    print(f"[fp16-range fp16 operands] actions rel-L2 {rel_l2(got_x, want_x):.3e} (clipped channels)")
    old = os.environ.get("ROSA_GEMM_DTYPE")
    os.environ["ROSA_GEMM_DTYPE"] = "bf16"
    try:
        lc = LoadedCase(case)
        got_x, got_v = lc.run(want_velocity=True)
        lc.close()
    finally:
        if old is None:
            del os.environ["ROSA_GEMM_DTYPE"]
        else:
            os.environ["ROSA_GEMM_DTYPE"] = old
    err = rel_l2(got_x, want_x)
    print(f"[fp16-range bf16 operands] actions rel-L2 {err:.3e}")
    assert np.all(np.isfinite(got_x)) and err <= TOL_ACT_REL


def test_adarms_variant_needs_the_tcgen05_attention_shape():
    """time_conditioning = 1 with a head layout the tcgen05 attention kernel does not cover (16 query heads, 2 KV
    heads) is refused at create, not run through null tensor maps."""
    from dataclasses import replace
    cfg = replace(MINI, n_q_heads=16, n_kv_heads=2, time_conditioning=1)
    case = cases.build_case("adarms-bad-heads", 3, cfg, bf16=True, prefix_lens=[20], n_steps=1)
    with pytest.raises(rosa.RosaError) as ei:
        LoadedCase(case)
    assert ei.value.status == rosa.ROSA_ERR_UNSUPPORTED


# ------------------------------------------------------------------ the step before: prefix K/V production (R29)
def test_prefix_kv_produce_matches_oracle_and_feeds_the_loop():
    """rosa_prefix_kv_produce against O.prefix_kv element by element (ragged lengths: one token, a full 64-key block,
    rows that straddle the 128- and 256-row GEMM tiles), then the produced cache is bound and the whole denoise loop is
    compared with the oracle running on the oracle's own K/V."""
    lens = [1, 64, 200, 333]
    case = edge_case(lens, seed=29, n_steps=3)
    cfg = case.cfg
    d_p, row = 320, cfg.n_kv_heads * cfg.head_dim
    rng = np.random.default_rng(290)
    wk = [cases.round_bf16(rng.standard_normal((row, d_p), dtype=np.float32) / np.sqrt(d_p)) for _ in range(cfg.layers)]
    wv = [cases.round_bf16(rng.standard_normal((row, d_p), dtype=np.float32) / np.sqrt(d_p)) for _ in range(cfg.layers)]
    hidden = [[cases.round_bf16(rng.standard_normal((L, d_p), dtype=np.float32)) for _ in range(cfg.layers)] for L in lens]
    want = [[O.prefix_kv(cfg, hidden[i][l], wk[l], wv[l]) for l in range(cfg.layers)] for i in range(len(lens))]
    for i in range(len(lens)):   # what an exact producer would store: the oracle's K/V rounded to the cache's bf16
        case.prefix_k[i] = cases.f32_to_bf16_bits(np.stack([want[i][l][0] for l in range(cfg.layers)]).astype(np.float32))
        case.prefix_v[i] = cases.f32_to_bf16_bits(np.stack([want[i][l][1] for l in range(cfg.layers)]).astype(np.float32))
    lc = LoadedCase(case)
    dev = lc.device
    to_dev = lambda a: torch.from_numpy(cases.f32_to_bf16_bits(a).view(np.int16)).to(dev)
    wk_d, wv_d = [to_dev(w) for w in wk], [to_dev(w) for w in wv]
    keep = []
    for i, L in enumerate(lens):
        h_d = [to_dev(hidden[i][l]) for l in range(cfg.layers)]
        k_d = [torch.zeros((L, row), dtype=torch.int16, device=dev) for _ in range(cfg.layers)]
        v_d = [torch.zeros((L, row), dtype=torch.int16, device=dev) for _ in range(cfg.layers)]
        rosa.rosa_prefix_kv_produce(lc.expert, d_p, h_d, wk_d, wv_d, L, k_d, v_d)
        torch.cuda.synchronize()
        for l in range(cfg.layers):
            for got_t, ref, name in ((k_d[l], want[i][l][0], "K"), (v_d[l], want[i][l][1], "V")):
                got = cases.bf16_bits_to_f32(got_t.cpu().numpy().view(np.uint16)).reshape(L, cfg.n_kv_heads, cfg.head_dim)
                err, big = rel_l2(got, ref), float(np.abs(got - ref).max())
                # one bf16 rounding of the stored value (2^-9 relative per element) on top of fp32 accumulation
                assert err <= 3e-3 and big <= 2.0 ** -8 * float(np.abs(ref).max()) + 1e-6, (i, l, name, err, big)
        rosa.rosa_prefix_kv_bind(lc.expert, i, k_d, v_d, L, rosa.ROSA_BF16)
        keep.append((h_d, k_d, v_d))
    print(f"[prefix-kv-produce] lens {lens}: K/V within one bf16 rounding of the oracle")
    check_against_oracle(case, lc, list(range(len(lens))), "prefix-kv-produce -> denoise")
    with pytest.raises(rosa.RosaError) as ei:
        rosa.rosa_prefix_kv_produce(lc.expert, 100, keep[0][0], wk_d, wv_d, 1, keep[0][1], keep[0][2])   # d_prefix % 64 != 0
    assert ei.value.status == rosa.ROSA_ERR_UNSUPPORTED
    lc.close()
