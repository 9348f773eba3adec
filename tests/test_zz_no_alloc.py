"""rosa_linear_noalloc (include/rosa.h): the allocation-free entry point against the existing GEMM paths, two calls in a
row.  In a file of its own, collected last (the suite runs with pytest -x).  Passes alone in a fresh process and after
the other tests: it creates no expert and depends on nothing they leave behind."""
import numpy as np
import pytest
import torch

from paper_2607_01088_b200 import binding as rosa
from paper_2607_01088_b200 import build as rosa_build
from paper_2607_01088_b200 import cases

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    rosa_build.build()
    rosa.load()


def _operands(M, N, K, fp16, seed):
    """Seeded operands both formats represent exactly (bf16-rounded values inside the fp16 normal range)."""
    rng = np.random.default_rng(seed)
    a = cases.round_bf16(rng.standard_normal((M, K), dtype=np.float32))
    w = cases.round_bf16(rng.standard_normal((N, K), dtype=np.float32) * 0.05)
    w[np.abs(w) < 2.0 ** -14] = 0.0
    if fp16:
        A = torch.from_numpy(a.astype(np.float16).view(np.int16)).cuda()
        W = torch.from_numpy(w.astype(np.float16).view(np.int16)).cuda()
    else:
        A = torch.from_numpy(cases.f32_to_bf16_bits(a).view(np.int16)).cuda()
        W = torch.from_numpy(cases.f32_to_bf16_bits(w).view(np.int16)).cuda()
    return a, w, A, W


def _tol(K, want):
    # the bound of the GEMM unit tests (tests/test_parity_gpu.py): fp32 accumulation of K products in any order
    return 2e-5 * K ** 0.5 * 4 + 1e-6 + 4e-7 * float(np.abs(want).max())


def _one_call(M, N, K, epi, fp16, seed, family_ref):
    a, w, A, W = _operands(M, N, K, fp16, seed)
    rng = np.random.default_rng(seed + 1)
    c0 = rng.standard_normal((M, N), dtype=np.float32)
    bias = rng.standard_normal(N, dtype=np.float32)
    bias_d = torch.from_numpy(bias).cuda() if epi == rosa.EPI_BIAS_F32 else None
    got = torch.from_numpy(c0.copy()).cuda()
    rosa.rosa_linear_noalloc(M, N, K, A, W, got, epi=epi, fp16=fp16, bias=bias_d)
    # the existing path on the same operands: the tcgen05 GEMM with the same fused epilogue (family 1), or the
    # CUDA-core GEMM writing straight into the output (family 0, plain store only)
    ref = torch.from_numpy(c0.copy()).cuda()
    rosa.rosa_debug_gemm(family_ref, M, N, K, A, W, ref, epi=epi, fp16=fp16, bias=bias_d)
    torch.cuda.synchronize()
    want = a.astype(np.float64) @ w.astype(np.float64).T
    if epi == rosa.EPI_BIAS_F32:
        want = want + bias.astype(np.float64)
    if epi == rosa.EPI_RESID:
        want = want + c0.astype(np.float64)
    g, r = got.cpu().numpy(), ref.cpu().numpy()
    tol = _tol(K, want)
    assert np.all(np.isfinite(g))
    assert np.abs(g - r).max() <= 2 * tol, (np.abs(g - r).max(), tol)      # new entry point vs the existing path
    assert np.abs(g - want).max() <= tol, (np.abs(g - want).max(), tol)    # and both against numpy fp64
    return g


def test_noalloc_linear_matches_existing_paths_two_calls_in_a_row():
    # call 1: a residual GEMM of the pi0-scale expert's kind (d = 1024, K = 2048, 8 robots' token rows), fp16 operands,
    # at the scratch limit's order of magnitude (400 x 1024 of 2^20 elements), against the tcgen05 path
    first = _one_call(400, 1024, 2048, rosa.EPI_RESID, 1, 101, family_ref=1)
    # call 2, straight after, SMALLER and with another epilogue and format: stale contents of the shared scratch from
    # call 1 would show here if anything read what this call did not write
    free_before = torch.cuda.mem_get_info()[0]
    second = _one_call(130, 256, 320, rosa.EPI_BIAS_F32, 0, 202, family_ref=1)
    third = _one_call(37, 50, 23, rosa.EPI_STORE_F32, 0, 303, family_ref=0)  # ragged everything: the shape-generic kernels
    # (torch's caching allocator serves the test's own tensors: device memory in use by the process must not have grown)
    assert torch.cuda.mem_get_info()[0] >= free_before - (8 << 20)
    # the same call again gives the same bits (nothing of the earlier calls leaks through the scratch)
    again = _one_call(400, 1024, 2048, rosa.EPI_RESID, 1, 101, family_ref=1)
    assert np.array_equal(first, again)
    assert second.shape == (130, 256) and third.shape == (37, 50)


def test_noalloc_linear_rejects_sizes_beyond_the_static_scratch():
    M, N, K = 1025, 1024, 64            # M * N = 2^20 + 1024 > ROSA_NOALLOC_MAX_ELEMS
    assert M * N > rosa.ROSA_NOALLOC_MAX_ELEMS
    A = torch.zeros((M, K), dtype=torch.int16, device="cuda")
    W = torch.zeros((N, K), dtype=torch.int16, device="cuda")
    C = torch.zeros((M, N), dtype=torch.float32, device="cuda")
    with pytest.raises(rosa.RosaError) as ei:
        rosa.rosa_linear_noalloc(M, N, K, A, W, C)
    assert ei.value.status == rosa.ROSA_ERR_CAPACITY and "ROSA_NOALLOC_MAX_ELEMS" in str(ei.value)
    with pytest.raises(rosa.RosaError) as ei:
        rosa.rosa_linear_noalloc(4, 4, 4, A, W, C, epi=rosa.EPI_BIAS_F32)   # bias missing
    assert ei.value.status == rosa.ROSA_ERR_INVALID_ARG
    rosa.rosa_linear_noalloc(1024, 1024, K, A, W, C)                        # exactly at the limit: accepted
    torch.cuda.synchronize()
    assert not np.any(C[:1024].cpu().numpy())
