// Ragged-KV GQA attention on tcgen05 (step a5 of the path).
//
// One CTA per (robot p, tile of 16 action tokens).  All n_q = 8 query heads share the single KV
// head, so the tile's 16 tokens x 8 heads = 128 query rows form ONE M=128 operand against the
// robot's key/value stream [prefix K/V (L_p rows, from the bound cache) ; own k/v (H rows, from
// the qkv buffer)], walked in blocks of 64 keys:
//     S = Q K_blk^T           tcgen05.mma  M=128 N=64  K=256   Q is the A operand FROM TENSOR MEMORY
//     P = exp2(S*c - m_ref)   8 softmax warps, two per query row (32 keys each; both read all 64 scores for
//                             the row maximum), running (m_ref, partial l) in registers; P (bf16) is written
//                             back into tensor memory over S
//     O += P V_blk            tcgen05.mma  M=128 N=256 K=64    P is the A operand from tensor memory,
//                             V the MN-major B operand from shared memory
// Tensor memory (512 columns): O [0,256) | S/P double buffer [256,384) | Q [384,512).
// Shared memory holds nothing but rings of K (4 stages) and V (3 stages) blocks of 32 KB, one 3-D TMA each
// (per-robot tensor maps made at bind time bound the ragged length: rows >= L_p are zero-filled and masked),
// K issued one block ahead of V, L2 prefetches AT_PF blocks ahead.  Q passes through the last two K stages once.
// CTAs are issued longest prefix first (Tables::attn_order), so the second wave pairs long with short.
// O stays in TMEM for the whole key stream; it is rescaled only when a row maximum grows by more
// than 2^8 (lazy rescaling), which for N(0,1)-like logits almost never happens after block 0.
#include <cstdlib>

#include "device_math.cuh"
#include "rosa_internal.h"
#include "tc_common.cuh"

namespace rosa {

using namespace tc;

constexpr int AT_HD = 256;        // head_dim
constexpr int AT_ROWS = 128;      // query rows per CTA = AT_TOK tokens x 8 heads
constexpr int AT_TOK = 16;
constexpr int AT_KV = 64;         // keys per block
constexpr int AT_KST = 4;         // K stages (K runs one block further ahead than V)
constexpr int AT_ST = 3;          // V stages
constexpr int AT_PF = 6;          // L2 prefetch distance in blocks
constexpr int AT_THREADS = 320;   // warp 0 TMA, warp 1 MMA, warps 2..9 softmax/epilogue (two per TMEM lane quarter)
constexpr int AT_Q_BYTES = AT_ROWS * AT_HD * 2;     // 64 KB: 4 chunks [128 x 64] SW128
constexpr int AT_KV_BYTES = AT_KV * AT_HD * 2;      // 32 KB: 4 chunks [64 x 64] SW128
constexpr int AT_XCH_BYTES = 2 * 2 * AT_ROWS * 4;   // row-sum exchange between the two warps of a row (epilogue)
constexpr int AT_SMEM = (AT_KST + AT_ST) * AT_KV_BYTES + 256 + AT_XCH_BYTES;
constexpr float AT_RESCALE_THR = 8.0f;              // log2 units

// exp2 on the SFU without the denormal-range fix-up sequence of exp2f (inputs here are <= 2^8)
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct AttnMaps {
  CUtensorMap q;    // qkv buffer as [M tokens][8 heads][256]   box {64, 8, 16}
  CUtensorMap own;  // qkv buffer as (64 cols, M tokens, qkv_n/64 column chunks)   box {64, 64, 4}
};

__global__ void __launch_bounds__(AT_THREADS, 1)
k_attn_tc(const __grid_constant__ AttnMaps maps, const CUtensorMap* __restrict__ kv_maps, Dims dm, Tables tb,
          int layer, op16* __restrict__ o, int k_iter, int tiles_per_robot, int dbg, long long* __restrict__ trace) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const int p = tb.attn_order[blockIdx.x / tiles_per_robot], tt = blockIdx.x % tiles_per_robot;
  if (p * dm.H >= tb.m_active[k_iter]) return;
  const int robot = tb.ids[p], L = tb.rlen[robot];
  const int nbp = (L + AT_KV - 1) / AT_KV, nb = nbp + 1;  // prefix blocks + one block of own tokens

  const uint32_t base = smem_u32(smem_raw);  // 1024-byte aligned (SWIZZLE_128B tiles)
  if ((dbg & 16) && threadIdx.x == 0 && (blockIdx.x == 0 || blockIdx.x == 200)) trace[((blockIdx.x == 0 ? 0 : 1) * 16 + 7) * 32] = clock64();
  auto k_smem = [&](int s) { return base + (uint32_t)s * AT_KV_BYTES; };
  auto v_smem = [&](int s) { return base + (uint32_t)(AT_KST + s) * AT_KV_BYTES; };
  const uint32_t q_smem = k_smem(AT_KST - 2);  // Q passes through the last two K stages before block AT_KST-2 needs them
  const uint32_t bars = base + (AT_KST + AT_ST) * AT_KV_BYTES;
  auto k_full = [&](int s) { return bars + 8u * s; };
  auto k_empty = [&](int s) { return bars + 8u * (4 + s); };
  auto v_full = [&](int s) { return bars + 8u * (8 + s); };
  auto v_empty = [&](int s) { return bars + 8u * (8 + AT_ST + s); };
  auto s_full = [&](int s) { return bars + 8u * (4 * AT_ST + s + 2); };
  // p_full is double-buffered like S/P: the softmax warps may finish block i+1 before the MMA thread
  // has looked at block i's barrier, and a single barrier two phases ahead reads as "not yet"
  auto p_full = [&](int s) { return bars + 8u * (4 * AT_ST + 4 + s); };
  const uint32_t pv_done = bars + 8u * (4 * AT_ST + 6);
  const uint32_t q_full = bars + 8u * (4 * AT_ST + 7), q_done = bars + 8u * (4 * AT_ST + 8);
  const uint32_t tmem_slot = bars + 8u * (4 * AT_ST + 9);
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // measurement aid (ROSA_DBG bit 4): clock64 at pipeline events of CTAs 0 and 200 -> trace[slot][role][block]
  const int tslot = (dbg & 16) ? (blockIdx.x == 0 ? 0 : (blockIdx.x == 200 ? 1 : -1)) : -1;
#define AT_TRACE(role, blk) do { if (tslot >= 0 && (blk) < 32) trace[(tslot * 16 + (role)) * 32 + (blk)] = clock64(); } while (0)
  const CUtensorMap* kmap = kv_maps + ((size_t)robot * dm.layers + layer) * 2;
  const CUtensorMap* vmap = kmap + 1;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&maps.q);
    prefetch_tensormap(&maps.own);
    // the per-robot prefix maps live in global memory
    prefetch_tensormap(kmap);
    prefetch_tensormap(vmap);
    for (int s = 0; s < AT_KST; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), 1); }
    for (int s = 0; s < AT_ST; ++s) { mbar_init(v_full(s), 1); mbar_init(v_empty(s), 1); }
    mbar_init(s_full(0), 1); mbar_init(s_full(1), 1);
    mbar_init(p_full(0), 8); mbar_init(p_full(1), 8);  // one arrival per softmax warp
    mbar_init(pv_done, 1);
    mbar_init(q_full, 1);
    mbar_init(q_done, 8);
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  const uint32_t tmem_o = tmem_base;            // columns [0, 256): O accumulator
  const uint32_t tmem_s = tmem_base + 256;      // columns [256, 384): S (fp32) / P (bf16 pairs), 2 x 64
  const uint32_t tmem_q = tmem_base + 384;      // columns [384, 512): Q, 256 bf16 per row

  const int tok0 = p * dm.H + tt * AT_TOK;      // first token row of this tile in the qkv buffer
  pdl_wait();     // everything above overlapped the previous kernel's tail
  pdl_trigger();

  if (warp == 0) {
    {  // ------------------------------------------------ TMA producer (whole warp; one lane issues)
      // one TMA per 64-key block: 3-D maps (64 columns, rows, 4 column chunks) land as [chunk][row][128 B]
      auto prefetch_blk = [&](int i) {
        if (i < nbp) { tma_prefetch_3d(kmap, 0, i * AT_KV, 0); tma_prefetch_3d(vmap, 0, i * AT_KV, 0); }
      };
      auto load_k = [&](int i) {
        const int s = i % AT_KST;
        if (i == AT_KST - 2) mbar_wait(q_done, 0);  // Q has left the last two K stages
        mbar_wait_idle(k_empty(s), ((i / AT_KST) & 1) ^ 1);
        if (elect_one()) {
          mbar_expect_tx(k_full(s), AT_KV_BYTES);
          if (i == nbp) tma_load_3d(k_smem(s), &maps.own, k_full(s), 0, p * dm.H, dm.q_n / 64);
          else tma_load_3d(k_smem(s), kmap, k_full(s), 0, i * AT_KV, 0);
          AT_TRACE(0, i);
        }
        __syncwarp();
      };
      // K(0) first: it usually comes from HBM (the prefix cache is streamed once per layer) while Q was just
      // written by the QKV GEMM and hits L2, so queueing Q's 64 KB ahead of it delayed the first S MMA
      load_k(0);
      if (elect_one()) {
        mbar_expect_tx(q_full, AT_Q_BYTES);
        for (int c = 0; c < 4; ++c) tma_load_3d(q_smem + c * (AT_ROWS * 128), &maps.q, q_full, c * 64, 0, tok0);
      }
      __syncwarp();
      for (int i = 0; i < nb; ++i) {  // K runs one block ahead of V: it is needed a whole softmax earlier
        if (i + 1 < nb) load_k(i + 1);
        const int s = i % AT_ST;
        mbar_wait_idle(v_empty(s), ((i / AT_ST) & 1) ^ 1);
        if (elect_one()) {
          mbar_expect_tx(v_full(s), AT_KV_BYTES);
          if (i == nbp) tma_load_3d(v_smem(s), &maps.own, v_full(s), 0, p * dm.H, (dm.q_n + AT_HD) / 64);
          else tma_load_3d(v_smem(s), vmap, v_full(s), 0, i * AT_KV, 0);
          // L2 prefetches go out only after everything the first MMAs wait for (Q, K0, K1, V0) is in flight
          if (i == 0) for (int j = 2; j < AT_PF; ++j) prefetch_blk(j);
          prefetch_blk(i + AT_PF);
          AT_TRACE(1, i);
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    {  // ------------------------------------------------ MMA issuer (whole warp; one lane issues)
      constexpr uint32_t idesc_s = make_idesc_bf16(AT_ROWS, AT_KV);
      constexpr uint32_t idesc_o = make_idesc_bf16(AT_ROWS, AT_HD, /*b_mn_major=*/true);
      auto issue_s = [&](int i) {  // S(i) = Q K_i^T into S buffer i&1 (overwrites P(i-2), consumed by PV(i-2))
        const int s = i % AT_KST;
        mbar_wait(k_full(s), (i / AT_KST) & 1);
        tc_fence_after();
        if (elect_one()) {
          if (!(dbg & 8)) {
#pragma unroll
            for (int kk = 0; kk < AT_HD / 16; ++kk) {
              const uint32_t ka = k_smem(s) + (kk >> 2) * (AT_KV * 128) + (kk & 3) * 32;
              umma_bf16_ts(tmem_s + (i & 1) * AT_KV, tmem_q + kk * 8, make_sdesc_k128(ka), idesc_s, kk != 0);
            }
          }
          umma_commit(k_empty(s));
          umma_commit(s_full(i & 1));
          AT_TRACE(2, i);
        }
        __syncwarp();
      };
      mbar_wait(q_done, 0);
      tc_fence_after();
      AT_TRACE(6, 0);
      issue_s(0);
      for (int i = 0; i < nb; ++i) {
        if (i + 1 < nb) issue_s(i + 1);
        const int s = i % AT_ST;
        mbar_wait(v_full(s), (i / AT_ST) & 1);
        mbar_wait(p_full(i & 1), (i >> 1) & 1);
        tc_fence_after();
        if (elect_one()) {
          if (!(dbg & 8)) {
#pragma unroll
            for (int kk = 0; kk < AT_KV / 16; ++kk) {
              // A = P [128 x 64] bf16 in TMEM (8 columns per 16 keys); B = V block, MN-major: 4 hd chunks
              // 8192 B apart (LBO), 8-key groups 1024 B apart (SBO); 16 keys per MMA = 2048 B
              const uint64_t b_desc = make_sdesc_mn128(v_smem(s) + kk * 2048, AT_KV * 128, 1024);
              umma_bf16_ts(tmem_o, tmem_s + (i & 1) * AT_KV + kk * 8, b_desc, idesc_o, (i | kk) != 0);
            }
          }
          umma_commit(v_empty(s));
          umma_commit(pv_done);
          AT_TRACE(3, i);
        }
        __syncwarp();
      }
    }
  } else {
    // ---------------------------------------------------------- softmax + epilogue warps (2..9)
    // Two warps per TMEM lane quarter: a query row's 64 scores of a block are split 32 / 32 between
    // warp w (half 0) and warp w + 4 (half 1).  Both read all 64 scores for the row maximum
    // (so both take the same rescale decision) and keep separate partial row sums until the end.
    const int q = warp & 3, half = (warp - 2) >> 2;
    const int r = q * 32 + lane;                       // query row of this thread
    const uint32_t lane_off = (uint32_t)(q * 32) << 16;
    float* xch = reinterpret_cast<float*>(smem_raw + ((AT_KST + AT_ST) * AT_KV_BYTES + 256));  // [2 buffers][2 halves][128]
    {  // Q: shared memory (SW128: 4 chunks of [128 rows x 128 B]) -> tensor memory, thread = row, 2 chunks per half
      mbar_wait(q_full, 0);
#pragma unroll 1
      for (int cc = half * 2; cc < half * 2 + 2; ++cc) {
        uint32_t w[32];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const uint32_t addr = q_smem + cc * (AT_ROWS * 128) + r * 128 + ((j ^ (r & 7)) << 4);
          asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                       : "=r"(w[4 * j]), "=r"(w[4 * j + 1]), "=r"(w[4 * j + 2]), "=r"(w[4 * j + 3]) : "r"(addr));
        }
        tmem_st32(tmem_q + lane_off + cc * 32, w);
      }
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(q_done);
    }
    const float c_log2 = rsqrtf((float)AT_HD) * 1.4426950408889634f;  // (1/sqrt(hd)) * log2(e)
    float m_ref = -INFINITY, l_sum = 0.f;                             // m_ref in log2 units; l_sum: this half's part
    for (int i = 0; i < nb; ++i) {
      const int sb = i & 1;
      const int n_tot = i == nbp ? dm.H : min(AT_KV, L - i * AT_KV);
      const int n_valid = n_tot - half * 32, n_other = n_tot - (half ^ 1) * 32;  // valid columns of this / the other half
      mbar_wait(s_full(sb), (i >> 1) & 1);
      tc_fence_after();
      if (threadIdx.x == 64) AT_TRACE(4, i);
      // Both warps of a row read all 64 scores for the row maximum (so they take the same rescale
      // decision without an exchange); each exponentiates only its own 32.
      float sc[32];
      float m_blk;
      {
        uint32_t r0[32], r1[32];
        tmem_ld32(tmem_s + lane_off + sb * AT_KV + half * 32, r0);
        tmem_ld32(tmem_s + lane_off + sb * AT_KV + (half ^ 1) * 32, r1);
        tmem_ld_wait();
#pragma unroll
        for (int c = 0; c < 32; ++c) sc[c] = __uint_as_float(r0[c]);
        float mo = -INFINITY;
        // warp-uniform branches; only the last prefix block and the own-token block are ragged, and there
        // only one of the two halves of a row is short
        if (n_valid < 32) {
#pragma unroll
          for (int c = 0; c < 32; ++c) sc[c] = c < n_valid ? sc[c] : -INFINITY;
        }
        if (n_other < 32) {
#pragma unroll
          for (int c = 0; c < 32; ++c) mo = fmaxf(mo, c < n_other ? __uint_as_float(r1[c]) : -INFINITY);
        } else {
#pragma unroll
          for (int c = 0; c < 32; ++c) mo = fmaxf(mo, __uint_as_float(r1[c]));
        }
        m_blk = mo;
      }
      if (threadIdx.x == 64) AT_TRACE(8, i);
#pragma unroll
      for (int c = 0; c < 32; ++c) m_blk = fmaxf(m_blk, sc[c]);
      m_blk *= c_log2;
      if (threadIdx.x == 64) AT_TRACE(9, i);
      float factor = 1.f;
      if (m_blk > m_ref + AT_RESCALE_THR) {            // first block always lands here
        factor = ex2_approx(m_ref - m_blk);            // 0 on the first block (m_ref = -inf)
        m_ref = m_blk;
      }
      uint32_t pk[16];
      float s0 = 0.f, s1 = 0.f;
      if (dbg & 4) {  // measurement aid: no softmax arithmetic
        s0 = 1.f;
#pragma unroll
        for (int c = 0; c < 16; ++c) pk[c] = __float_as_uint(sc[2 * c]);
      } else {
        const float neg_m = -m_ref;
#pragma unroll
        for (int c = 0; c < 32; c += 2) {
          const float a = ex2_approx(fmaf(sc[c], c_log2, neg_m)), b = ex2_approx(fmaf(sc[c + 1], c_log2, neg_m));
          s0 += a;
          s1 += b;
          __nv_bfloat162 v2 = __floats2bfloat162_rn(a, b);
          pk[c >> 1] = *reinterpret_cast<uint32_t*>(&v2);
        }
      }
      l_sum = l_sum * factor + (s0 + s1);
      if (threadIdx.x == 64) AT_TRACE(10, i);
      // Every block, not only when rescaling: a parity wait is only meaningful while the waiter is at
      // most one phase behind the barrier (PV(i-1) was issued ~a softmax block ago, so this is free).
      if (i > 0) mbar_wait(pv_done, (i - 1) & 1);
      if (threadIdx.x == 64) AT_TRACE(11, i);
      if (i > 0 && __any_sync(0xffffffffu, factor != 1.f)) {  // rare: rescale this warp's rows, its half of O's columns
        tc_fence_after();                                     // O quiescent: PV(i-1) done, PV(i) needs this P
#pragma unroll 1
        for (int c = half * 4; c < half * 4 + 4; ++c) {
          uint32_t rr[32];
          tmem_ld32(tmem_o + lane_off + c * 32, rr);
          tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 32; ++e) rr[e] = __float_as_uint(__uint_as_float(rr[e]) * factor);
          tmem_st32(tmem_o + lane_off + c * 32, rr);
        }
      }
      // P row r, this half's 32 keys (16 columns of bf16 pairs) over the start of S(i): the A operand of PV(i)
      tmem_st16(tmem_s + lane_off + sb * AT_KV + half * 16, pk);
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(p_full(sb));  // 256 arrivals on one barrier would serialise on the critical path
      if (threadIdx.x == 64) AT_TRACE(5, i);
    }
    // epilogue: O / l -> o[(token, head)]; row r = (token jj, head a) with r = jj * 8 + a.  Each half
    // stores 128 of the 256 columns, transposed through shared memory (the K stages are free: every
    // MMA has completed) for coalesced row stores.
    mbar_wait(pv_done, (nb - 1) & 1);
    tc_fence_after();
    if (threadIdx.x == 64) AT_TRACE(6, 1);
    xch[half * AT_ROWS + r] = l_sum;
    named_bar_sync(1 + q, 64);
    const float inv = 1.f / (l_sum + xch[(half ^ 1) * AT_ROWS + r]);
    // 32 x 32 chunks through a private scratch (pitch 36 floats), then 8 lanes x 4 columns per row
    constexpr int P = 36;
    float* scr = reinterpret_cast<float*>(smem_raw) + (warp - 2) * (32 * P);
    const int lr = lane >> 3, lc = (lane & 7) * 4;
    size_t orow[8];   // output row offsets of the 8 rows this lane stores per chunk; -1 = padding row
#pragma unroll
    for (int x = 0; x < 8; ++x) {
      const int row = q * 32 + x * 4 + lr, j = tt * AT_TOK + (row >> 3);
      orow[x] = j < dm.H ? (size_t)(p * dm.H + j) * dm.q_n + (row & 7) * AT_HD + lc : (size_t)-1;
    }
    uint32_t rbuf[2][32];  // the next chunk's TMEM load is in flight while this one is transposed and stored
    tmem_ld32(tmem_o + lane_off + (half * 4) * 32, rbuf[0]);
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
      const int c = half * 4 + cc;
      uint32_t (&rr)[32] = rbuf[cc & 1];
      tmem_ld_wait();
      if (cc + 1 < 4) tmem_ld32(tmem_o + lane_off + (c + 1) * 32, rbuf[(cc + 1) & 1]);
#pragma unroll
      for (int e = 0; e < 32; e += 4)
        *reinterpret_cast<float4*>(&scr[lane * P + e]) =
            make_float4(__uint_as_float(rr[e]) * inv, __uint_as_float(rr[e + 1]) * inv, __uint_as_float(rr[e + 2]) * inv,
                        __uint_as_float(rr[e + 3]) * inv);
      __syncwarp();
      float4 ov[8];
#pragma unroll
      for (int x = 0; x < 8; ++x) ov[x] = *reinterpret_cast<const float4*>(&scr[(x * 4 + lr) * P + lc]);
#pragma unroll
      for (int x = 0; x < 8; ++x) {
        if (orow[x] != (size_t)-1)
          *reinterpret_cast<uint2*>(o + orow[x] + c * 32) =
              make_uint2(pack_op2(ov[x].x, ov[x].y, dm.fp16), pack_op2(ov[x].z, ov[x].w, dm.fp16));
      }
      __syncwarp();
    }
    if (threadIdx.x == 64) AT_TRACE(6, 2);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

// ------------------------------------------------------------------ host side
static long long* g_attn_trace = nullptr;
// copies the last trace (ROSA_DBG bit 4) to host: [2 CTAs][8 roles][32 blocks] clock64 values
int tc_attn_read_trace(long long* host, int n) {
  if (!g_attn_trace) return 0;
  if (n > 2 * 16 * 32) n = 2 * 16 * 32;
  cudaMemcpy(host, g_attn_trace, n * sizeof(long long), cudaMemcpyDeviceToHost);
  return n;
}

bool tc_attn_supported(const Dims& dm) { return dm.hd == AT_HD && dm.nq == 8 && dm.nkv == 1; }
size_t tc_attn_map_bytes() { return sizeof(CUtensorMap); }

// Tensor maps of one robot's prefix K and V of one layer: [len, 256] bf16, box {64, 64}.
// `out2` = two consecutive CUtensorMap (host memory).
bool tc_attn_make_prefix_maps(void* out2, const bf16* k, const bf16* v, int len, const Dims& dm) {
  CUtensorMap* m = (CUtensorMap*)out2;
  const uint64_t dims[3] = {64, (uint64_t)len, (uint64_t)dm.hd / 64};
  const uint64_t strides[2] = {(uint64_t)dm.nkv * dm.hd * 2, 128};
  const uint32_t box[3] = {64, AT_KV, AT_HD / 64};
  return encode_tmap(&m[0], k, 3, dims, strides, box) && encode_tmap(&m[1], v, 3, dims, strides, box);
}

cudaError_t launch_attn_tc(const Dims& dm, const Tables& tb, int layer, const bf16* qkv, op16* o, int k_iter,
                           int M, const void* d_kv_maps, cudaStream_t s) {
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_attn_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, AT_SMEM);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  AttnMaps maps;
  {
    const uint64_t dims[3] = {(uint64_t)dm.hd, (uint64_t)dm.nq, (uint64_t)M};
    const uint64_t strides[2] = {(uint64_t)dm.hd * 2, (uint64_t)dm.qkv_n * 2};
    const uint32_t box[3] = {64, 8, AT_TOK};
    if (!encode_tmap(&maps.q, qkv, 3, dims, strides, box)) return cudaErrorInvalidValue;
  }
  {
    const uint64_t dims[3] = {64, (uint64_t)M, (uint64_t)dm.qkv_n / 64};
    const uint64_t strides[2] = {(uint64_t)dm.qkv_n * 2, 128};
    const uint32_t box[3] = {64, AT_KV, AT_HD / 64};
    if (!encode_tmap(&maps.own, qkv, 3, dims, strides, box)) return cudaErrorInvalidValue;
  }
  const int tpr = (dm.H + AT_TOK - 1) / AT_TOK;
  static int dbg = -1;  // ROSA_DBG bits 2-4: measurement aids (skip softmax arithmetic / skip the MMAs / trace)
  if (dbg < 0) { const char* e = getenv("ROSA_DBG"); dbg = e ? atoi(e) : 0; }
  if ((dbg & 16) && !g_attn_trace) cudaMalloc((void**)&g_attn_trace, 2 * 16 * 32 * sizeof(long long));
  return launch_k(k_attn_tc, dim3(tb.batch * tpr), dim3(AT_THREADS), AT_SMEM, s, maps, (const CUtensorMap*)d_kv_maps, dm,
                  tb, layer, o, k_iter, tpr, dbg, g_attn_trace);
}

}  // namespace rosa
