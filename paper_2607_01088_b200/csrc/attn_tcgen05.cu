// Ragged-KV GQA attention on tcgen05 (step a5 of the path).
//
// Work item = (robot p, tile of 16 action tokens): all n_q = 8 query heads share the single KV head, so the
// tile's 16 tokens x 8 heads = 128 query rows form ONE M=128 operand against the robot's key/value stream
// [prefix K/V (L_p rows, from the bound cache) ; own k/v (H rows, from the qkv buffer)], walked in blocks of
// 64 keys:
//     S = Q K_blk^T           tcgen05.mma  M=128 N=64  K=256   Q is the A operand FROM TENSOR MEMORY
//     P = exp2(S*c - m_ref)   8 softmax warps, two per query row (32 keys each; both read all 64 scores for
//                             the row maximum), running (m_ref, partial l) in registers; P (bf16) is written
//                             back into tensor memory over S
//     O += P V_blk            tcgen05.mma  M=128 N=256 K=64    P is the A operand from tensor memory,
//                             V the MN-major B operand from shared memory
// Tensor memory (512 columns): O [0,256) | S/P double buffer [256,384) | Q [384,512).
//
// PERSISTENT CTAs over a stream-K work list.  The host cuts the concatenation of all items' key streams into
// one share per CTA (attn_build_list below): a CTA's list is a run of SEGMENTS (item, key blocks [kb0, kb1)).
// An item that straddles a cut is finished by its HEAD segment (kb0 = 0, the last entry of CTA a's list), which
// merges the partial (O, m, l) that the following CTAs (a+1 ..., where the item's other segments are the FIRST
// entry of the list) left in a global scratch slot long before.  Nothing else waits on another CTA, every CTA
// of the grid is resident (grid <= number of SMs, one CTA per SM), so the merge cannot deadlock.
// Inside a CTA the three roles walk the same list; the K/V/Q ring (6 stages of 32 KB, one 3-D TMA per 64-key
// block; per-robot tensor maps made at bind time bound the ragged length: rows >= L_p are zero-filled and
// masked) keeps flowing across segments, the next segment's Q is copied into tensor memory before the current
// segment's O is drained, and its first two S blocks run on the tensor pipe while the softmax warps drain.
// O stays in TMEM for a whole segment; it is rescaled only when a row maximum grows by more than 2^8
// (lazy rescaling), which for N(0,1)-like logits almost never happens after block 0.
#include <algorithm>
#include <cstdlib>
#include <vector>

#include "device_math.cuh"
#include "rosa_internal.h"
#include "tc_common.cuh"

namespace rosa {

using namespace tc;

constexpr int AT_HD = 256;        // head_dim
constexpr int AT_ROWS = 128;      // query rows per item = AT_TOK tokens x 8 heads
constexpr int AT_TOK = 16;
constexpr int AT_KV = 64;         // keys per block
constexpr int AT_RING = 6;        // ring stages: Q (2 entries per segment), K and V blocks in MMA issue order
constexpr int AT_PF = 6;          // L2 prefetch distance in blocks
constexpr int AT_THREADS = 320;   // warp 0 TMA, warp 1 MMA, warps 2..9 softmax/drain (two per TMEM lane quarter)
constexpr int AT_STAGE_BYTES = AT_KV * AT_HD * 2;   // 32 KB: 4 chunks [64 x 64] SW128 (K/V) or 2 chunks [128 x 64] (Q)
constexpr int AT_SCR_PITCH = 40;                    // 16-bit elements per scratch row (80 B: 16-byte aligned rows)
constexpr int AT_SCR_BYTES = 8 * 32 * AT_SCR_PITCH * 2;  // per softmax warp: a 32 x 32 chunk of 16-bit outputs
constexpr int AT_XCH_BYTES = 2 * AT_ROWS * 4;       // row-sum exchange between the two warps of a row
constexpr int AT_SMEM = AT_RING * AT_STAGE_BYTES + AT_SCR_BYTES + AT_XCH_BYTES + 256;
constexpr float AT_RESCALE_THR = 8.0f;              // log2 units
// partial results of cut items: per CTA slot O [256 cols][128 rows] fp32 (row-contiguous per column: coalesced for
// thread = row), then m[2][128], l[2][128] (one copy per column half), and 8 ready flags (one per softmax warp)
constexpr size_t AT_PART_O = (size_t)AT_HD * AT_ROWS;          // floats
constexpr size_t AT_PART_FLOATS = AT_PART_O + 4 * AT_ROWS;

// exp2 on the SFU without the denormal-range fix-up sequence of exp2f (inputs here are <= 2^8)
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
  asm volatile("st.release.gpu.global.b32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ float ld_cg(const float* p) {  // L2 only: written by another SM during this launch
  float v;
  asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}

struct AttnMaps {
  CUtensorMap q;    // qkv buffer as [M tokens][8 heads][256]   box {64, 8, 16}
  CUtensorMap own;  // qkv buffer as (64 cols, M tokens, qkv_n/64 column chunks)   box {64, 64, 4}
};

__global__ void __launch_bounds__(AT_THREADS, 1)
k_attn_tc(const __grid_constant__ AttnMaps maps, const CUtensorMap* __restrict__ kv_maps, Dims dm, Tables tb,
          int layer, op16* __restrict__ o, int k_iter, float* __restrict__ part, int* __restrict__ part_flag) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // this CTA's run of segments in the list of iteration k_iter
  const int* offs = tb.attn_offs + tb.attn_iter[k_iter];
  const int seg_beg = offs[blockIdx.x], seg_end = offs[blockIdx.x + 1];
  if (seg_beg >= seg_end) return;
  const AttnSeg* segs = tb.attn_segs;

  const uint32_t base = smem_u32(smem_raw);  // 1024-byte aligned (SWIZZLE_128B tiles)
  auto stage = [&](int s) { return base + (uint32_t)s * AT_STAGE_BYTES; };
  const uint32_t scr_base = base + AT_RING * AT_STAGE_BYTES;
  const uint32_t bars = scr_base + AT_SCR_BYTES + AT_XCH_BYTES;
  auto full = [&](int s) { return bars + 8u * s; };
  auto empty = [&](int s) { return bars + 8u * (AT_RING + s); };
  auto s_full = [&](int b) { return bars + 8u * (2 * AT_RING + b); };
  // p_full is double-buffered like S/P: the softmax warps may finish block i+1 before the MMA thread
  // has looked at block i's barrier, and a single barrier two phases ahead reads as "not yet"
  auto p_full = [&](int b) { return bars + 8u * (2 * AT_RING + 2 + b); };
  const uint32_t pv_done = bars + 8u * (2 * AT_RING + 4);
  const uint32_t q_ready = bars + 8u * (2 * AT_RING + 5), o_empty = bars + 8u * (2 * AT_RING + 6);
  const uint32_t tmem_slot = bars + 8u * (2 * AT_RING + 7);
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - base));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&maps.q);
    prefetch_tensormap(&maps.own);
    for (int s = 0; s < AT_RING; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); }
    mbar_init(s_full(0), 1); mbar_init(s_full(1), 1);
    mbar_init(p_full(0), 8); mbar_init(p_full(1), 8);  // one arrival per softmax warp
    mbar_init(pv_done, 1);
    mbar_init(q_ready, 8);
    mbar_init(o_empty, 8);
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

  pdl_wait();     // everything above overlapped the previous kernel's tail
  pdl_trigger();

  if (warp == 0) {
    // ------------------------------------------------ TMA producer (whole warp; one lane issues)
    // Ring entries in MMA consumption order: Q (2 entries), K(0), then K(i+1), V(i) for every block.
    uint32_t rp = 0;  // entries issued so far
    auto acquire = [&]() {
      const int s = (int)(rp % AT_RING);
      mbar_wait_idle(empty(s), ((rp / AT_RING) & 1) ^ 1);
      ++rp;
      return s;
    };
    for (int si = seg_beg; si < seg_end; ++si) {
      const AttnSeg sg = segs[si];
      const int p = sg.p, robot = tb.ids[p], L = tb.rlen[robot];
      const int nbp = (L + AT_KV - 1) / AT_KV;  // prefix blocks; block nbp = the robot's own tokens
      const CUtensorMap* kmap = kv_maps + ((size_t)robot * dm.layers + layer) * 2;
      const CUtensorMap* vmap = kmap + 1;
      const int tok0 = p * dm.H + sg.tt * AT_TOK;
      if (lane == 0) { prefetch_tensormap(kmap); prefetch_tensormap(vmap); }
      // one TMA per 64-key block: 3-D maps (64 columns, rows, 4 column chunks) land as [chunk][row][128 B]
      auto load_kv = [&](int i, bool is_v) {
        const int s = acquire();
        if (elect_one()) {
          mbar_expect_tx(full(s), AT_STAGE_BYTES);
          if (i == nbp) tma_load_3d(stage(s), &maps.own, full(s), 0, p * dm.H, (dm.q_n + (is_v ? AT_HD : 0)) / 64);
          else tma_load_3d(stage(s), is_v ? vmap : kmap, full(s), 0, i * AT_KV, 0);
        }
        __syncwarp();
      };
      for (int e = 0; e < 2; ++e) {
        const int s = acquire();
        if (elect_one()) {
          mbar_expect_tx(full(s), AT_STAGE_BYTES);
          for (int c = 0; c < 2; ++c) tma_load_3d(stage(s) + c * (AT_ROWS * 128), &maps.q, full(s), (2 * e + c) * 64, 0, tok0);
        }
        __syncwarp();
      }
      load_kv(sg.kb0, false);
      for (int i = sg.kb0; i < sg.kb1; ++i) {  // K runs one block ahead of V: it is needed a whole softmax earlier
        if (i + 1 < sg.kb1) load_kv(i + 1, false);
        load_kv(i, true);
        if (elect_one()) {
          // L2 prefetches go out only after everything the first MMAs wait for (Q, K0, K1, V0) is in flight
          const int lim = min(sg.kb1, nbp);
          if (i == sg.kb0)
            for (int j = sg.kb0 + 2; j < sg.kb0 + AT_PF; ++j)
              if (j < lim) { tma_prefetch_3d(kmap, 0, j * AT_KV, 0); tma_prefetch_3d(vmap, 0, j * AT_KV, 0); }
          if (i + AT_PF < lim) { tma_prefetch_3d(kmap, 0, (i + AT_PF) * AT_KV, 0); tma_prefetch_3d(vmap, 0, (i + AT_PF) * AT_KV, 0); }
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------ MMA issuer (whole warp; one lane issues)
    constexpr uint32_t idesc_s = make_idesc_bf16(AT_ROWS, AT_KV);
    constexpr uint32_t idesc_o = make_idesc_bf16(AT_ROWS, AT_HD, /*b_mn_major=*/true);
    uint32_t rp = 0;  // ring entries consumed
    uint32_t g = 0;   // key blocks issued so far in this CTA (selects the S/P buffer and the barrier parities)
    uint32_t j = 0;   // segments started
    for (int si = seg_beg; si < seg_end; ++si, ++j) {
      const AttnSeg sg = segs[si];
      const int n = sg.kb1 - sg.kb0;
      auto issue_s = [&](uint32_t gi) {  // S(gi) = Q K^T into S buffer gi&1 (overwrites P(gi-2), consumed by PV(gi-2))
        const int s = (int)(rp % AT_RING);
        mbar_wait(full(s), (rp / AT_RING) & 1);
        ++rp;
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int kk = 0; kk < AT_HD / 16; ++kk) {
            const uint32_t ka = stage(s) + (kk >> 2) * (AT_KV * 128) + (kk & 3) * 32;
            umma_bf16_ts(tmem_s + (gi & 1) * AT_KV, tmem_q + kk * 8, make_sdesc_k128(ka), idesc_s, kk != 0);
          }
          umma_commit(empty(s));
          umma_commit(s_full(gi & 1));
        }
        __syncwarp();
      };
      // Q of this segment is in tensor memory (softmax warps); its two ring entries are free again
      mbar_wait(q_ready, j & 1);
      tc_fence_after();
      if (elect_one()) {
        mbar_arrive(empty((int)(rp % AT_RING)));
        mbar_arrive(empty((int)((rp + 1) % AT_RING)));
      }
      __syncwarp();
      rp += 2;
      issue_s(g);
      for (int i = 0; i < n; ++i) {
        const uint32_t gi = g + i;
        if (i + 1 < n) issue_s(gi + 1);
        const int s = (int)(rp % AT_RING);
        mbar_wait(full(s), (rp / AT_RING) & 1);
        ++rp;
        if (i == 0 && j > 0) mbar_wait(o_empty, (j - 1) & 1);  // the previous segment's O has been drained
        mbar_wait(p_full(gi & 1), (gi >> 1) & 1);
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int kk = 0; kk < AT_KV / 16; ++kk) {
            // A = P [128 x 64] bf16 in TMEM (8 columns per 16 keys); B = V block, MN-major: 4 hd chunks
            // 8192 B apart (LBO), 8-key groups 1024 B apart (SBO); 16 keys per MMA = 2048 B
            const uint64_t b_desc = make_sdesc_mn128(stage(s) + kk * 2048, AT_KV * 128, 1024);
            umma_bf16_ts(tmem_o, tmem_s + (gi & 1) * AT_KV + kk * 8, b_desc, idesc_o, (i | kk) != 0);
          }
          umma_commit(empty(s));
          umma_commit(pv_done);
        }
        __syncwarp();
      }
      g += n;
    }
  } else {
    // ---------------------------------------------------------- softmax + drain warps (2..9)
    // Two warps per TMEM lane quarter: a query row's 64 scores of a block are split 32 / 32 between
    // warp w (half 0) and warp w + 4 (half 1).  Both read all 64 scores for the row maximum
    // (so both take the same rescale decision) and keep separate partial row sums until the end.
    const int q = warp & 3, half = (warp - 2) >> 2, sw = warp - 2;
    const int r = q * 32 + lane;                       // query row of this thread
    const uint32_t lane_off = (uint32_t)(q * 32) << 16;
    float* xch = reinterpret_cast<float*>(smem_raw + (AT_RING * AT_STAGE_BYTES + AT_SCR_BYTES));  // [2 halves][128]
    const uint32_t scr = scr_base + (uint32_t)sw * (32 * AT_SCR_PITCH * 2);
    const float c_log2 = rsqrtf((float)AT_HD) * 1.4426950408889634f;  // (1/sqrt(hd)) * log2(e)
    const int lr = lane >> 3, lc = (lane & 7) * 4;
    // Q of a segment: shared memory (SW128 chunks of [128 rows x 128 B]) -> tensor memory, thread = row; this half's
    // two chunks are one ring entry (rq = ring position of the segment's first entry).  Called when every S MMA of
    // the previous segment has completed (its last s_full was waited on), so tmem_q is free.
    auto copy_q = [&](uint32_t rq) {
      const uint32_t e = rq + half;
      const int s = (int)(e % AT_RING);
      mbar_wait(full(s), (e / AT_RING) & 1);
#pragma unroll 1
      for (int cc = 0; cc < 2; ++cc) {
        uint32_t w[32];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
          const uint32_t addr = stage(s) + cc * (AT_ROWS * 128) + r * 128 + ((x ^ (r & 7)) << 4);
          asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                       : "=r"(w[4 * x]), "=r"(w[4 * x + 1]), "=r"(w[4 * x + 2]), "=r"(w[4 * x + 3]) : "r"(addr));
        }
        tmem_st32(tmem_q + lane_off + (half * 2 + cc) * 32, w);
      }
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(q_ready);
    };
    uint32_t rp = 0, g = 0;
    copy_q(0);
    for (int si = seg_beg; si < seg_end; ++si) {
      const AttnSeg sg = segs[si];
      const int p = sg.p, L = tb.rlen[tb.ids[p]], nbp = (L + AT_KV - 1) / AT_KV;
      const int n = sg.kb1 - sg.kb0;
      rp += 2 + 2 * n;   // ring position of the next segment's Q
      float m_ref = -INFINITY, l_sum = 0.f;            // m_ref in log2 units; l_sum: this half's part
      for (int i = 0; i < n; ++i) {
        const uint32_t gi = g + i;
        const int sb = gi & 1, kb = sg.kb0 + i;
        const int n_tot = kb == nbp ? dm.H : min(AT_KV, L - kb * AT_KV);
        const int n_valid = n_tot - half * 32, n_other = n_tot - (half ^ 1) * 32;  // valid columns of this / the other half
        mbar_wait(s_full(sb), (gi >> 1) & 1);
        tc_fence_after();
        // Both warps of a row read all 64 scores for the row maximum (so they take the same rescale
        // decision without an exchange); each exponentiates only its own 32.
        float sc[32];
        float m_blk;
        {
          uint32_t r0[32], r1[32];
          tmem_ld32(tmem_s + lane_off + sb * AT_KV + half * 32, r0);
          tmem_ld32(tmem_s + lane_off + sb * AT_KV + (half ^ 1) * 32, r1);
          tmem_ld_wait();
          // P(gi) is written IN PLACE over S(gi), and each warp of a row's pair has just read the other's scores
          // too: neither may store its P before both have read (the two were released by the same s_full, so
          // this barrier costs little; without it a warp held up for more than a block - by a merge wait, say -
          // reads scores its partner has already overwritten)
          named_bar_sync(5 + q, 64);
#pragma unroll
          for (int c = 0; c < 32; ++c) sc[c] = __uint_as_float(r0[c]);
          float mo = -INFINITY;
          // warp-uniform branches; only the last prefix block and the own-token block are ragged
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
#pragma unroll
        for (int c = 0; c < 32; ++c) m_blk = fmaxf(m_blk, sc[c]);
        m_blk *= c_log2;
        float factor = 1.f;
        if (m_blk > m_ref + AT_RESCALE_THR) {            // first block always lands here
          factor = ex2_approx(m_ref - m_blk);            // 0 on the first block (m_ref = -inf)
          m_ref = m_blk;
        }
        uint32_t pk[16];
        float s0 = 0.f, s1 = 0.f;
        {
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
        // Every block, not only when rescaling: a parity wait is only meaningful while the waiter is at
        // most one phase behind the barrier (PV(gi-1) was issued ~a softmax block ago, so this is free).
        if (gi > 0) mbar_wait(pv_done, (gi - 1) & 1);
        if (i > 0 && __any_sync(0xffffffffu, factor != 1.f)) {  // rare: rescale this warp's rows, its half of O's columns
          tc_fence_after();                                     // O quiescent: PV(gi-1) done, PV(gi) needs this P
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
        // P row r, this half's 32 keys (16 columns of bf16 pairs) over the start of S(gi): the A operand of PV(gi)
        tmem_st16(tmem_s + lane_off + sb * AT_KV + half * 16, pk);
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(p_full(sb));  // 256 arrivals on one barrier would serialise on the critical path
      }
      g += n;
      // The next segment's Q goes into tensor memory BEFORE this segment's O is drained: its first two S blocks then
      // run on the tensor pipe while these warps drain.
      if (si + 1 < seg_end) copy_q(rp);
      // ------------------------------------------------ drain: O (+ partials of the item's other segments) -> o,
      // or this segment's partial -> scratch.  Row r = (token jj, head a) with r = jj * 8 + a; each half owns 128
      // of the 256 columns.
      mbar_wait(pv_done, (g - 1) & 1);
      tc_fence_after();
      xch[half * AT_ROWS + r] = l_sum;
      named_bar_sync(1 + q, 64);
      float l_tot = l_sum + xch[(half ^ 1) * AT_ROWS + r];
      named_bar_sync(1 + q, 64);   // xch is reused by the next segment

      if (sg.n_part < 0) {
        // not the head segment: leave (O, m, l) for the CTA that holds the head
        float* slot = part + (size_t)blockIdx.x * AT_PART_FLOATS;
#pragma unroll 1
        for (int cc = 0; cc < 4; ++cc) {
          const int c = half * 4 + cc;
          uint32_t rr[32];
          tmem_ld32(tmem_o + lane_off + c * 32, rr);
          tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 32; ++e) slot[(size_t)(c * 32 + e) * AT_ROWS + r] = __uint_as_float(rr[e]);
        }
        slot[AT_PART_O + half * AT_ROWS + r] = m_ref;
        slot[AT_PART_O + (2 + half) * AT_ROWS + r] = l_tot;
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(o_empty);
        __threadfence();
        __syncwarp();
        if (lane == 0) st_release_gpu(part_flag + blockIdx.x * 8 + sw, 1);
        __syncwarp();
      } else {
        float f_own = 1.f;
        float fc[3] = {0.f, 0.f, 0.f};   // at most 3 other segments are merged per pass (attn_build_list guarantees <= 3)
        const int np = sg.n_part;
        if (np > 0) {
          float mc[3] = {-INFINITY, -INFINITY, -INFINITY}, lcs[3] = {0.f, 0.f, 0.f};
          float m_new = m_ref;
          for (int t = 0; t < np; ++t) {
            const int c_id = sg.part0 + t;
            const int* fl = part_flag + c_id * 8 + sw;
            for (uint32_t spin = 0; ld_acquire_gpu(fl) == 0; ++spin) {
              __nanosleep(64);
              if (spin > (1u << 24)) __trap();
            }
            __syncwarp();   // the lanes leave the spin at different polls; the TMEM loads below are .sync.aligned
            const float* slot = part + (size_t)c_id * AT_PART_FLOATS;
            mc[t] = ld_cg(slot + AT_PART_O + half * AT_ROWS + r);
            lcs[t] = ld_cg(slot + AT_PART_O + (2 + half) * AT_ROWS + r);
            m_new = fmaxf(m_new, mc[t]);
          }
          f_own = ex2_approx(m_ref - m_new);
          l_tot *= f_own;
          for (int t = 0; t < np; ++t) { fc[t] = ex2_approx(mc[t] - m_new); l_tot += lcs[t] * fc[t]; }
        }
        const float inv = 1.f / l_tot;
        size_t orow[8];   // output row offsets of the 8 rows this lane stores per chunk; -1 = padding row
#pragma unroll
        for (int x = 0; x < 8; ++x) {
          const int row = q * 32 + x * 4 + lr, jj = sg.tt * AT_TOK + (row >> 3);
          orow[x] = jj < dm.H ? (size_t)(p * dm.H + jj) * dm.q_n + (row & 7) * AT_HD + lc : (size_t)-1;
        }
#pragma unroll 1
        for (int cc = 0; cc < 4; ++cc) {
          const int c = half * 4 + cc;
          float v[32];
          {
            uint32_t rr[32];
            tmem_ld32(tmem_o + lane_off + c * 32, rr);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 32; ++e) v[e] = __uint_as_float(rr[e]) * f_own;
          }
          if (cc == 3) {  // this warp has read all of its part of O
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(o_empty);
          }
          for (int t = 0; t < np; ++t) {
            const float* src = part + (size_t)(sg.part0 + t) * AT_PART_FLOATS + (size_t)(c * 32) * AT_ROWS + r;
            const float f = fc[t];
#pragma unroll
            for (int e = 0; e < 32; ++e) v[e] = fmaf(ld_cg(src + (size_t)e * AT_ROWS), f, v[e]);
          }
          // 16-bit outputs transposed through the warp's scratch: thread = row writes 64 B, then 8 lanes x 4 columns per row
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const uint32_t a0 = pack_op2(v[8 * x + 0] * inv, v[8 * x + 1] * inv, dm.fp16), a1 = pack_op2(v[8 * x + 2] * inv, v[8 * x + 3] * inv, dm.fp16);
            const uint32_t a2 = pack_op2(v[8 * x + 4] * inv, v[8 * x + 5] * inv, dm.fp16), a3 = pack_op2(v[8 * x + 6] * inv, v[8 * x + 7] * inv, dm.fp16);
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(scr + lane * (AT_SCR_PITCH * 2) + x * 16), "r"(a0), "r"(a1), "r"(a2), "r"(a3) : "memory");
          }
          __syncwarp();
          uint2 ov[8];
#pragma unroll
          for (int x = 0; x < 8; ++x)
            asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(ov[x].x), "=r"(ov[x].y) : "r"(scr + (x * 4 + lr) * (AT_SCR_PITCH * 2) + lc * 2));
#pragma unroll
          for (int x = 0; x < 8; ++x)
            if (orow[x] != (size_t)-1) *reinterpret_cast<uint2*>(o + orow[x] + c * 32) = ov[x];
          __syncwarp();
        }
        if (np > 0) {  // the slots are free for the next launch
          __syncwarp();
          if (lane == 0)
            for (int t = 0; t < np; ++t) part_flag[(sg.part0 + t) * 8 + sw] = 0;
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

// ------------------------------------------------------------------ host side
bool tc_attn_supported(const Dims& dm) { return dm.hd == AT_HD && dm.nq == 8 && dm.nkv == 1; }
size_t tc_attn_map_bytes() { return sizeof(CUtensorMap); }
size_t tc_attn_part_bytes(int n_cta) { return (size_t)n_cta * AT_PART_FLOATS * sizeof(float); }
int tc_attn_tiles(const Dims& dm) { return (dm.H + AT_TOK - 1) / AT_TOK; }

// Stream-K work list of one Euler iteration: the first `n_active` robots (internal order) with prefix lengths
// len[p]; item (p, tt) has ceil(len/64) + 1 key blocks; every segment costs its blocks + kSegOvh units (Q load,
// drain).  The concatenated items are cut into equal shares for `n_cta` CTAs (fewer when there is little work:
// a share is at least kMinShare units); no segment is shorter than kMinSeg blocks and no item has more than 4
// segments.  offs[c] .. offs[c+1] = segments of CTA c (offs has n_cta + 1 entries; CTAs without work get none).
int attn_build_list(const Dims& dm, int n_active, const int* len, int n_cta, std::vector<AttnSeg>& segs, int* offs) {
  constexpr double kSegOvh = 2.0, kMinShare = 6.0;
  constexpr int kMinSeg = 2;
  const int tpr = tc_attn_tiles(dm);
  const size_t seg0 = segs.size();
  double total = 0.0;
  for (int p = 0; p < n_active; ++p) total += tpr * ((len[p] + AT_KV - 1) / AT_KV + 1 + kSegOvh);
  const int used = (int)std::min<double>(n_cta, std::max(1.0, std::floor(total / kMinShare)));
  // units not yet assigned, counting one extra segment overhead for each of the used - 1 CTA boundaries still ahead
  // (most of them cut an item in two); a boundary that falls between two items gives its overhead back
  double left = total + kSegOvh * (used - 1);
  double target = left / used;  // share of the current CTA: re-derived at every CTA from what is left
  int cta = 0;
  double acc = 0.0;
  offs[0] = (int)seg0;
  auto next_cta = [&](bool cut) {
    if (cta + 1 < used) {
      if (!cut) left -= kSegOvh;
      ++cta; offs[cta] = (int)segs.size(); acc = 0.0; target = left / (used - cta);
    }
  };
  for (int p = 0; p < n_active; ++p) {
    const int nb = (len[p] + AT_KV - 1) / AT_KV + 1;
    for (int tt = 0; tt < tpr; ++tt) {
      int kb = 0, n_seg = 0;
      const size_t head = segs.size();
      while (kb < nb) {
        const int rem = nb - kb;
        const double room = target - acc;
        int take = rem;
        if (cta + 1 < used && rem + kSegOvh > room + 0.5 && n_seg < 3) {
          take = (int)std::floor(room - kSegOvh + 0.5);
          if (take < kMinSeg) {            // not worth starting here: the next CTA takes it
            if (acc > 0.0) { next_cta(kb > 0); continue; }
            take = std::min(rem, kMinSeg);
          }
          if (rem - take < kMinSeg) take = rem;   // no crumbs at the end either
        }
        AttnSeg sg;
        sg.p = p; sg.tt = (int16_t)tt; sg.kb0 = (int16_t)kb; sg.kb1 = (int16_t)(kb + take);
        sg.n_part = kb == 0 ? 0 : -1; sg.part0 = -1; sg.pad = 0;
        if (kb > 0) {  // a continuation is the first entry of a CTA's list; the head segment collects it
          segs[head].n_part += 1;
          if (segs[head].part0 < 0) segs[head].part0 = (int16_t)cta;
        }
        segs.push_back(sg);
        ++n_seg;
        kb += take;
        acc += take + kSegOvh;
        left -= take + kSegOvh;
        if (kb < nb || acc >= target - 0.5) next_cta(kb < nb);
      }
    }
  }
  for (int c = cta + 1; c <= n_cta; ++c) offs[c] = (int)segs.size();
  return (int)(segs.size() - seg0);
}

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
                           int M, const void* d_kv_maps, float* part, int* part_flag, int n_cta, cudaStream_t s) {
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
  return launch_k(k_attn_tc, dim3(n_cta), dim3(AT_THREADS), AT_SMEM, s, maps, (const CUtensorMap*)d_kv_maps, dm,
                  tb, layer, o, k_iter, part, part_flag);
}

}  // namespace rosa
