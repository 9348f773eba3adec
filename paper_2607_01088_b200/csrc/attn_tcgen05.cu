// Ragged-KV GQA attention on tcgen05 (step a5 of the path).
//
// Work item = (robot p, tile of 16 action tokens): all n_q = 8 query heads share the single KV head, so the
// tile's 16 tokens x 8 heads = 128 query rows form ONE M=128 operand against the robot's key/value stream
// [prefix K/V (L_p rows, from the bound cache) ; own k/v (H rows, from the qkv buffer)], walked in blocks of
// 64 keys:
//     S = Q K_blk^T           tcgen05.mma  M=128 N=64  K=256   Q is the A operand FROM TENSOR MEMORY
//     P = exp2(S*c - m_ref)   8 softmax warps, two per query row: one takes the even key blocks, the other the odd ones
//                             (whole rows of 64 scores; the row's reference m_ref is handed from block to block
//                             through shared memory), each with its own partial l in registers; P (bf16) is
//                             written back into tensor memory over the scores
//     O += P V_blk            tcgen05.mma  M=128 N=256 K=64    P is the A operand from tensor memory,
//                             V the MN-major B operand from shared memory
// Tensor memory (512 columns): O [0,256) | S/P double buffer [256,384) | Q [384,512).
//
// PERSISTENT CTAs over a stream-K work list.  The host cuts the concatenation of all items' key streams into
// one share per CTA (attn_build_list below): a CTA's list is a run of SEGMENTS (item, key blocks [kb0, kb1)).
// An item that straddles a cut is finished by its HEAD segment (kb0 = 0, the last entry of CTA a's list), which
// merges the partial (O, m, l) that CTA a+1 (where the item's other segment is the FIRST entry of the list) left
// in its global scratch slot long before.  Nothing else waits on another CTA, every CTA of the grid is resident
// (grid <= number of SMs, one CTA per SM), so the merge cannot deadlock.  (When whole items, longest first, are
// estimated to finish no later, the planner keeps that plan instead: no cuts, no merges.)
// Inside a CTA the three roles walk the same list; the K/V/Q ring (5 stages of 32 KB, one 3-D TMA per 64-key
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
constexpr int AT_RING = 5;        // ring stages: Q (2 entries per segment), K and V blocks in MMA issue order
constexpr int AT_PF = 6;          // L2 prefetch distance in blocks
constexpr int AT_THREADS = 320;   // warp 0 TMA, warp 1 MMA, warps 2..9 softmax/drain (two per TMEM lane quarter)
constexpr int AT_STAGE_BYTES = AT_KV * AT_HD * 2;   // 32 KB: 4 chunks [64 x 64] SW128 (K/V) or 2 chunks [128 x 64] (Q)
// Output staging: the segment's 128 x 256 result as 16-bit values, four SWIZZLE_128B boxes [128 rows x 64 columns],
// followed by the row statistics (m[128], l[128], fp32) of a partial result.  The drain only moves O from tensor
// memory into this tile (thread = row, 16-byte shared-memory stores); from there a head segment stores its rows
// to o with coalesced 16-byte accesses, a continuation hands the whole tile to the copy engine (one bulk copy into
// the CTA's scratch slot).  (TMA tensor stores into o were measured at ~1k cycles of issue time each.)
constexpr int AT_STG_BYTES = AT_ROWS * AT_HD * 2;   // 64 KB
constexpr int AT_ML_BYTES = 2 * AT_ROWS * 4;
constexpr int AT_MX_BYTES = AT_ROWS * 4;            // the row's softmax reference, handed from the warp of block i to the warp of block i + 1
constexpr int AT_SMEM = AT_RING * AT_STAGE_BYTES + AT_STG_BYTES + AT_ML_BYTES + AT_MX_BYTES + 256;
static_assert(AT_SMEM <= 232448, "shared memory of one CTA");
constexpr float AT_RESCALE_THR = 8.0f;              // log2 units
constexpr size_t AT_PART_BYTES = AT_STG_BYTES + AT_ML_BYTES;   // scratch slot of a CTA: a copy of staging + statistics

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
__device__ __forceinline__ int ld_relaxed_gpu(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
  asm volatile("st.release.gpu.global.b32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// generic <-> async proxy ordering for global and shared memory alike
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
// asynchronous copies out of / into shared memory (bulk groups are per thread: the issuing thread also waits)
__device__ __forceinline__ void tma_store_4d(const CUtensorMap* tm, uint32_t src, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
               ::"l"(tm), "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ AttnSeg ld_seg(const AttnSeg* p) {   // read-only table: two 16-byte loads
  union { AttnSeg s; uint4 u[2]; } v;
  v.u[0] = __ldg(reinterpret_cast<const uint4*>(p));
  v.u[1] = __ldg(reinterpret_cast<const uint4*>(p) + 1);
  return v.s;
}

// Measurement aid, compiled in only with -DROSA_TRACE: clock64 of pipeline events per CTA, [cta][64]:
// 0 entry, 1 after the dependency wait, 2 exit, 3 / 4 cycles the MMA thread waited for ring data / for P; per segment
// j < 4 at 8 + 8 j: +0 softmax: first S block ready, +1 softmax loop done, +2 next Q copied, +7 last PV done, +3 O out of
// tensor memory, +4 drain done; +5 MMA: segment start (Q ready), +6 last PV issued.  Blocks 4 (warp 2, slots 40..45) and 5
// (warp 6, 48..53) of the CTA's first segment: block start, S ready, maximum done, reference received, P stored, arrived;
// 47 / 55 = start of blocks 6 / 7.  MMA thread, same blocks (56..59, 60..63): waiting for P from, P seen, PV issued, S(i+2) issued.
#ifdef ROSA_TRACE
__device__ long long g_attn_trace[160 * 64];
#define AT_TRACE(slot) do { if (lane == 0 && (slot) < 64) g_attn_trace[blockIdx.x * 64 + (slot)] = clock64(); } while (0)
extern "C" int rosa_trace_attn(long long* host) { return (int)cudaMemcpyFromSymbol(host, g_attn_trace, sizeof(g_attn_trace)); }
#else
#define AT_TRACE(slot) do { } while (0)
#endif

struct AttnMaps {
  CUtensorMap q;    // qkv buffer as [M tokens][8 heads][256]   box {64, 8, 16}
  CUtensorMap own;  // qkv buffer as (64 cols, M tokens, qkv_n/64 column chunks)   box {64, 64, 4}
};

__global__ void __launch_bounds__(AT_THREADS, 1)
k_attn_tc(const __grid_constant__ AttnMaps maps, const CUtensorMap* __restrict__ kv_maps, Dims dm, Tables tb,
          int layer, op16* __restrict__ o, int k_iter, uint8_t* __restrict__ part, int* __restrict__ part_flag) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // this CTA's run of segments in the list of iteration k_iter
  const int* offs = tb.attn_offs + tb.attn_iter[k_iter];
  const int seg_beg = offs[blockIdx.x], seg_end = offs[blockIdx.x + 1];
  if (seg_beg >= seg_end) return;
  const AttnSeg* segs = tb.attn_segs;

  const uint32_t base = smem_u32(smem_raw);  // 1024-byte aligned (SWIZZLE_128B tiles)
  auto stage = [&](int s) { return base + (uint32_t)s * AT_STAGE_BYTES; };
  const uint32_t stg = base + AT_RING * AT_STAGE_BYTES;   // output staging (+ statistics right behind it)
  const uint32_t bars = stg + AT_STG_BYTES + AT_ML_BYTES + AT_MX_BYTES;
  auto full = [&](int s) { return bars + 8u * s; };
  auto empty = [&](int s) { return bars + 8u * (AT_RING + s); };
  auto s_full = [&](int b) { return bars + 8u * (2 * AT_RING + b); };
  // p_full is double-buffered like S/P: the softmax warps may finish block i+1 before the MMA thread
  // has looked at block i's barrier, and a single barrier two phases ahead reads as "not yet"
  auto p_full = [&](int b) { return bars + 8u * (2 * AT_RING + 2 + b); };
  // PV(x) completes pv_done(x & 3), phase x >> 2.  A parity wait is only meaningful while the barrier is at most one
  // phase ahead of the waiter; the softmax warps look at these barriers rarely (an O rescale, the drain) and with four
  // of them "PV(x - 4) is known to be complete, PV(x + 4) cannot have been issued" is all a waiter for PV(x) needs -
  // both hold wherever PV(x) is waited for (the MMA thread issues PV(x + 1) only after this warp's or its partner's P).
  auto pv_done = [&](uint32_t x) { return bars + 8u * (2 * AT_RING + 4 + (x & 3u)); };
  const uint32_t q_ready = bars + 8u * (2 * AT_RING + 8), o_empty = bars + 8u * (2 * AT_RING + 9);
  const uint32_t part_full = bars + 8u * (2 * AT_RING + 10);   // the partner's partial result has landed in staging
  const uint32_t tmem_slot = bars + 8u * (2 * AT_RING + 11);
  // hand(q, b): the warp of lane quarter q that did block gi (b = gi & 1) has left the rows' reference in shared memory
  auto hand = [&](int qq, int b) { return bars + 8u * (2 * AT_RING + 12 + qq * 2 + b); };
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - base));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 2) AT_TRACE(0);

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&maps.q);
    prefetch_tensormap(&maps.own);
    for (int s = 0; s < AT_RING; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); }
    mbar_init(s_full(0), 1); mbar_init(s_full(1), 1);
    mbar_init(p_full(0), 4); mbar_init(p_full(1), 4);  // one arrival per softmax warp of the block's set
    for (uint32_t x = 0; x < 4; ++x) mbar_init(pv_done(x), 1);
    for (int x = 0; x < 8; ++x) mbar_init(hand(x >> 1, x & 1), 1);
    mbar_init(q_ready, 8);
    mbar_init(o_empty, 8);
    mbar_init(part_full, 1);
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

  if (warp == 0) {
    // ------------------------------------------------ TMA producer: ONE thread from start to end
    // Ring entries in MMA consumption order: Q (2 entries), K(0), then K(i+1), V(i) for every block.
    const bool issuer = elect_one();
    uint32_t rp = 0;  // entries issued so far
    AttnSeg nxt = ld_seg(segs + seg_beg);
    // The prefix cache does not depend on the previous kernel: the first segment's K(kb0), K(kb0+1), V(kb0) go out
    // BEFORE the dependency wait, straight into the ring entries they will be consumed from (2, 3, 4); Q and the
    // block of the robot's own tokens (written by the QKV GEMM) follow after it.
    uint32_t pre_mask = 0;
    if (issuer) {
      const CUtensorMap* km = kv_maps + ((size_t)nxt.robot * dm.layers + layer) * 2;
      prefetch_tensormap(km); prefetch_tensormap(km + 1);
      const int nbp = (nxt.len + AT_KV - 1) / AT_KV, n = nxt.kb1 - nxt.kb0;
      const int blk[3] = {nxt.kb0, n > 1 ? nxt.kb0 + 1 : nxt.kb0, nxt.kb0};
      const bool isv[3] = {false, n > 1 ? false : true, true};
      const int cnt = n > 1 ? 3 : 2;
      for (int x = 0; x < cnt; ++x)
        if (blk[x] < nbp) {
          mbar_expect_tx(full(2 + x), AT_STAGE_BYTES);
          tma_load_3d(stage(2 + x), isv[x] ? km + 1 : km, full(2 + x), 0, blk[x] * AT_KV, 0);
          pre_mask |= 1u << (2 + x);
        }
    }
    pdl_wait();     // everything above overlapped the previous kernel's tail
    pdl_trigger();
    if (issuer) {
    auto acquire = [&](bool& issue) {   // next ring entry; issue = false if it was filled before the wait
      const int s = (int)(rp % AT_RING);
      issue = !(rp < AT_RING && ((pre_mask >> rp) & 1u));
      if (issue) mbar_wait_idle(empty(s), ((rp / AT_RING) & 1) ^ 1);
      ++rp;
      return s;
    };
    for (int si = seg_beg; si < seg_end; ++si) {
      const AttnSeg sg = nxt;
      if (si + 1 < seg_end) {   // the next record and its robot's tensor maps are fetched a whole segment ahead
        nxt = ld_seg(segs + si + 1);
        if (nxt.robot != sg.robot) {
          const CUtensorMap* km = kv_maps + ((size_t)nxt.robot * dm.layers + layer) * 2;
          prefetch_tensormap(km); prefetch_tensormap(km + 1);
        }
      }
      const int p = sg.p, L = sg.len;
      const int nbp = (L + AT_KV - 1) / AT_KV;  // prefix blocks; block nbp = the robot's own tokens
      const CUtensorMap* kmap = kv_maps + ((size_t)sg.robot * dm.layers + layer) * 2;
      const CUtensorMap* vmap = kmap + 1;
      const int tok0 = p * dm.H + sg.tt * AT_TOK;
      // one TMA per 64-key block: 3-D maps (64 columns, rows, 4 column chunks) land as [chunk][row][128 B]
      auto load_kv = [&](int i, bool is_v) {
        bool issue;
        const int s = acquire(issue);
        if (issue) {
          mbar_expect_tx(full(s), AT_STAGE_BYTES);
          if (i == nbp) tma_load_3d(stage(s), &maps.own, full(s), 0, p * dm.H, (dm.q_n + (is_v ? AT_HD : 0)) / 64);
          else tma_load_3d(stage(s), is_v ? vmap : kmap, full(s), 0, i * AT_KV, 0);
        }
      };
      for (int e = 0; e < 2; ++e) {
        bool issue;
        const int s = acquire(issue);
        mbar_expect_tx(full(s), AT_STAGE_BYTES);
        for (int c = 0; c < 2; ++c) tma_load_3d(stage(s) + c * (AT_ROWS * 128), &maps.q, full(s), (2 * e + c) * 64, 0, tok0);
      }
      load_kv(sg.kb0, false);
      for (int i = sg.kb0; i < sg.kb1; ++i) {  // K runs one block ahead of V: it is needed a whole softmax earlier
        if (i + 1 < sg.kb1) load_kv(i + 1, false);
        load_kv(i, true);
        // L2 prefetches go out only after everything the first MMAs wait for (Q, K0, K1, V0) is in flight
        const int lim = min(sg.kb1, nbp);
        if (i == sg.kb0)
          for (int j = sg.kb0 + 2; j < sg.kb0 + AT_PF; ++j)
            if (j < lim) { tma_prefetch_3d(kmap, 0, j * AT_KV, 0); tma_prefetch_3d(vmap, 0, j * AT_KV, 0); }
        if (i + AT_PF < lim) { tma_prefetch_3d(kmap, 0, (i + AT_PF) * AT_KV, 0); tma_prefetch_3d(vmap, 0, (i + AT_PF) * AT_KV, 0); }
      }
    }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ------------------------------------------------ MMA issuer: ONE thread from start to end.  Its instruction
    // stream is a chain of dependent instructions on the path P ready -> PV issued -> O / next S; as a warp-wide
    // loop with an elect and a warp sync per step and a descriptor built per MMA it took longer to ISSUE the 16 MMAs
    // of an S block than the tensor pipe takes to run them (the GEMM issue loops).
    pdl_wait();
    pdl_trigger();
    if (elect_one()) {
    constexpr uint32_t idesc_s = make_idesc_bf16(AT_ROWS, AT_KV);
    constexpr uint32_t idesc_o = make_idesc_bf16(AT_ROWS, AT_HD, /*b_mn_major=*/true);
    // shared-memory descriptors: everything but the 14-bit start address is constant
    const uint64_t kdesc_hi = make_sdesc_k128(0);                       // K block, K-major
    const uint64_t vdesc_hi = make_sdesc_mn128(0, AT_KV * 128, 1024);   // V block, MN-major: 4 hd chunks 8192 B apart (LBO), 8-key groups 1024 B apart (SBO)
    const uint32_t base16 = (base >> 4) & 0x3FFF;
    uint32_t rp = 0;  // ring entries consumed
    uint32_t g = 0;   // key blocks issued so far in this CTA (selects the S/P buffer and the barrier parities)
    uint32_t j = 0;   // segments started
#ifdef ROSA_TRACE
    const int lane = 0;   // AT_TRACE
    long long w_full = 0, w_p = 0;   // cycles this thread waited for ring data / for the softmax warps
#define AT_WAIT(acc, stmt) do { const long long t_ = clock64(); stmt; acc += clock64() - t_; } while (0)
#else
#define AT_WAIT(acc, stmt) do { stmt; } while (0)
#endif
    AttnSeg nxt = ld_seg(segs + seg_beg);
    for (int si = seg_beg; si < seg_end; ++si, ++j) {
      const AttnSeg sg = nxt;
      if (si + 1 < seg_end) nxt = ld_seg(segs + si + 1);
      const int n = sg.kb1 - sg.kb0;
      auto issue_s = [&](uint32_t gi) {  // S(gi) = Q K^T into S buffer gi&1 (overwrites P(gi-2), consumed by PV(gi-2))
        const int s = (int)(rp % AT_RING);
        AT_WAIT(w_full, mbar_wait(full(s), (rp / AT_RING) & 1));
        ++rp;
        tc_fence_after();
        const uint32_t k16 = base16 + (uint32_t)s * (AT_STAGE_BYTES >> 4);
        const uint32_t d_s = tmem_s + (gi & 1) * AT_KV;
#pragma unroll
        for (int kk = 0; kk < AT_HD / 16; ++kk)   // 64-column chunk kk >> 2 of the block (AT_KV * 128 B apart), 32 B per 16 columns
          umma_bf16_ts(d_s, tmem_q + kk * 8, kdesc_hi | (uint64_t)(k16 + (kk >> 2) * ((AT_KV * 128) >> 4) + (kk & 3) * 2), idesc_s, kk != 0);
        umma_commit(empty(s));
        umma_commit(s_full(gi & 1));
#ifdef ROSA_TRACE
        if (si == seg_beg && (gi - g == 6 || gi - g == 7)) g_attn_trace[blockIdx.x * 64 + 56 + (gi - g - 6) * 4 + 3] = clock64();   // S(i + 2) issued
#endif
      };
      // Q of this segment is in tensor memory (softmax warps); its two ring entries are free again
      mbar_wait(q_ready, j & 1);
      tc_fence_after();
      AT_TRACE(8 + 8 * j + 5);
      mbar_arrive(empty((int)(rp % AT_RING)));
      mbar_arrive(empty((int)((rp + 1) % AT_RING)));
      rp += 2;
      issue_s(g);
      for (int i = 0; i < n; ++i) {
        const uint32_t gi = g + i;
        if (i + 1 < n) issue_s(gi + 1);
        const int s = (int)(rp % AT_RING);
        AT_WAIT(w_full, mbar_wait(full(s), (rp / AT_RING) & 1));
        ++rp;
        if (i == 0 && j > 0) mbar_wait(o_empty, (j - 1) & 1);  // the previous segment's O has left tensor memory
#ifdef ROSA_TRACE
        if (si == seg_beg && (i == 4 || i == 5)) g_attn_trace[blockIdx.x * 64 + 56 + (i - 4) * 4 + 0] = clock64();   // about to wait for P(i)
#endif
        AT_WAIT(w_p, mbar_wait(p_full(gi & 1), (gi >> 1) & 1));
#ifdef ROSA_TRACE
        if (si == seg_beg && (i == 4 || i == 5)) g_attn_trace[blockIdx.x * 64 + 56 + (i - 4) * 4 + 1] = clock64();   // P(i) seen
#endif
        tc_fence_after();
        const uint32_t v16 = base16 + (uint32_t)s * (AT_STAGE_BYTES >> 4);
        const uint32_t a_p = tmem_s + (gi & 1) * AT_KV;
#pragma unroll
        for (int kk = 0; kk < AT_KV / 16; ++kk) {
          // A = P [128 x 64] bf16 in TMEM (8 columns per 16 keys): keys 16 kk .. 16 kk + 15 are columns 8 (kk & 1) of the
          // half (kk >> 1) that wrote them (32 columns apart); B = V block, 16 keys per MMA = 2048 B
          umma_bf16_ts(tmem_o, a_p + (kk >> 1) * 32 + (kk & 1) * 8, vdesc_hi | (uint64_t)(v16 + kk * (2048 >> 4)), idesc_o,
                       kk ? 1u : (uint32_t)(i != 0));
        }
        umma_commit(empty(s));
        umma_commit(pv_done(gi));
#ifdef ROSA_TRACE
        if (si == seg_beg && (i == 4 || i == 5)) g_attn_trace[blockIdx.x * 64 + 56 + (i - 4) * 4 + 2] = clock64();   // PV(i) issued
#endif
      }
      AT_TRACE(8 + 8 * j + 6);
      g += n;
    }
#ifdef ROSA_TRACE
    g_attn_trace[blockIdx.x * 64 + 3] = w_full; g_attn_trace[blockIdx.x * 64 + 4] = w_p;
#endif
    }
    __syncwarp();
  } else {
    // ---------------------------------------------------------- softmax + drain warps (2..9)
    // Two warps per TMEM lane quarter: a query row's 64 scores of a block are split 32 / 32 between
    // warp w (half 0) and warp w + 4 (half 1).  Both read all 64 scores for the row maximum
    // (so both take the same rescale decision) and keep separate partial row sums until the end.
    pdl_wait();
    pdl_trigger();
    if (warp == 2) AT_TRACE(1);
    const int q = warp & 3, set = (warp - 2) >> 2;     // set: does the softmax of the key blocks with (CTA-wide count) & 1 == set
    const int half = set;                              // which half of O's columns / of Q's chunks this warp moves
    const int r = q * 32 + lane;                       // query row of this thread
    const uint32_t lane_off = (uint32_t)(q * 32) << 16;
    float* ml = reinterpret_cast<float*>(smem_raw + (AT_RING * AT_STAGE_BYTES + AT_STG_BYTES));   // m[128], l[128]
    float* xch = ml;   // the drain's row-sum exchange [2 halves][128] uses the same kilobyte (see the drain)
    float* mref_sm = ml + 2 * AT_ROWS;                 // [128] the rows' reference after the latest block
    auto pv_wait = [&](uint32_t x) { mbar_wait(pv_done(x), (x >> 2) & 1); };   // PV(x) has completed
    auto exp2_int = [](float d) {   // 2^d for an integer d <= 0 (or -inf), exactly; 0 below the normal range
      return d < -126.f ? 0.f : __int_as_float(((int)d + 127) << 23);
    };
    const float c_log2 = rsqrtf((float)AT_HD) * 1.4426950408889634f;  // (1/sqrt(hd)) * log2(e)
    const bool issuer = warp == 2 && lane == 0;        // the thread that owns this CTA's bulk-copy groups
    // Q of a segment: shared memory (SW128 chunks of [128 rows x 128 B]) -> tensor memory, thread = row; this half's
    // two chunks are one ring entry (rq = ring position of the segment's first entry).  Called when every S MMA of
    // the previous segment has completed (its last s_full was waited on), so tmem_q is free.
    auto q_landed = [&](uint32_t rq) {   // warp-uniform: has this half's ring entry of the segment's Q arrived?
      const uint32_t e = rq + half;
      return __all_sync(0xffffffffu, mbar_try_wait(full((int)(e % AT_RING)), (e / AT_RING) & 1)) != 0;
    };
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
    bool flag_owed = false;     // issuer: a continuation's bulk copy is in flight; its ready flag is still to be set
    auto settle = [&]() {       // issuer: staging is no longer being read; a pending partial result gets published
      if (flag_owed) {
        bulk_wait_all();
        fence_proxy_async_all();
        st_release_gpu(part_flag + blockIdx.x, 1);
        flag_owed = false;
      } else {
        bulk_wait_read();
      }
    };
    auto fetch_partial = [&](int cta) {   // issuer: the partial result CTA `cta` has published -> staging
      settle();
      (void)ld_acquire_gpu(part_flag + cta);
      fence_proxy_async_all();
      mbar_expect_tx(part_full, (uint32_t)AT_PART_BYTES);
      bulk_load(stg, part + (size_t)cta * AT_PART_BYTES, (uint32_t)AT_PART_BYTES, part_full);
    };
    AttnSeg nxt = ld_seg(segs + seg_beg);
    copy_q(0);
    for (int si = seg_beg; si < seg_end; ++si) {
      const AttnSeg sg = nxt;
      if (si + 1 < seg_end) nxt = ld_seg(segs + si + 1);
      const int p = sg.p, L = sg.len, nbp = (L + AT_KV - 1) / AT_KV;
      const int n = sg.kb1 - sg.kb0;
      const bool merge = sg.n_part > 0;   // head segment of a cut item: always the last entry of the list
      rp += 2 + 2 * n;   // ring position of the next segment's Q
      bool part_issued = false;           // issuer: the partner's partial result is on its way into staging
      // Reference m (log2 units, an integer) and this warp's part of the row sum, relative to the reference at this
      // warp's last own block (m_own); the row's current reference travels through mref_sm from block to block.
      float m_own = -INFINITY, l_own = 0.f;
      for (int i = (int)((g ^ (uint32_t)set) & 1u); i < n; i += 2) {   // the blocks with (g + i) & 1 == set
        const uint32_t gi = g + i;
        const int sb = set, kb = sg.kb0 + i;
        const int n_tot = kb == nbp ? dm.H : min(AT_KV, L - kb * AT_KV);   // valid keys of the block
        // Housekeeping of the asynchronous copies by the issuing thread, off the critical path.
        //  * from the segment's second block on: the previous drain's copy out of staging is (almost certainly)
        //    complete, so a continuation's partial result is in global memory: publish it;
        //  * this thread's last block of the segment: staging may be overwritten by this segment's drain (every warp's
        //    drain follows the last PV, whose P needs this block's reference or P: both come after this point);
        //  * head of a cut item: as soon as the other CTA has published its partial, pull it into staging (the drain
        //    merges it in place).  The flag is polled with a relaxed load issued here and looked at after the block.
        int flag_seen = 0;
        if (issuer) {
          if (i >= 1 || i + 2 >= n) settle();
          if (merge && !part_issued) flag_seen = ld_relaxed_gpu(part_flag + sg.part0);
        }
        __syncwarp();
#ifdef ROSA_TRACE
#define AT_BLK(k) do { if ((warp == 2 || warp == 6) && (i == 4 || i == 5) && si == seg_beg) AT_TRACE((warp == 2 ? 40 : 48) + (k)); \
                       if ((warp == 2 || warp == 6) && (i == 6 || i == 7) && si == seg_beg && (k) == 0) AT_TRACE((warp == 2 ? 47 : 55)); } while (0)
#else
#define AT_BLK(k) do { } while (0)
#endif
        AT_BLK(0);
        // The row's reference after block gi - 1, from the other set's warp of this lane quarter.  It was published right
        // after that warp's row maximum, i.e. about when S(gi - 1) arrived: long before S(gi) does, so waiting for it and
        // reading it HERE takes the hand-over off the chain S ready -> P ready.  (Waited for at every block but the CTA's
        // first, so that nobody is ever more than one phase behind these barriers.)
        if (gi > 0) mbar_wait(hand(q, (int)((gi - 1) & 1)), ((gi - 1) >> 1) & 1);
        float m_ref = i > 0 ? mref_sm[r] : -INFINITY;
        mbar_wait(s_full(sb), (gi >> 1) & 1);
        tc_fence_after();
        AT_BLK(1);
        if (warp == 2 + 4 * (int)(g & 1) && i < 2) AT_TRACE(8 + 8 * (si - seg_beg) + 0);
        // The warp takes the block's whole rows (64 scores per thread): no exchange of the maximum, and the two
        // warps of a scheduler are in different phases of different blocks - one in its 64 ex2 per thread while the
        // other loads, reduces or stores - instead of both queueing on the SFU at the same moment.
        float sc[64];
        {
          uint32_t r0[32], r1[32];
          tmem_ld32(tmem_s + lane_off + sb * AT_KV, r0);
          tmem_ld32(tmem_s + lane_off + sb * AT_KV + 32, r1);
          tmem_ld_wait();
#pragma unroll
          for (int c = 0; c < 32; ++c) { sc[c] = __uint_as_float(r0[c]); sc[32 + c] = __uint_as_float(r1[c]); }
        }
        if (n_tot < AT_KV) {  // warp-uniform; only the last prefix block and the own-token block are ragged
#pragma unroll
          for (int c = 0; c < 64; ++c) sc[c] = c < n_tot ? sc[c] : -INFINITY;
        }
        float mo;
        {   // four independent chains (the serial one is 32 dependent 3-input maxima on the critical path)
          float m4[4] = {sc[0], sc[1], sc[2], sc[3]};
#pragma unroll
          for (int c = 4; c < 64; c += 4) {
#pragma unroll
            for (int x = 0; x < 4; ++x) m4[x] = fmaxf(m4[x], sc[c + x]);
          }
          mo = fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
        }
        // The reference is an INTEGER in the log2 domain: a different reference (another lazy-rescale history,
        // another cut of the key stream between CTAs: R27) then scales P, l and O by an exact power of two, so the
        // bf16 rounding of P - the dominant rounding of the whole attention step - is the same whichever way the
        // item was planned.  What is left between two plans is fp32 summation order and the 16-bit hand-over.
        const float m_blk = ceilf(mo * c_log2);
        AT_BLK(2);
        AT_BLK(3);
        float factor = 1.f;
        if (m_blk > m_ref + AT_RESCALE_THR) {            // the segment's first block always lands here
          factor = exp2_int(m_ref - m_blk);              // 2^(an integer <= -8), exactly; 0 on the first block
          m_ref = m_blk;
        }
        mref_sm[r] = m_ref;
        __syncwarp();
        if (lane == 0) mbar_arrive(hand(q, (int)(gi & 1)));
        if (i > 0 && __any_sync(0xffffffffu, factor != 1.f)) {  // rare: rescale this warp's rows of O (all 256 columns)
          pv_wait(gi - 1);
          tc_fence_after();                                     // O quiescent: PV(gi-1) done, PV(gi) needs this P
#pragma unroll 1
          for (int c = 0; c < 8; ++c) {
            uint32_t rr[32];
            tmem_ld32(tmem_o + lane_off + c * 32, rr);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 32; ++e) rr[e] = __float_as_uint(__uint_as_float(rr[e]) * factor);
            tmem_st32(tmem_o + lane_off + c * 32, rr);
          }
        }
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
        const float neg_m = -m_ref;
        // P row r: keys 32 h .. 32 h + 31 as 16 columns of bf16 pairs at columns 32 h of the S buffer (over scores this
        // thread already holds in registers): the A operand of PV(gi)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          uint32_t pk[16];
#pragma unroll
          for (int c = 0; c < 32; c += 2) {
            const float a = ex2_approx(fmaf(sc[32 * h + c], c_log2, neg_m)), b = ex2_approx(fmaf(sc[32 * h + c + 1], c_log2, neg_m));
            if (c & 2) { s2 += a; s3 += b; } else { s0 += a; s1 += b; }   // fixed order: four partial sums per thread
            __nv_bfloat162 v2 = __floats2bfloat162_rn(a, b);
            pk[c >> 1] = *reinterpret_cast<uint32_t*>(&v2);
          }
          tmem_st16(tmem_s + lane_off + sb * AT_KV + h * 32, pk);
        }
        AT_BLK(4);
        l_own = l_own * exp2_int(m_own - m_ref) + ((s0 + s1) + (s2 + s3));   // m_own = -inf on the first own block: 0 * 0
        m_own = m_ref;
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(p_full(sb));  // 128 arrivals on one barrier would serialise on the critical path
        AT_BLK(5);
        if (issuer && flag_seen != 0) { fetch_partial(sg.part0); part_issued = true; }
        __syncwarp();
      }
      g += n;
      if (warp == 2) AT_TRACE(8 + 8 * (si - seg_beg) + 1);
      // The next segment's Q goes into tensor memory BEFORE this segment's O is drained (if it has landed): its first
      // two S blocks then run on the tensor pipe while these warps drain.
      bool q_pending = si + 1 < seg_end;
      // tmem_q is free once every S MMA of this segment has completed: the warps of the set that did not take the last
      // block have not seen its s_full yet (one phase behind at most: they saw the hand-over that followed S(g - 2))
      if (q_pending && ((g - 1) & 1u) != (uint32_t)set) {
        mbar_wait(s_full((int)((g - 1) & 1u)), ((g - 1) >> 1) & 1);
        tc_fence_after();
      }
      if (q_pending && q_landed(rp)) { copy_q(rp); q_pending = false; }
      if (warp == 2) AT_TRACE(8 + 8 * (si - seg_beg) + 2);
      // ------------------------------------------------ drain.  Row r = (token jj, head a) with r = jj * 8 + a; each
      // half owns 128 of the 256 columns.  O leaves tensor memory as 16-bit values into the staging tile (normalised
      // by the row sum; a head segment first adds the other CTA's partial result, which is already in staging, in
      // place), O is released, and one thread hands the tile to the copy engine.
      if (merge && issuer && !part_issued) {   // the other CTA has not published yet: wait for it here
        for (uint32_t spin = 0; ld_acquire_gpu(part_flag + sg.part0) == 0; ++spin) {
          __nanosleep(64);
          if (spin > (1u << 24)) __trap();
        }
        fetch_partial(sg.part0);
      }
      __syncwarp();
      if (n == 1 && ((g - 1) & 1u) != 0u) {
        // the issuing thread's set had no block in this one-block segment: its settle (staging free) comes here, ahead
        // of everybody's staging writes
        if (issuer) settle();
        named_bar_sync(9, 256);
      }
      pv_wait(g - 1);   // the segment's last PV, hence all of them, has completed
      tc_fence_after();
      if (warp == 2) AT_TRACE(8 + 8 * (si - seg_beg) + 7);
      // The statistics kilobyte behind the staging tile serves three purposes in turn: a merge reads the other
      // segment's (m, l) from it, then the two warps of a row exchange their partial row sums through it, then a
      // continuation leaves its own (m, l) there for the bulk copy.  The pair barriers keep the three apart.
      float m_c = 0.f, l_c = 0.f;
      if (merge) {
        mbar_wait(part_full, 0);   // at most one merge per CTA (the last entry of its list)
        m_c = ml[r];
        l_c = ml[AT_ROWS + r];
      }
      named_bar_sync(1 + q, 64);   // both warps of the row are through their blocks: mref_sm holds the final reference
      const float m_ref = mref_sm[r];
      const float l_sum = l_own * exp2_int(m_own - m_ref);   // this set's part, brought to the final reference (0 if it had no block)
      xch[half * AT_ROWS + r] = l_sum;
      named_bar_sync(1 + q, 64);
      float l_tot = l_sum + xch[(half ^ 1) * AT_ROWS + r];
      named_bar_sync(1 + q, 64);
      float w_own = 1.f / l_tot, w_part = 0.f;
      if (merge) {
        const float m_new = fmaxf(m_ref, m_c);
        const float f_own = ex2_approx(m_ref - m_new), f_c = ex2_approx(m_c - m_new);
        const float l_new = l_tot * f_own + l_c * f_c;
        w_own = f_own / l_new;           // applied to this segment's unnormalised O
        w_part = l_c * f_c / l_new;      // applied to the other segment's normalised O
      } else if (sg.n_part < 0 && half == 0) {
        ml[r] = m_ref;                   // a continuation leaves its statistics behind the staging tile
        ml[AT_ROWS + r] = l_tot;
      }
      {
        uint32_t rbuf[2][32];  // the next chunk's TMEM load is in flight while this one is converted and stored
        tmem_ld32(tmem_o + lane_off + (half * 4) * 32, rbuf[0]);
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          const int c = half * 4 + cc;     // 32-column chunk; box c >> 1, 16-byte units (c & 1) * 4 .. + 3 of row r
          const uint32_t rowaddr = stg + (uint32_t)(c >> 1) * (AT_ROWS * 128) + (uint32_t)r * 128;
          uint32_t (&rr)[32] = rbuf[cc & 1];
          tmem_ld_wait();
          if (cc + 1 < 4) tmem_ld32(tmem_o + lane_off + (c + 1) * 32, rbuf[(cc + 1) & 1]);
          float v[32];
#pragma unroll
          for (int e = 0; e < 32; ++e) v[e] = __uint_as_float(rr[e]) * w_own;
          if (cc == 3) {  // this warp has read all of its part of O
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(o_empty);
          }
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const uint32_t addr = rowaddr + (uint32_t)((((c & 1) * 4 + x) ^ (r & 7)) << 4);
            if (merge) {
              uint32_t u[4];
              asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]) : "r"(addr));
#pragma unroll
              for (int y = 0; y < 4; ++y) {
                const uint16_t lo = (uint16_t)(u[y] & 0xffffu), hi = (uint16_t)(u[y] >> 16);
                v[8 * x + 2 * y] = fmaf(op2f(lo, dm.fp16), w_part, v[8 * x + 2 * y]);
                v[8 * x + 2 * y + 1] = fmaf(op2f(hi, dm.fp16), w_part, v[8 * x + 2 * y + 1]);
              }
            }
            const uint32_t a0 = pack_op2(v[8 * x + 0], v[8 * x + 1], dm.fp16), a1 = pack_op2(v[8 * x + 2], v[8 * x + 3], dm.fp16);
            const uint32_t a2 = pack_op2(v[8 * x + 4], v[8 * x + 5], dm.fp16), a3 = pack_op2(v[8 * x + 6], v[8 * x + 7], dm.fp16);
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a0), "r"(a1), "r"(a2), "r"(a3) : "memory");
          }
        }
      }
      if (warp == 2) AT_TRACE(8 + 8 * (si - seg_beg) + 3);
      if (sg.n_part < 0) {
        // continuation: the tile and its statistics go, verbatim, into this CTA's scratch slot: one bulk copy
        fence_proxy_async();              // this thread's staging writes -> visible to the copy engine
        named_bar_sync(9, 256);           // all eight warps have written their part of the tile
        if (issuer) {
          bulk_store(part + (size_t)blockIdx.x * AT_PART_BYTES, stg, (uint32_t)AT_PART_BYTES);
          bulk_commit();
          flag_owed = true;
        }
      } else {
        // head: this warp's 32 rows x 128 columns back out of staging, 8 lanes x 16 bytes per row (one 128-byte row
        // segment of o per 8 lanes, 4 rows per instruction); rows of tokens >= H are padding and are not stored
        __syncwarp();
        const int lr = lane >> 3, lu = lane & 7;
#pragma unroll
        for (int bb = 0; bb < 2; ++bb) {
          const int b = half * 2 + bb;
          uint4 ov[8];
#pragma unroll
          for (int x = 0; x < 8; ++x) {
            const int row = q * 32 + x * 4 + lr;
            const uint32_t addr = stg + (uint32_t)b * (AT_ROWS * 128) + (uint32_t)row * 128 + (uint32_t)((lu ^ (row & 7)) << 4);
            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(ov[x].x), "=r"(ov[x].y), "=r"(ov[x].z), "=r"(ov[x].w) : "r"(addr));
          }
#pragma unroll
          for (int x = 0; x < 8; ++x) {
            const int row = q * 32 + x * 4 + lr, jj = sg.tt * AT_TOK + (row >> 3);
            if (jj < dm.H)
              *reinterpret_cast<uint4*>(o + (size_t)(p * dm.H + jj) * dm.q_n + (row & 7) * AT_HD + b * 64 + lu * 8) = ov[x];
          }
        }
        if (merge) {   // every warp is done with the partner's data once it has left the drain loop: free the slot
          named_bar_sync(9, 256);
          if (issuer) st_release_gpu(part_flag + sg.part0, 0);
        }
      }
      if (q_pending) copy_q(rp);
      if (warp == 2) AT_TRACE(8 + 8 * (si - seg_beg) + 4);
    }
    if (issuer) {   // nothing of this CTA's may be in flight when it exits
      bulk_wait_all();
      if (flag_owed) {
        fence_proxy_async_all();
        st_release_gpu(part_flag + blockIdx.x, 1);
      }
    }
    if (warp == 2) AT_TRACE(2);
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
size_t tc_attn_part_bytes(int n_cta) { return (size_t)n_cta * AT_PART_BYTES; }
int tc_attn_tiles(const Dims& dm) { return (dm.H + AT_TOK - 1) / AT_TOK; }

// Stream-K work list of one Euler iteration: the first `n_active` robots (internal order) with prefix lengths
// len[p]; item (p, tt) has ceil(len/64) + 1 key blocks; every segment costs its blocks + kSegOvh units (Q load,
// drain).  The concatenated items are cut into equal shares for `n_cta` CTAs (fewer when there is little work:
// a share is at least kMinShare units); no segment is shorter than kMinSeg blocks and no item has more than 2
// segments (the head merges at most one partial result).  offs[c] .. offs[c+1] = segments of CTA c (offs has n_cta + 1 entries; CTAs without work get none).
// Cost model of the planners, in units of one 64-key block inside a running segment (~1.7k cycles): what a segment
// costs on top of its blocks (Q load and copy, pipeline refill, O drain: clock trace DESIGN.md section 5d).
constexpr double kSegOvh = 6.0;

// Stream-K over ROBOTS on GROUPS of tpr CTAs: CTA tpr g + t of group g handles tile t of the robots (and parts of
// robots) assigned to the group, so the tpr tiles of a robot run side by side, in lockstep (they cost the same),
// and the robot's K/V stream is read from HBM once and from L2 by the other tiles - whatever the batch size (a
// layer's prefix K/V stops fitting in L2 at B >= 128).  The concatenated key streams of the robots are cut into
// equal shares per group; a robot that straddles a cut is cut at the same key block for all its tiles: tile t's
// head segment ends the list of CTA tpr g + t, its continuation starts the list of CTA tpr (g + 1) + t.
static int attn_plan_cut(const Dims& dm, int n_active, const int* len, int n_cta, std::vector<AttnSeg>& segs, int* offs) {
  constexpr double kMinShare = 10.0;
  constexpr int kMinSeg = 2;
  const int tpr = tc_attn_tiles(dm);
  const size_t seg0 = segs.size();
  const int groups = n_cta / tpr;
  std::vector<std::vector<AttnSeg>> lists(n_cta);
  if (groups >= 1) {
    double total = 0.0;
    for (int p = 0; p < n_active; ++p) total += (len[p] + AT_KV - 1) / AT_KV + 1 + kSegOvh;
    const int used = (int)std::min<double>(groups, std::max(1.0, std::floor(total / kMinShare)));
    // units not yet assigned, counting one extra segment overhead for each of the used - 1 group boundaries still
    // ahead (most of them cut a robot in two); a boundary that falls between two robots gives its overhead back
    double left = total + kSegOvh * (used - 1);
    double target = left / used;  // share of the current group: re-derived at every group from what is left
    int g = 0;
    double acc = 0.0;
    auto next_group = [&](bool cut) {
      if (g + 1 < used) {
        if (!cut) left -= kSegOvh;
        ++g; acc = 0.0; target = left / (used - g);
      }
    };
    for (int p = 0; p < n_active; ++p) {
      const int nb = (len[p] + AT_KV - 1) / AT_KV + 1;
      int kb = 0, n_seg = 0;
      int head_g = -1;
      while (kb < nb) {
        const int rem = nb - kb;
        const double room = target - acc;
        int take = rem;
        if (g + 1 < used && rem + kSegOvh > room + 0.5 && n_seg < 1) {
          take = (int)std::floor(room - kSegOvh + 0.5);
          if (take < kMinSeg) {            // not worth starting here: the next group takes it
            if (acc > 0.0) { next_group(false); continue; }
            take = std::min(rem, kMinSeg);
          }
          if (rem - take < kMinSeg) take = rem;   // no crumbs at the end either
        }
        for (int tt = 0; tt < tpr; ++tt) {
          AttnSeg sg{};
          sg.p = p; sg.robot = p; sg.len = len[p]; sg.tt = (int16_t)tt; sg.kb0 = (int16_t)kb; sg.kb1 = (int16_t)(kb + take);
          sg.n_part = kb == 0 ? 0 : -1; sg.part0 = -1;
          if (kb > 0) {  // a continuation is the first entry of its CTA's list; the head segment of the same tile collects it
            AttnSeg& head = lists[head_g * tpr + tt].back();
            head.n_part = 1;
            head.part0 = (int16_t)(g * tpr + tt);
          }
          lists[g * tpr + tt].push_back(sg);
        }
        if (kb == 0) head_g = g;
        ++n_seg;
        kb += take;
        acc += take + kSegOvh;
        left -= take + kSegOvh;
        if (kb < nb || acc >= target - 0.5) next_group(kb < nb);
      }
    }
  }
  for (int c = 0; c < n_cta; ++c) {
    offs[c] = (int)segs.size();
    segs.insert(segs.end(), lists[c].begin(), lists[c].end());
  }
  offs[n_cta] = (int)segs.size();
  return (int)(segs.size() - seg0);
}

// The alternative without cuts: whole items, longest first, each to the CTA with the least work so far (LPT).
// No partial results, no merges; at most (longest + shortest) per CTA when there are up to two items per CTA.
static int attn_plan_whole(const Dims& dm, int n_active, const int* len, int n_cta, std::vector<AttnSeg>& segs, int* offs) {
  const int tpr = tc_attn_tiles(dm);
  const size_t seg0 = segs.size();
  std::vector<int> order(n_active);
  for (int p = 0; p < n_active; ++p) order[p] = p;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return len[a] > len[b]; });
  std::vector<double> load(n_cta, 0.0);
  std::vector<std::vector<AttnSeg>> lists(n_cta);
  // Robot-major: the tiles of one robot go to the (then) least loaded CTAs one after the other, i.e. to CTAs that
  // reach them at about the same time, so the robot's K/V is read from HBM once and from L2 by the other tiles
  // (at B >= 128 a layer's prefix K/V no longer fits in L2: tile-major order re-read it from HBM for every tile).
  for (int x = 0; x < n_active; ++x)
    for (int tt = 0; tt < tpr; ++tt) {
      const int p = order[x], nb = (len[p] + AT_KV - 1) / AT_KV + 1;
      int c = 0;
      for (int k = 1; k < n_cta; ++k) if (load[k] < load[c]) c = k;
      AttnSeg sg{};
      sg.p = p; sg.robot = p; sg.len = len[p]; sg.tt = (int16_t)tt; sg.kb0 = 0; sg.kb1 = (int16_t)nb; sg.n_part = 0; sg.part0 = -1;
      lists[c].push_back(sg);
      load[c] += nb + kSegOvh;
    }
  for (int c = 0; c < n_cta; ++c) {
    offs[c] = (int)segs.size();
    segs.insert(segs.end(), lists[c].begin(), lists[c].end());
  }
  offs[n_cta] = (int)segs.size();
  return (int)(segs.size() - seg0);
}

static double attn_plan_makespan(const std::vector<AttnSeg>& segs, size_t seg0, const int* offs, int n_cta) {
  double worst = 0.0;
  for (int c = 0; c < n_cta; ++c) {
    double t = 0.0;
    for (int i = offs[c]; i < offs[c + 1]; ++i)
      t += segs[i].kb1 - segs[i].kb0 + kSegOvh + (segs[i].n_part != 0 ? 1.5 : 0.0);   // a cut costs a partial hand-off on both sides
    worst = std::max(worst, t);
  }
  (void)seg0;
  return worst;
}

// Work list of one Euler iteration: both plans are built, the one whose busiest CTA is estimated to finish first is kept.
int attn_build_list(const Dims& dm, int n_active, const int* len, int n_cta, std::vector<AttnSeg>& segs, int* offs) {
  const size_t seg0 = segs.size();
  std::vector<AttnSeg> a(segs), b(segs);
  std::vector<int> oa(n_cta + 1), ob(n_cta + 1);
  attn_plan_cut(dm, n_active, len, n_cta, a, oa.data());
  attn_plan_whole(dm, n_active, len, n_cta, b, ob.data());
  const double ta = attn_plan_makespan(a, seg0, oa.data(), n_cta), tb2 = attn_plan_makespan(b, seg0, ob.data(), n_cta);
  const bool use_cut = a.size() > seg0 && ta < tb2;
  segs.swap(use_cut ? a : b);
  for (int c = 0; c <= n_cta; ++c) offs[c] = use_cut ? oa[c] : ob[c];
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
                           int M, const void* d_kv_maps, void* part, int* part_flag, int n_cta, cudaStream_t s) {
  static uint64_t configured = 0;
  if (first_use_on_device(configured)) {
    cudaError_t e = cudaFuncSetAttribute(k_attn_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, AT_SMEM);
    if (e != cudaSuccess) return e;
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
                  tb, layer, o, k_iter, (uint8_t*)part, part_flag);
}

}  // namespace rosa
