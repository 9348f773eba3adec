// Ragged-KV GQA attention on tcgen05 (step a5 of the path).
//
// One CTA per (robot p, tile of 16 action tokens).  All n_q = 8 query heads share the single KV
// head, so the tile's 16 tokens x 8 heads = 128 query rows form ONE M=128 operand against the
// robot's key/value stream [prefix K/V (L_p rows, from the bound cache) ; own k/v (H rows, from
// the qkv buffer)], walked in blocks of 64 keys:
//     S = Q K_blk^T           tcgen05.mma  M=128 N=64  K=256   (S double-buffered in TMEM)
//     P = exp2(S*c - m_ref)   4 softmax warps, thread = query row, running (m_ref, l) in registers
//     O += P V_blk            tcgen05.mma  M=128 N=256 K=64    (V is the MN-major B operand)
// K/V blocks arrive by TMA (per-robot tensor maps made at bind time bound the ragged length:
// rows >= L_p are zero-filled and masked).  O stays in TMEM for the whole key stream; it is
// rescaled only when a row maximum grows by more than 2^8 (lazy rescaling), which for the
// N(0,1)-like logits of this workload almost never happens after the first block.
#include "device_math.cuh"
#include "rosa_internal.h"
#include "tc_common.cuh"

namespace rosa {

using namespace tc;

constexpr int AT_HD = 256;        // head_dim
constexpr int AT_ROWS = 128;      // query rows per CTA = AT_TOK tokens x 8 heads
constexpr int AT_TOK = 16;
constexpr int AT_KV = 64;         // keys per block
constexpr int AT_THREADS = 192;   // warp 0 TMA, warp 1 MMA, warps 2..5 softmax/epilogue
constexpr int AT_Q_BYTES = AT_ROWS * AT_HD * 2;     // 64 KB: 4 chunks [128 x 64] SW128
constexpr int AT_KV_BYTES = AT_KV * AT_HD * 2;      // 32 KB: 4 chunks [64 x 64] SW128
constexpr int AT_P_BYTES = AT_ROWS * AT_KV * 2;     // 16 KB: [128 x 64] SW128
constexpr int AT_SMEM = AT_Q_BYTES + 4 * AT_KV_BYTES + AT_P_BYTES + 1024 + 256;
constexpr float AT_RESCALE_THR = 8.0f;              // log2 units

struct AttnMaps {
  CUtensorMap q;    // qkv buffer as [M tokens][8 heads][256]   box {64, 8, 16}
  CUtensorMap own;  // qkv buffer as [M tokens][qkv_n]          box {64, 64}
};

__global__ void __launch_bounds__(AT_THREADS, 1)
k_attn_tc(const __grid_constant__ AttnMaps maps, const CUtensorMap* __restrict__ kv_maps, Dims dm, Tables tb,
          int layer, op16* __restrict__ o, int k_iter, int tiles_per_robot) {
  extern __shared__ uint8_t smem_raw[];
  const int p = blockIdx.x / tiles_per_robot, tt = blockIdx.x % tiles_per_robot;
  if (p * dm.H >= tb.m_active[k_iter]) return;
  const int robot = tb.ids[p], L = tb.rlen[robot];
  const int nbp = (L + AT_KV - 1) / AT_KV, nb = nbp + 1;  // prefix blocks + one block of own tokens

  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t q_smem = base;
  const uint32_t k_smem = base + AT_Q_BYTES;                    // 2 stages
  const uint32_t v_smem = k_smem + 2 * AT_KV_BYTES;             // 2 stages
  const uint32_t p_smem = v_smem + 2 * AT_KV_BYTES;
  const uint32_t bars = p_smem + AT_P_BYTES;
  const uint32_t q_full = bars;
  auto k_full = [&](int s) { return bars + 8u * (1 + s); };
  auto k_empty = [&](int s) { return bars + 8u * (3 + s); };
  auto v_full = [&](int s) { return bars + 8u * (5 + s); };
  auto v_empty = [&](int s) { return bars + 8u * (7 + s); };
  auto s_full = [&](int s) { return bars + 8u * (9 + s); };
  auto s_empty = [&](int s) { return bars + 8u * (11 + s); };
  const uint32_t p_full = bars + 8u * 13, pv_done = bars + 8u * 14;
  const uint32_t tmem_slot = bars + 8u * 15;
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const CUtensorMap* kmap = kv_maps + ((size_t)robot * dm.layers + layer) * 2;
  const CUtensorMap* vmap = kmap + 1;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&maps.q);
    prefetch_tensormap(&maps.own);
    mbar_init(q_full, 1);
    for (int s = 0; s < 2; ++s) {
      mbar_init(k_full(s), 1); mbar_init(k_empty(s), 1);
      mbar_init(v_full(s), 1); mbar_init(v_empty(s), 1);
      mbar_init(s_full(s), 1); mbar_init(s_empty(s), 128);
    }
    mbar_init(p_full, 128);
    mbar_init(pv_done, 1);
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
  const uint32_t tmem_s = tmem_base + 256;      // columns [256, 384): S, 2 x 64

  const int tok0 = p * dm.H + tt * AT_TOK;      // first token row of this tile in the qkv buffer

  if (warp == 0) {
    if (lane == 0) {  // ------------------------------------------------ TMA producer
      mbar_expect_tx(q_full, AT_Q_BYTES);
      for (int c = 0; c < 4; ++c) tma_load_3d(q_smem + c * (AT_ROWS * 128), &maps.q, q_full, c * 64, 0, tok0);
      for (int i = 0; i < nb; ++i) {
        const int s = i & 1;
        const uint32_t ph = (i >> 1) & 1;
        const bool own = i == nbp;
        mbar_wait(k_empty(s), ph ^ 1);
        mbar_expect_tx(k_full(s), AT_KV_BYTES);
        for (int c = 0; c < 4; ++c) {
          const uint32_t dst = k_smem + s * AT_KV_BYTES + c * (AT_KV * 128);
          if (own) tma_load_2d(dst, &maps.own, k_full(s), dm.q_n + c * 64, p * dm.H);
          else tma_load_2d(dst, kmap, k_full(s), c * 64, i * AT_KV);
        }
        mbar_wait(v_empty(s), ph ^ 1);
        mbar_expect_tx(v_full(s), AT_KV_BYTES);
        for (int c = 0; c < 4; ++c) {
          const uint32_t dst = v_smem + s * AT_KV_BYTES + c * (AT_KV * 128);
          if (own) tma_load_2d(dst, &maps.own, v_full(s), dm.q_n + AT_HD + c * 64, p * dm.H);
          else tma_load_2d(dst, vmap, v_full(s), c * 64, i * AT_KV);
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {  // ------------------------------------------------ MMA issuer
      constexpr uint32_t idesc_s = make_idesc_bf16(AT_ROWS, AT_KV);
      constexpr uint32_t idesc_o = make_idesc_bf16(AT_ROWS, AT_HD, /*b_mn_major=*/true);
      auto issue_s = [&](int i) {  // S(i) = Q K_i^T into S buffer i&1
        const int s = i & 1;
        const uint32_t ph = (i >> 1) & 1;
        mbar_wait(k_full(s), ph);
        mbar_wait(s_empty(s), ph ^ 1);
        tc_fence_after();
#pragma unroll
        for (int kk = 0; kk < AT_HD / 16; ++kk) {
          const uint32_t qa = q_smem + (kk >> 2) * (AT_ROWS * 128) + (kk & 3) * 32;
          const uint32_t ka = k_smem + s * AT_KV_BYTES + (kk >> 2) * (AT_KV * 128) + (kk & 3) * 32;
          umma_bf16(tmem_s + s * AT_KV, make_sdesc_k128(qa), make_sdesc_k128(ka), idesc_s, kk != 0);
        }
        umma_commit(k_empty(s));
        umma_commit(s_full(s));
      };
      mbar_wait(q_full, 0);
      issue_s(0);
      for (int i = 0; i < nb; ++i) {
        if (i + 1 < nb) issue_s(i + 1);
        const int s = i & 1;
        mbar_wait(v_full(s), (i >> 1) & 1);
        mbar_wait(p_full, i & 1);
        tc_fence_after();
#pragma unroll
        for (int kk = 0; kk < AT_KV / 16; ++kk) {
          // A = P [128 x 64] K-major; B = V block, MN-major: 4 hd chunks 8192 B apart (LBO),
          // 8-key groups 1024 B apart (SBO); 16 keys per MMA = 2048 B
          const uint64_t a_desc = make_sdesc_k128(p_smem + kk * 32);
          const uint64_t b_desc = make_sdesc_mn128(v_smem + s * AT_KV_BYTES + kk * 2048, AT_KV * 128, 1024);
          umma_bf16(tmem_o, a_desc, b_desc, idesc_o, (i | kk) != 0);
        }
        umma_commit(v_empty(s));
        umma_commit(pv_done);
      }
    }
  } else {  // ---------------------------------------------------------- softmax + epilogue warps
    const int q = warp & 3;
    const int r = q * 32 + lane;                       // query row of this thread
    const uint32_t lane_off = (uint32_t)(q * 32) << 16;
    const float c_log2 = rsqrtf((float)AT_HD) * 1.4426950408889634f;  // (1/sqrt(hd)) * log2(e)
    float m_ref = -INFINITY, l_sum = 0.f;
    for (int i = 0; i < nb; ++i) {
      const int s = i & 1;
      const int n_valid = i == nbp ? dm.H : min(AT_KV, L - i * AT_KV);
      mbar_wait(s_full(s), (i >> 1) & 1);
      tc_fence_after();
      float sc[AT_KV];
      {
        uint32_t r0[32], r1[32];
        tmem_ld32(tmem_s + lane_off + s * AT_KV, r0);
        tmem_ld32(tmem_s + lane_off + s * AT_KV + 32, r1);
        tmem_ld_wait();
#pragma unroll
        for (int c = 0; c < 32; ++c) { sc[c] = __uint_as_float(r0[c]); sc[32 + c] = __uint_as_float(r1[c]); }
      }
      tc_fence_before();
      mbar_arrive(s_empty(s));
      float m_blk = -INFINITY;
#pragma unroll
      for (int c = 0; c < AT_KV; ++c) {
        sc[c] = c < n_valid ? sc[c] * c_log2 : -INFINITY;
        m_blk = fmaxf(m_blk, sc[c]);
      }
      float factor = 1.f;
      if (m_blk > m_ref + AT_RESCALE_THR) {            // first block always lands here
        factor = exp2f(m_ref - m_blk);                 // 0 on the first block (m_ref = -inf)
        m_ref = m_blk;
      }
      uint32_t pk[AT_KV / 2];
      float psum = 0.f;
#pragma unroll
      for (int c = 0; c < AT_KV; c += 2) {
        const float a = exp2f(sc[c] - m_ref), b = exp2f(sc[c + 1] - m_ref);
        psum += a + b;
        __nv_bfloat162 v2 = __floats2bfloat162_rn(a, b);
        pk[c >> 1] = *reinterpret_cast<uint32_t*>(&v2);
      }
      l_sum = l_sum * factor + psum;
      if (i > 0) {
        mbar_wait(pv_done, (i - 1) & 1);               // P buffer free, O quiescent
        tc_fence_after();
        if (__any_sync(0xffffffffu, factor != 1.f)) {  // rare: rescale this warp's 32 rows of O
#pragma unroll 1
          for (int c = 0; c < AT_HD / 32; ++c) {
            uint32_t rr[32];
            tmem_ld32(tmem_o + lane_off + c * 32, rr);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 32; ++e) rr[e] = __float_as_uint(__uint_as_float(rr[e]) * factor);
            tmem_st32(tmem_o + lane_off + c * 32, rr);
          }
          tmem_st_wait();
        }
      }
      // P row r -> shared memory, K-major SWIZZLE_128B: 16-byte chunk c at (c ^ (r & 7))
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const uint32_t addr = p_smem + r * 128 + ((c ^ (r & 7)) << 4);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(pk[4 * c]), "r"(pk[4 * c + 1]),
                     "r"(pk[4 * c + 2]), "r"(pk[4 * c + 3]) : "memory");
      }
      fence_proxy_async();
      tc_fence_before();
      mbar_arrive(p_full);
    }
    // epilogue: O / l -> o[(token, head)] ; row r = (token jj, head a) with r = jj * 8 + a
    mbar_wait(pv_done, (nb - 1) & 1);
    tc_fence_after();
    const int jj = r >> 3, a = r & 7, j = tt * AT_TOK + jj;
    const bool ok = j < dm.H;
    const float inv = 1.f / l_sum;
    uint16_t* dst = o + (size_t)(p * dm.H + (ok ? j : 0)) * dm.q_n + a * AT_HD;
#pragma unroll 1
    for (int c = 0; c < AT_HD / 32; ++c) {
      uint32_t rr[32];
      tmem_ld32(tmem_o + lane_off + c * 32, rr);
      tmem_ld_wait();
      if (ok) {
        uint4* d4 = reinterpret_cast<uint4*>(dst + c * 32);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          uint4 u;
          u.x = pack_op2(__uint_as_float(rr[8 * e + 0]) * inv, __uint_as_float(rr[8 * e + 1]) * inv, dm.fp16);
          u.y = pack_op2(__uint_as_float(rr[8 * e + 2]) * inv, __uint_as_float(rr[8 * e + 3]) * inv, dm.fp16);
          u.z = pack_op2(__uint_as_float(rr[8 * e + 4]) * inv, __uint_as_float(rr[8 * e + 5]) * inv, dm.fp16);
          u.w = pack_op2(__uint_as_float(rr[8 * e + 6]) * inv, __uint_as_float(rr[8 * e + 7]) * inv, dm.fp16);
          d4[e] = u;
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

// Tensor maps of one robot's prefix K and V of one layer: [len, 256] bf16, box {64, 64}.
// `out2` = two consecutive CUtensorMap (host memory).
bool tc_attn_make_prefix_maps(void* out2, const bf16* k, const bf16* v, int len, const Dims& dm) {
  CUtensorMap* m = (CUtensorMap*)out2;
  const uint64_t dims[2] = {(uint64_t)dm.hd, (uint64_t)len};
  const uint64_t strides[1] = {(uint64_t)dm.nkv * dm.hd * 2};
  const uint32_t box[2] = {64, AT_KV};
  return encode_tmap(&m[0], k, 2, dims, strides, box) && encode_tmap(&m[1], v, 2, dims, strides, box);
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
    const uint64_t dims[2] = {(uint64_t)dm.qkv_n, (uint64_t)M};
    const uint64_t strides[1] = {(uint64_t)dm.qkv_n * 2};
    const uint32_t box[2] = {64, AT_KV};
    if (!encode_tmap(&maps.own, qkv, 2, dims, strides, box)) return cudaErrorInvalidValue;
  }
  const int tpr = (dm.H + AT_TOK - 1) / AT_TOK;
  k_attn_tc<<<tb.batch * tpr, AT_THREADS, AT_SMEM, s>>>(maps, (const CUtensorMap*)d_kv_maps, dm, tb, layer, o,
                                                       k_iter, tpr);
  return cudaGetLastError();
}

}  // namespace rosa
