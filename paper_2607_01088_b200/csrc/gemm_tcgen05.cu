// tcgen05 / TMEM / TMA bf16 GEMM with fused epilogues (steps a1, a3+a4, a6, a7, a8 of the path).
//
//   C[M,N] = A[M,K] * W[N,K]^T   (A activations, W weights; both K-major bf16; fp32 accumulate)
//
// Persistent, warp-specialised, one CTA per SM:
//   warp 0      TMA producer: A tile [128 x 64] + W tile [BN x 64] per k-block into a ring of
//               SWIZZLE_128B stages, completion on "full" mbarriers
//   warp 1      MMA issuer: one lane issues 4 x tcgen05.mma (M=128, N=BN, K=16) per stage into a
//               TMEM accumulator; tcgen05.commit frees the stage ("empty") and, after the last
//               k-block, publishes the accumulator ("tmem full")
//   warps 2..5  epilogue: tcgen05.ld the accumulator (thread = one row, 32 columns at a time),
//               apply the fused epilogue, store to global, release the accumulator ("tmem empty")
// The accumulator is double-buffered in TMEM (2 x BN columns) so the epilogue of tile i overlaps
// the MMAs of tile i+1.
#include <map>
#include <mutex>

#include "device_math.cuh"
#include "rosa_internal.h"
#include "tc_common.cuh"

namespace rosa {

using namespace tc;

constexpr int BM = 128, BK = 64;
constexpr int kGemmThreads = 192;

template <int BN>
struct GemmCfg {
  static constexpr int STAGES = BN == 256 ? 4 : (BN == 128 ? 6 : 8);
  static constexpr int A_BYTES = BM * BK * 2;
  static constexpr int B_BYTES = BN * BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int SMEM = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
  static constexpr int TMEM_COLS = 2 * BN < 32 ? 32 : 2 * BN;
};

// 32 consecutive 16-bit outputs (fp16 or bf16 bits) = 64 contiguous bytes per thread
__device__ __forceinline__ void store_op16x32(uint16_t* dst, const float (&v)[32], int fp16) {
  uint4* d = reinterpret_cast<uint4*>(dst);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint4 u;
    u.x = pack_op2(v[8 * i + 0], v[8 * i + 1], fp16);
    u.y = pack_op2(v[8 * i + 2], v[8 * i + 3], fp16);
    u.z = pack_op2(v[8 * i + 4], v[8 * i + 5], fp16);
    u.w = pack_op2(v[8 * i + 6], v[8 * i + 7], fp16);
    d[i] = u;
  }
}
__device__ __forceinline__ void ld_acc32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  tmem_ld32(taddr, r);
  tmem_ld_wait();
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

template <int BN, int EPI>
__global__ void __launch_bounds__(kGemmThreads, 1)
k_gemm_tc(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int M, int N, int K,
          EpiArgs ea) {
  using Cfg = GemmCfg<BN>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + Cfg::STAGES * Cfg::STAGE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (Cfg::STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * Cfg::STAGES + 4);
  volatile uint32_t* tmem_slot_ptr =
      reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_lim = ea.m_active ? min(M, *ea.m_active) : M;
  const int n_m = (m_lim + BM - 1) / BM, n_n = N / BN;
  const int n_tiles = n_m * n_n, n_kb = K / BK;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tmA);
    prefetch_tensormap(&tmB);
    for (int s = 0; s < Cfg::STAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull_bar(a), 1);
      mbar_init(tempty_bar(a), 128);
    }
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == 0) {
    if (lane == 0) {  // ---------------- TMA producer
      int s = 0;
      uint32_t ph = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const int m0 = (t % n_m) * BM, n0 = (t / n_m) * BN;
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(empty_bar(s), ph ^ 1);
          mbar_expect_tx(full_bar(s), Cfg::STAGE_BYTES);
          const uint32_t a_dst = smem_base + s * Cfg::STAGE_BYTES;
          tma_load_2d(a_dst, &tmA, full_bar(s), kb * BK, m0);
          tma_load_2d(a_dst + Cfg::A_BYTES, &tmB, full_bar(s), kb * BK, n0);
          if (++s == Cfg::STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {  // ---------------- MMA issuer
      // fp16 operands: A/B format bits 0 instead of 1 (bf16)
      const uint32_t idesc = ea.in_fp16 ? (make_idesc_bf16(BM, BN) & ~((1u << 7) | (1u << 10))) : make_idesc_bf16(BM, BN);
      int s = 0, it = 0;
      uint32_t ph = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
        const int acc = it & 1;
        const uint32_t acc_ph = (it >> 1) & 1;
        mbar_wait(tempty_bar(acc), acc_ph ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN;
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(full_bar(s), ph);
          tc_fence_after();
          const uint32_t a_addr = smem_base + s * Cfg::STAGE_BYTES;
          const uint32_t b_addr = a_addr + Cfg::A_BYTES;
#pragma unroll
          for (int kk = 0; kk < BK / 16; ++kk) {
            umma_bf16(d_tmem, make_sdesc_k128(a_addr + kk * 32), make_sdesc_k128(b_addr + kk * 32), idesc,
                      (kb | kk) != 0);
          }
          umma_commit(empty_bar(s));
          if (++s == Cfg::STAGES) { s = 0; ph ^= 1; }
        }
        umma_commit(tfull_bar(acc));
      }
    }
  } else {  // ---------------- epilogue warps 2..5
    const int q = warp & 3;  // TMEM lane quarter this warp may access
    int it = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
      const int acc = it & 1;
      const uint32_t acc_ph = (it >> 1) & 1;
      const int m0 = (t % n_m) * BM, n0 = (t / n_m) * BN;
      const int row = m0 + q * 32 + lane;
      const bool ok = row < m_lim;
      mbar_wait(tfull_bar(acc), acc_ph);
      tc_fence_after();
      const uint32_t t_acc = tmem_base + ((uint32_t)(q * 32) << 16) + acc * BN;

      if constexpr (EPI == EPI_STORE_F32 || EPI == EPI_BIAS_F32 || EPI == EPI_RESID) {
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
          float v[32];
          ld_acc32(t_acc + c * 32, v);
          if (ok) {
            float4* dst = reinterpret_cast<float4*>(ea.out_f32 + (size_t)row * ea.ld_out + n0 + c * 32);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              float4 o = make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
              if constexpr (EPI == EPI_RESID) {
                const float4 h = dst[i];
                o.x += h.x; o.y += h.y; o.z += h.z; o.w += h.w;
              }
              if constexpr (EPI == EPI_BIAS_F32) {
                const float4 b = *reinterpret_cast<const float4*>(ea.bias + n0 + c * 32 + 4 * i);
                o.x += b.x; o.y += b.y; o.z += b.z; o.w += b.w;
              }
              dst[i] = o;
            }
          }
        }
      } else if constexpr (EPI == EPI_SWISH_ROWBIAS) {
        const float* rb = ea.rowbias + (size_t)((ok ? row : 0) / ea.H) * N + n0;
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
          float v[32];
          ld_acc32(t_acc + c * 32, v);
          if (ok) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const float4 b = *reinterpret_cast<const float4*>(rb + c * 32 + 4 * i);
              v[4 * i] = swish_f(v[4 * i] + b.x);
              v[4 * i + 1] = swish_f(v[4 * i + 1] + b.y);
              v[4 * i + 2] = swish_f(v[4 * i + 2] + b.z);
              v[4 * i + 3] = swish_f(v[4 * i + 3] + b.w);
            }
            store_op16x32((uint16_t*)ea.out16 + (size_t)row * ea.ld_out + n0 + c * 32, v, ea.out_fp16);
          }
        }
      } else if constexpr (EPI == EPI_ROPE) {
        // BN == head_dim: the tile is exactly one head; pairs (c, c + hd/2) are both in TMEM.
        static_assert(EPI != EPI_ROPE || BN == 256, "RoPE epilogue assumes BN == head_dim == 256");
        const bool rot = n0 < ea.rope_cols;
        int pos = 0;
        if (ok && rot) {
          const int p = row / ea.H;
          pos = ea.rlen[ea.ids[p]] + (row - p * ea.H);
        }
        const float2* tab = ea.rope_tab + (size_t)pos * (BN / 2);
#pragma unroll 1
        for (int c = 0; c < BN / 64; ++c) {
          float lo[32], hi[32];
          ld_acc32(t_acc + c * 32, lo);
          ld_acc32(t_acc + BN / 2 + c * 32, hi);
          if (ok) {
            if (rot) {
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                const float2 cs = tab[c * 32 + i];
                const float a = lo[i], b = hi[i];
                lo[i] = a * cs.x - b * cs.y;
                hi[i] = b * cs.x + a * cs.y;
              }
            }
            uint16_t* dst = (uint16_t*)ea.out16 + (size_t)row * ea.ld_out + n0 + c * 32;
            store_op16x32(dst, lo, 0);  // q/k/v feed the attention kernel: always bf16
            store_op16x32(dst + BN / 2, hi, 0);
          }
        }
      } else if constexpr (EPI == EPI_GEGLU) {
        // packed columns: [gate 64 | up 64] blocks (gu_blk = 64); output column = n/2 region
#pragma unroll 1
        for (int blk = 0; blk < BN / 128; ++blk) {
#pragma unroll 1
          for (int c = 0; c < 2; ++c) {
            float g[32], u[32];
            ld_acc32(t_acc + blk * 128 + c * 32, g);
            ld_acc32(t_acc + blk * 128 + 64 + c * 32, u);
            if (ok) {
#pragma unroll
              for (int i = 0; i < 32; ++i) g[i] = gelu_tanh_f(g[i]) * u[i];
              store_op16x32((uint16_t*)ea.out16 + (size_t)row * ea.ld_out + n0 / 2 + blk * 64 + c * 32, g, ea.out_fp16);
            }
          }
        }
      }
      tc_fence_before();
      mbar_arrive(tempty_bar(acc));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

// ------------------------------------------------------------------ host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  });
  return fn;
}

// 2-D K-major bf16 matrix [rows, K] -> tensor map with box [box_rows, 64], SWIZZLE_128B.
bool make_tmap_2d(CUtensorMap* tm, const void* ptr, uint64_t rows, uint64_t K, uint32_t box_rows, int fp16) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[2] = {K, rows};
  cuuint64_t strides[1] = {K * 2};
  cuuint32_t box[2] = {64, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(tm, fp16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// Generic tiled map over 16-bit elements, SWIZZLE_128B (inner box = 64 elements = 128 B).
// dims/box innermost first; strides_bytes has rank-1 entries (dims 1..rank-1).
bool encode_tmap(CUtensorMap* tm, const void* ptr, int rank, const uint64_t* dims, const uint64_t* strides_bytes,
                 const uint32_t* box) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t d[5], st[4];
  cuuint32_t b[5], es[5];
  for (int i = 0; i < rank; ++i) { d[i] = dims[i]; b[i] = box[i]; es[i] = 1; }
  for (int i = 0; i + 1 < rank; ++i) st[i] = strides_bytes[i];
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(ptr), d, st, b, es,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int num_sms() {
  static int n = 0;
  if (!n) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  }
  return n;
}

bool tc_gemm_supported(int N, int K) { return N % 64 == 0 && K % 64 == 0 && N >= 64; }

template <int BN, int EPI>
static cudaError_t launch_one(const op16* A, const op16* W, int M, int N, int K, const EpiArgs& a, cudaStream_t s) {
  using Cfg = GemmCfg<BN>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_gemm_tc<BN, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  CUtensorMap tmA, tmB;
  if (!make_tmap_2d(&tmA, A, (uint64_t)M, (uint64_t)K, BM, a.in_fp16) ||
      !make_tmap_2d(&tmB, W, (uint64_t)N, (uint64_t)K, BN, a.in_fp16))
    return cudaErrorInvalidValue;
  const int tiles = ((M + BM - 1) / BM) * (N / BN);
  const int grid = tiles < num_sms() ? tiles : num_sms();
  k_gemm_tc<BN, EPI><<<grid, kGemmThreads, Cfg::SMEM, s>>>(tmA, tmB, M, N, K, a);
  return cudaGetLastError();
}

cudaError_t launch_gemm_tc(Epi epi, const op16* A, const op16* W, int M, int N, int K, const EpiArgs& a,
                           cudaStream_t s) {
  switch (epi) {
    case EPI_STORE_F32:
      if (N % 256 == 0) return launch_one<256, EPI_STORE_F32>(A, W, M, N, K, a, s);
      if (N % 128 == 0) return launch_one<128, EPI_STORE_F32>(A, W, M, N, K, a, s);
      return launch_one<64, EPI_STORE_F32>(A, W, M, N, K, a, s);
    case EPI_SWISH_ROWBIAS:
      return N % 128 == 0 ? launch_one<128, EPI_SWISH_ROWBIAS>(A, W, M, N, K, a, s)
                          : launch_one<64, EPI_SWISH_ROWBIAS>(A, W, M, N, K, a, s);
    case EPI_BIAS_F32:
      return N % 128 == 0 ? launch_one<128, EPI_BIAS_F32>(A, W, M, N, K, a, s)
                          : launch_one<64, EPI_BIAS_F32>(A, W, M, N, K, a, s);
    case EPI_RESID:
      return N % 128 == 0 ? launch_one<128, EPI_RESID>(A, W, M, N, K, a, s)
                          : launch_one<64, EPI_RESID>(A, W, M, N, K, a, s);
    case EPI_ROPE:
      if (a.hd != 256 || N % 256) return cudaErrorNotSupported;
      return launch_one<256, EPI_ROPE>(A, W, M, N, K, a, s);
    case EPI_GEGLU:
      if (a.gu_blk != 64 || N % 256) return cudaErrorNotSupported;
      return launch_one<256, EPI_GEGLU>(A, W, M, N, K, a, s);
  }
  return cudaErrorNotSupported;
}

}  // namespace rosa
