// tcgen05 / TMEM / TMA GEMMs with fused epilogues (steps a1, a2+a3+a4, a6, a2+a7, a8, a9+a10 of the path).
//
//   C[M,N] = A[M,K] * W[N,K]^T   (A activations, W weights; both K-major fp16 or bf16; fp32 accumulate)
//
// Persistent, warp-specialised, one CTA per SM, 10 warps:
//   warp 0      TMA producer: A tile [128 x 64] + W tile per k-block into a ring of SWIZZLE_128B
//               stages, completion on "full" mbarriers
//   warp 1      MMA issuer: 4 x tcgen05.mma per k-block into a TMEM accumulator; tcgen05.commit frees the
//               stage ("empty") and, after the last k-block, publishes the accumulator ("tmem full")
//               Both run on ONE elected lane from start to end: each is a chain of dependent instructions, and what
//               it executes per k-block (not the tensor pipe, not the feed) bounded every tile narrower than 256
//               columns while the loops were warp-wide with an elect and a warp sync per k-block (DESIGN 5d).
//   warps 2..9  epilogue, two warps per TMEM lane quarter (half of the tile's columns each): tcgen05.ld,
//               fused epilogue (epilogue_tile below), coalesced global stores, release ("tmem empty")
// The accumulator is double-buffered in TMEM (2 x BN columns) so the epilogue of tile i overlaps the
// MMAs of tile i+1.  Two kernels share the pipeline: k_gemm_tc2 (CTA pairs, cta_group::2, 256-row tiles:
// the workhorse for M > 128) and k_gemm_tc (single CTA, 128-row tiles: small batches).
#include <algorithm>
#include <cstdlib>
#include <map>
#include <vector>
#include <mutex>

#include <type_traits>

#include "device_math.cuh"
#include "rosa_internal.h"
#include "tc_common.cuh"

namespace rosa {

using namespace tc;

bool make_tmap_2d(CUtensorMap* tm, const void* ptr, uint64_t rows, uint64_t K, uint32_t box_rows, int fp16);

constexpr int BM = 128, BK = 64;
constexpr int kGemmThreads = 320;      // warp 0 TMA, warp 1 MMA, warps 2..9 epilogue (two per TMEM lane quarter)
constexpr int kEpiWarps = 8;
constexpr int kScrFloats = 32 * 36;    // per epilogue warp: a 32 x 32 fp32 chunk, pitch 36

template <int BN>
struct GemmCfg {
  // The operand ring takes whatever the fixed parts leave of the 227 KB; the number of stages is a launch-time
  // value: a stage is [a_rows x 64] of A (a_rows = the launch's live rows rounded up to 8, at most 128; the TMA box
  // is that high) and [BN x 64] of W, so a launch with few rows gets more, shorter stages.
  static constexpr int MAX_STAGES = 16;
  static constexpr int A_BYTES = BM * BK * 2;
  static constexpr int B_BYTES = BN * BK * 2;
  static constexpr int FIXED = 1024 /*align slack*/ + 512 /*barriers*/ + kEpiWarps * kScrFloats * 4;
  static constexpr int RING = ((232448 - FIXED) / 1024) * 1024;
  static constexpr int SMEM = RING + FIXED;
  static_assert(RING >= 3 * (A_BYTES + B_BYTES), "three full stages");
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
template <bool FP16>
__device__ __forceinline__ uint32_t pack_op2_t(float lo, float hi) {  // pack_op2 with the format fixed at compile time
  if constexpr (FP16) {
    __half2 v = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
  } else {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
  }
}
__device__ __forceinline__ void ld_acc32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  tmem_ld32(taddr, r);
  tmem_ld_wait();
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// Fused RMSNorm (a2, R5): the A operand was the un-normalised residual h (16-bit copy) and the gain
// is folded into W, so the accumulator row only needs the scale r = rsqrt(mean(h^2) + eps); the
// producing GEMM left n_part partial sums of squares per row, added here in a fixed order.
// The partials are one per 32 consecutive columns of h (n_part = d / 32), whatever tile width produced them, and are
// added left to right: a row's statistics do not depend on the batch it was computed in (pin P2).
__device__ __forceinline__ float row_rscale(const EpiArgs& ea, int row) {
  if (!ea.ssq_in) return 1.f;
  float ss = 0.f;
  const float* p = ea.ssq_in + (size_t)row * ea.n_part;
  if ((ea.n_part & 3) == 0) {
    for (int i = 0; i < ea.n_part; i += 4) {
      const float4 v = *reinterpret_cast<const float4*>(p + i);
      ss += v.x; ss += v.y; ss += v.z; ss += v.w;
    }
  } else {
    for (int i = 0; i < ea.n_part; ++i) ss += p[i];
  }
  return rsqrtf(ss * ea.inv_d + ea.eps);
}

// ---------------------------------------------------------------- residual / bias tiles (a6, a8, a1)
// h <- h + acc (or acc + bias), its 16-bit copy (A operand of the next GEMM) and the sum of squares of each
// 32-column group of the new row (fused RMSNorm, a2).  One warp = 32 rows (its TMEM lane quarter) x half of the
// tile's columns, in 32-column chunks: TMEM gives thread = row, global memory wants lanes along columns, so a chunk
// is transposed through the warp's scratch and then handled 8 lanes x 4 columns per row, 4 rows per instruction.
// Interior rows take no masks; the 16-bit format is fixed at compile time; row offsets live in registers (the clock
// trace of round 1 showed this epilogue bound by instruction issue before that).
// Tried in round 2 and dropped: starting the accumulator as h (written into tensor memory by these warps before the
// tile's first MMA, for the first tiles before the dependency wait) so that the epilogue only writes.  The clock trace
// shows why it does not pay: the ~10k cycles after the last MMA are the 130 CTAs of the
// single-round launch storing 22 MB at the same time, not the residual loads; the preload delayed the first MMA and
// pulled 13 MB through L2 under the previous kernel's tail: +1 ms per call.
// 16-bit copy of h: fp16 saturates at the largest finite value instead of becoming inf (include/rosa.h: range of the
// residual stream in the default operand format; bf16 has the range of fp32).
template <bool FP16>
__device__ __forceinline__ uint32_t pack_h16(float lo, float hi) {
  if constexpr (FP16) {
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
  } else {
    return pack_op2_t<false>(lo, hi);
  }
}

template <int BN, int EPI, typename Release>
__device__ __forceinline__ void epilogue_tile_resid(const EpiArgs& ea, float* scr, uint32_t t_acc, int r0, int n0, int m_lim,
                                                    int N, int lane, int half, Release release) {
  constexpr int P = 36;
  constexpr int NCT = (BN + 31) / 32, NC0 = (NCT + 1) / 2;
  const int c_beg = half ? NC0 : 0, c_end = half ? NCT : NC0;
  const int lr = lane >> 3, lc = (lane & 7) * 4;
  const int n32 = N >> 5;
  int c_last = c_end - 1;   // last chunk of this warp that lies inside N (the last column tile may hang over)
  while (c_last >= c_beg && n0 + c_last * 32 >= N) --c_last;
  if (c_last < c_beg) { release(); return; }
  // FULL: all 32 rows live, 16-bit copy and statistics wanted (every tile of the path but the ragged last row block):
  // no predicates in the loop
  auto run = [&](auto fp16_tag, auto full_tag) {
    constexpr bool FP16 = decltype(fp16_tag)::value;
    constexpr bool FULL = decltype(full_tag)::value;
    uint32_t off[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) off[i] = (uint32_t)(i * 4 + lr) * (uint32_t)ea.ld_out;
    const bool b0 = lane & 1, b1 = lane & 2, b2 = lane & 4;
    const int srow = r0 + ((b0 ? 4 : 0) + (b1 ? 2 : 0) + (b2 ? 1 : 0)) * 4 + lr;   // the row whose statistics this lane ends up with
#pragma unroll 1
    for (int c = c_beg; c <= c_last; ++c) {
      const int col0 = n0 + c * 32;
      float* const gc = ea.out_f32 + (size_t)r0 * ea.ld_out + col0 + lc;
      uint16_t* const hc = (uint16_t*)ea.h16 + (size_t)r0 * ea.ld_out + col0 + lc;
      float4 hres[8];
      if constexpr (EPI == EPI_RESID) {  // requested first: the latency overlaps the accumulator load and the transpose
#pragma unroll
        for (int i = 0; i < 8; ++i)
          hres[i] = FULL || r0 + i * 4 + lr < m_lim ? *reinterpret_cast<const float4*>(gc + off[i]) : make_float4(0.f, 0.f, 0.f, 0.f);
      } else {
        const float4 b = *reinterpret_cast<const float4*>(ea.bias + col0 + lc);
#pragma unroll
        for (int i = 0; i < 8; ++i) hres[i] = b;
      }
      {
        float v[32];
        ld_acc32(t_acc + c * 32, v);
        if (c == c_last) release();
#pragma unroll
        for (int i = 0; i < 32; i += 4)
          *reinterpret_cast<float4*>(&scr[lane * P + i]) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
      }
      __syncwarp();
      float4 o[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) o[i] = *reinterpret_cast<const float4*>(&scr[(i * 4 + lr) * P + lc]);
      float sq[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        o[i].x += hres[i].x; o[i].y += hres[i].y; o[i].z += hres[i].z; o[i].w += hres[i].w;
        if (FULL || r0 + i * 4 + lr < m_lim) {
          *reinterpret_cast<float4*>(gc + off[i]) = o[i];
          if (FULL || ea.h16)
            *reinterpret_cast<uint2*>(hc + off[i]) = make_uint2(pack_h16<FP16>(o[i].x, o[i].y), pack_h16<FP16>(o[i].z, o[i].w));
        }
        sq[i] = o[i].x * o[i].x + o[i].y * o[i].y + o[i].z * o[i].z + o[i].w * o[i].w;
      }
      if (FULL || ea.ssq_out) {
        // One partial per 32-column group of the row: the 8 lanes of a row group hold 4 columns each of 8 rows;
        // a transposing butterfly (4 + 2 + 1 shuffles) leaves each lane with the group's sum for ONE row, added
        // in a fixed order whatever the tile width: the row statistics, and with them the whole result, do not
        // depend on the batch a robot is served in (pin P2).
        float w[4], u[2];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float send = b0 ? sq[j] : sq[j + 4], keep = b0 ? sq[j + 4] : sq[j];
          w[j] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const float send = b1 ? w[j] : w[j + 2], keep = b1 ? w[j + 2] : w[j];
          u[j] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
        }
        const float send = b2 ? u[0] : u[1], keep = b2 ? u[1] : u[0];
        const float tot = keep + __shfl_xor_sync(0xffffffffu, send, 4);
        if (FULL || srow < m_lim) ea.ssq_out[(size_t)srow * n32 + (col0 >> 5)] = tot;
      }
      __syncwarp();
    }
  };
  const bool full = r0 + 32 <= m_lim && ea.h16 && ea.ssq_out;
  if (ea.out_fp16) { if (full) run(std::true_type{}, std::true_type{}); else run(std::true_type{}, std::false_type{}); }
  else { if (full) run(std::false_type{}, std::true_type{}); else run(std::false_type{}, std::false_type{}); }
}

// What an epilogue warp fetches BEFORE it waits for its accumulator, so that the latency sits under the main
// loop instead of after it (clock trace, profiles/r1_gemm_epilogue_trace.md: the residual epilogue's h loads were
// four exposed round trips, 17k cycles of a 39k-cycle O-projection launch; the RoPE epilogue began with three
// dependent ones: ids -> rlen, the sum-of-squares partials, the cos/sin rows).
struct EpiPre {
  float rs;            // row_rscale of this thread's row (ROPE / GEGLU / FINAL)
  int posr;            // ROPE: position L_p + j of this thread's row
  float4 cs0[8], cs1[8];  // ROPE: (cos, sin) of the first 32-column chunk, rows i * 4 + lr, columns lc..lc+3
};
template <int BN, int EPI>
__device__ __forceinline__ void rope_load_cs(const EpiArgs& ea, int posr, int c, int lane, float4 (&cs0)[8], float4 (&cs1)[8]) {
  const int lr = lane >> 3, lc = (lane & 7) * 4;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int pos = __shfl_sync(0xffffffffu, posr, i * 4 + lr);
    const float4* tp = reinterpret_cast<const float4*>(ea.rope_tab + (size_t)pos * (BN / 2) + c * 32 + lc);
    cs0[i] = tp[0];
    cs1[i] = tp[1];
  }
}
template <int BN, int EPI>
__device__ __forceinline__ void epilogue_pre(EpiPre& pre, const EpiArgs& ea, int r0, int n0, int m_lim, int N, int lane, int half,
                                             bool same_rows = false) {   // same_rows: pre.rs / pre.posr are those of the previous tile's rows
  const int row = r0 + lane;
  const bool ok = row < m_lim;
  if constexpr (EPI == EPI_RESID) {
    // h (32 rows x half a tile of fp32) towards L2: the weights streamed since it was written may have pushed it out
    constexpr int NCT = (BN + 31) / 32, NC0 = (NCT + 1) / 2;
    const int c_beg = half ? NC0 : 0, c_end = half ? NCT : NC0;
    const int n_end = min(n0 + BN, N);
    if (ok) {
      const float* hp = ea.out_f32 + (size_t)row * ea.ld_out;
      for (int col = n0 + c_beg * 32; col < min(n0 + c_end * 32, n_end); col += 32)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(hp + col));
    }
  }
  if constexpr (EPI == EPI_ROPE || EPI == EPI_GEGLU || EPI == EPI_FINAL) { if (!same_rows) pre.rs = row_rscale(ea, ok ? row : 0); }
  if constexpr (EPI == EPI_ROPE) {
    if (!same_rows) {   // the position does not depend on the head: kept across the heads of a row block
      pre.posr = 0;
      if (ok) {
        const int p = row / ea.H;
        pre.posr = ea.rlen[ea.ids[p]] + (row - p * ea.H);
      }
    }
    if (n0 < ea.rope_cols)   // warp-uniform (one head per tile)
      rope_load_cs<BN, EPI>(ea, pre.posr, half * 2, lane, pre.cs0, pre.cs1);
  }
}

// Epilogue of one accumulator tile for one warp: its 32 rows (TMEM lane quarter) x ONE HALF of the
// tile's BN columns (`half`: the 8 epilogue warps are two per lane quarter).  `release()` is called
// once, as soon as this warp has read its part of the accumulator.
// TMEM -> registers is thread = row (tcgen05.ld 32x32b); global memory wants lanes along columns:
// the warp transposes 32 x 32 chunks through its private scratch `scr` (pitch 36 floats: 16-byte
// rows, conflict-free both ways) and then works with 8 lanes x 4 columns per row, 4 rows per
// instruction, so every global access is a coalesced 64..128-byte row segment.
template <int BN, int EPI, typename Release>
__device__ __forceinline__ void epilogue_tile(const EpiArgs& ea, EpiPre& pre, float* scr, uint32_t t_acc, int r0, int n0, int m_lim,
                                              int N, int lane, int half, Release release) {
  constexpr int P = 36;
  const int lr = lane >> 3, lc = (lane & 7) * 4;
  auto to_scratch = [&](const float (&v)[32]) {
#pragma unroll
    for (int i = 0; i < 32; i += 4)
      *reinterpret_cast<float4*>(&scr[lane * P + i]) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
  };
  auto from_scratch = [&](float4 (&o)[8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) o[i] = *reinterpret_cast<const float4*>(&scr[(i * 4 + lr) * P + lc]);
  };
  if constexpr (EPI == EPI_STORE_F32 || EPI == EPI_BIAS_F32 || EPI == EPI_RESID) {
    // Read-modify-write form, used where the accumulator cannot start as h: the plain store of the GEMM unit
    // test, and the adaptive-norm variant's gated residual h += gate * acc (R25).  Everything else goes through
    // epilogue_tile_resid above.  32-column chunks: half 0 takes the first NC0, half 1 the rest;
    // BN need not divide N: chunks at or beyond N are skipped (N is a multiple of 32).
    constexpr int NCT = (BN + 31) / 32, NC0 = (NCT + 1) / 2;
    const int c_beg = half ? NC0 : 0, c_end = half ? NCT : NC0;
    const int n32 = N >> 5;
    const bool want_h16 = EPI != EPI_STORE_F32 && ea.h16 != nullptr;
#pragma unroll 1
    for (int c = c_beg; c < c_end; ++c) {
      const int col = n0 + c * 32 + lc;
      const bool colok = n0 + c * 32 < N;
      float4 add = make_float4(0.f, 0.f, 0.f, 0.f);
      if constexpr (EPI == EPI_BIAS_F32) { if (colok) add = *reinterpret_cast<const float4*>(ea.bias + col); }
      float* gp = ea.out_f32 + (size_t)(r0 + lr) * ea.ld_out + col;
      uint16_t* hp = (uint16_t*)ea.h16 + (size_t)(r0 + lr) * ea.ld_out + col;
      const size_t step = (size_t)4 * ea.ld_out;
      // the residual rows are requested first: their latency overlaps the accumulator load and the transpose
      float4 hres[8];
      if constexpr (EPI == EPI_RESID) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
          hres[i] = colok && r0 + i * 4 + lr < m_lim ? *reinterpret_cast<const float4*>(gp + i * step)
                                                      : make_float4(0.f, 0.f, 0.f, 0.f);
      }
      {
        float v[32];
        ld_acc32(t_acc + c * 32, v);
        if (c == c_end - 1) release();
        to_scratch(v);
      }
      __syncwarp();
      float4 o[8];
      from_scratch(o);
      if constexpr (EPI == EPI_RESID) {
        if (ea.gate) {  // adaptive-norm variant (R25): per-robot gate on the sublayer output, h += gate * acc.
          // Addresses are clamped into range instead of predicated so the 8 loads issue back to back.
          const int colc = colok ? col : n0;
          float4 g[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int rr = min(r0 + i * 4 + lr, m_lim - 1);
            g[i] = *reinterpret_cast<const float4*>(ea.gate + (size_t)(rr / ea.H) * ea.gate_ld + colc);
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) { o[i].x *= g[i].x; o[i].y *= g[i].y; o[i].z *= g[i].z; o[i].w *= g[i].w; }
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) { o[i].x += hres[i].x; o[i].y += hres[i].y; o[i].z += hres[i].z; o[i].w += hres[i].w; }
      }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        o[i].x += add.x; o[i].y += add.y; o[i].z += add.z; o[i].w += add.w;
        const bool ok = colok && r0 + i * 4 + lr < m_lim;
        if (ok) {
          *reinterpret_cast<float4*>(gp + i * step) = o[i];
          if (want_h16)
            *reinterpret_cast<uint2*>(hp + i * step) =
                make_uint2(pack_op2(o[i].x, o[i].y, ea.out_fp16), pack_op2(o[i].z, o[i].w, ea.out_fp16));
        }
        if constexpr (EPI != EPI_STORE_F32) {
          if (ea.ssq_out) {  // one partial per 32-column group: the layout row_rscale reads
            float v = o[i].x * o[i].x + o[i].y * o[i].y + o[i].z * o[i].z + o[i].w * o[i].w;
            v += __shfl_xor_sync(0xffffffffu, v, 1);
            v += __shfl_xor_sync(0xffffffffu, v, 2);
            v += __shfl_xor_sync(0xffffffffu, v, 4);
            if ((lane & 7) == 0 && ok) ea.ssq_out[(size_t)(r0 + i * 4 + lr) * n32 + ((n0 >> 5) + c)] = v;
          }
        }
      }
      __syncwarp();
    }
  } else if constexpr (EPI == EPI_FINAL) {
    // a9 + a10: columns are action dimensions (N = 64 covers A <= 64): v = r acc + b_out, x += dt_p v
    static_assert(EPI != EPI_FINAL || BN == 64, "final projection uses one 64-column tile");
    const float rs = pre.rs;
    {
      float v[32];
      ld_acc32(t_acc + half * 32, v);
      release();
#pragma unroll
      for (int i = 0; i < 32; ++i) v[i] *= rs;
      to_scratch(v);
    }
    __syncwarp();
    float4 o[8];
    from_scratch(o);
    float* vel_out = ea.cp->vel;
    const int batch_ext = ea.cp->batch_ext;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int m = r0 + i * 4 + lr;
      if (m < m_lim) {
        const int p = m / ea.H, j = m - p * ea.H;
        const float dt = ea.dt[p];
        const float vv[4] = {o[i].x, o[i].y, o[i].z, o[i].w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int a = half * 32 + lc + e;
          if (a < ea.A) {
            const float v = vv[e] + ea.bias[a];
            float* xp = ea.x + (size_t)m * ea.A + a;
            *xp = fmaf(dt, v, *xp);
            if (vel_out) vel_out[(((size_t)ea.k_iter * batch_ext + ea.src[p]) * ea.H + j) * ea.A + a] = v;
          }
        }
      }
    }
    __syncwarp();
  } else if constexpr (EPI == EPI_ROPE) {
    // BN == head_dim: the tile is exactly one head; pairs (c, c + hd/2) are both in TMEM.  This
    // warp covers low columns [64 half, 64 half + 64) and their partners 128 further on.
    static_assert(EPI != EPI_ROPE || BN == 256, "RoPE epilogue assumes BN == head_dim == 256");
    const bool rot = n0 < ea.rope_cols;
    const float rs = pre.rs;
    const int posr = pre.posr;
    uint16_t* outp = (uint16_t*)ea.out16;
#pragma unroll 1
    for (int cc = 0; cc < 2; ++cc) {
      const int c = half * 2 + cc;  // 32-column chunk of the low half
      float4 lo[8], hi[8];
      {
        float v[32];
        ld_acc32(t_acc + c * 32, v);
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] *= rs;
        to_scratch(v);
        __syncwarp();
        from_scratch(lo);
        __syncwarp();
        ld_acc32(t_acc + BN / 2 + c * 32, v);
        if (cc == 1) release();
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] *= rs;
        to_scratch(v);
        __syncwarp();
        from_scratch(hi);
      }
      if (rot) {  // warp-uniform (one head per tile)
        // (cos, sin) of columns lc, lc+1 | lc+2, lc+3: chunk cc = 0 was loaded before the accumulator wait
        // (epilogue_pre), chunk 1 is requested below while chunk 0 is stored
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float4 a = lo[i], b = hi[i], cs0 = pre.cs0[i], cs1 = pre.cs1[i];
          lo[i].x = a.x * cs0.x - b.x * cs0.y; hi[i].x = b.x * cs0.x + a.x * cs0.y;
          lo[i].y = a.y * cs0.z - b.y * cs0.w; hi[i].y = b.y * cs0.z + a.y * cs0.w;
          lo[i].z = a.z * cs1.x - b.z * cs1.y; hi[i].z = b.z * cs1.x + a.z * cs1.y;
          lo[i].w = a.w * cs1.z - b.w * cs1.w; hi[i].w = b.w * cs1.z + a.w * cs1.w;
        }
        if (cc == 0) rope_load_cs<BN, EPI>(ea, posr, c + 1, lane, pre.cs0, pre.cs1);
      }
      uint16_t* dst = outp + (size_t)(r0 + lr) * ea.ld_out + n0 + c * 32 + lc;
      const size_t step = (size_t)4 * ea.ld_out;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (r0 + i * 4 + lr < m_lim) {  // q/k/v feed the attention kernel: always bf16
          *reinterpret_cast<uint2*>(dst + i * step) = make_uint2(pack_op2(lo[i].x, lo[i].y, 0), pack_op2(lo[i].z, lo[i].w, 0));
          *reinterpret_cast<uint2*>(dst + i * step + BN / 2) =
              make_uint2(pack_op2(hi[i].x, hi[i].y, 0), pack_op2(hi[i].z, hi[i].w, 0));
        }
      }
      __syncwarp();
    }
  } else if constexpr (EPI == EPI_GEGLU) {
    // packed columns: [gate 64 | up 64] blocks (gu_blk = 64) -> 64 outputs; this warp takes block `half`
    // BN = 256: two 128-column blocks, one per half-warp; BN = 128 (single-CTA kernel, small batches): one block,
    // each half-warp takes 32 of its 64 outputs
    static_assert(EPI != EPI_GEGLU || BN == 256 || BN == 128, "GeGLU epilogue: one or two 128-column blocks per tile");
    const float rs = pre.rs;
    uint16_t* outp = (uint16_t*)ea.out16;
    const int blk = BN == 256 ? half : 0;
    const int hh_beg = BN == 256 ? 0 : half, hh_end = BN == 256 ? 2 : half + 1;
    // The 32 x 32 chunk goes through the scratch as PACKED 16-bit pairs (pitch 20 words: conflict-free 16-byte writes): half the
    // shared-memory traffic of an fp32 transpose, and the main loop of the next tile is running on the same 128 B/clk
    uint32_t* scr16 = reinterpret_cast<uint32_t*>(scr);
    constexpr int P16 = 20;
    auto run = [&](auto fp16_tag) {
      constexpr bool FP16 = decltype(fp16_tag)::value;
#pragma unroll 1
      for (int hh = hh_beg; hh < hh_end; ++hh) {
        {
          float g[32], u[32];
          ld_acc32(t_acc + blk * 128 + hh * 32, g);
          ld_acc32(t_acc + blk * 128 + 64 + hh * 32, u);
          if (hh == hh_end - 1) release();
#pragma unroll
          for (int i = 0; i < 32; ++i) g[i] = gelu_tanh_f(g[i] * rs) * (u[i] * rs);
#pragma unroll
          for (int i = 0; i < 32; i += 8)
            *reinterpret_cast<uint4*>(&scr16[lane * P16 + (i >> 1)]) =
                make_uint4(pack_op2_t<FP16>(g[i], g[i + 1]), pack_op2_t<FP16>(g[i + 2], g[i + 3]),
                           pack_op2_t<FP16>(g[i + 4], g[i + 5]), pack_op2_t<FP16>(g[i + 6], g[i + 7]));
        }
        __syncwarp();
        uint2 o[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) o[i] = *reinterpret_cast<const uint2*>(&scr16[(i * 4 + lr) * P16 + (lc >> 1)]);
        uint16_t* dst = outp + (size_t)(r0 + lr) * ea.ld_out + n0 / 2 + blk * 64 + hh * 32 + lc;
        const size_t step = (size_t)4 * ea.ld_out;
#pragma unroll
        for (int i = 0; i < 8; ++i)
          if (r0 + i * 4 + lr < m_lim) *reinterpret_cast<uint2*>(dst + i * step) = o[i];
        __syncwarp();
      }
    };
    if (ea.out_fp16) run(std::true_type{}); else run(std::false_type{});   // warp-uniform
  }
}

// Role loops of the single-CTA kernel.  A stage of the ring holds KC consecutive k-blocks (64 columns each) of A and
// of W behind ONE full / empty barrier pair: the MMA issuer is one thread running dependent instructions, and what it
// spends per barrier round trip (wait, fence, commit, ring bookkeeping: ~200 cycles, measured) is amortised over KC
// times the MMAs.  Barrier slots: full[s] at 8 s, empty[s] at 8 (MAX_STAGES + s), then the two accumulator pairs.
template <int BN, int KC>
__device__ __forceinline__ void gemm1_producer(const CUtensorMap* tmA, const CUtensorMap* tmB, uint32_t smem_base,
                                               uint32_t bar_base, uint32_t a_chunk, int n_stages, int n_tiles, int n_m,
                                               int n_kb) {
  using Cfg = GemmCfg<BN>;
  const uint32_t a_span = a_chunk * KC, stage_bytes = a_span + Cfg::B_BYTES * KC;
  const bool issuer = elect_one();
  // weights do not depend on the previous kernel: the W tiles of the first ring-full of stages go out before the
  // dependency wait, the A tiles of the same stages after it (they complete the same barriers)
  const int pre = (int)blockIdx.x < n_tiles ? min(n_stages, n_kb) : 0;
  if (issuer) {
    const int n0 = ((int)blockIdx.x / n_m) * BN;
    for (int kb = 0; kb < pre; ++kb) {
      mbar_expect_tx(bar_base + 8u * kb, stage_bytes);
#pragma unroll
      for (int c = 0; c < KC; ++c)
        tma_load_2d(smem_base + kb * stage_bytes + a_span + c * Cfg::B_BYTES, tmB, bar_base + 8u * kb, (kb * KC + c) * BK, n0);
    }
  }
  pdl_wait();
  pdl_trigger();
  if (issuer) {
    int s = 0;
    uint32_t ph = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
      const int m0 = (t % n_m) * BM, n0 = (t / n_m) * BN;
      for (int kb = 0; kb < n_kb; ++kb) {
        const uint32_t full = bar_base + 8u * s;
        const uint32_t a_dst = smem_base + s * stage_bytes;
        const bool first_pass = t == (int)blockIdx.x && kb < pre;
        if (!first_pass) {
          mbar_wait_idle(bar_base + 8u * (Cfg::MAX_STAGES + s), ph ^ 1);
          mbar_expect_tx(full, stage_bytes);
        }
#pragma unroll
        for (int c = 0; c < KC; ++c) {
          tma_load_2d(a_dst + c * a_chunk, tmA, full, (kb * KC + c) * BK, m0);
          if (!first_pass) tma_load_2d(a_dst + a_span + c * Cfg::B_BYTES, tmB, full, (kb * KC + c) * BK, n0);
        }
        if (++s == n_stages) { s = 0; ph ^= 1; }
      }
    }
  }
  __syncwarp();
}

template <int BN, int KC>
__device__ __forceinline__ void gemm1_mma(uint32_t smem_base, uint32_t bar_base, uint32_t tmem_base, uint32_t idesc,
                                          uint32_t a_chunk, int n_stages, int n_tiles, int n_kb) {
  using Cfg = GemmCfg<BN>;
  const uint32_t tfull0 = bar_base + 8u * (2 * Cfg::MAX_STAGES), tempty0 = tfull0 + 16u;
  if (elect_one()) {
    // shared-memory descriptors (make_sdesc_k128): everything but the 14-bit start address is constant
    const uint64_t desc_hi = make_sdesc_k128(0);
    const uint32_t a_chunk16 = a_chunk >> 4, stage16 = (a_chunk * KC + Cfg::B_BYTES * KC) >> 4;
    const uint32_t base16 = (smem_base >> 4) & 0x3FFF;
    int s = 0, it = 0;
    uint32_t ph = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
      const int acc = it & 1;
      mbar_wait(tempty0 + 8u * acc, ((it >> 1) & 1) ^ 1);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + acc * BN;
      for (int kb = 0; kb < n_kb; ++kb) {
        mbar_wait(bar_base + 8u * s, ph);
        tc_fence_after();
        const uint32_t a16 = base16 + s * stage16, b16 = a16 + KC * a_chunk16;
#pragma unroll
        for (int c = 0; c < KC; ++c) {
#pragma unroll
          for (int kk = 0; kk < BK / 16; ++kk) {
            umma_bf16(d_tmem, desc_hi | (uint64_t)(a16 + c * a_chunk16 + kk * 2),
                      desc_hi | (uint64_t)(b16 + c * (Cfg::B_BYTES >> 4) + kk * 2), idesc, (c | kk) ? 1u : (uint32_t)(kb != 0));
          }
        }
        umma_commit(bar_base + 8u * (Cfg::MAX_STAGES + s));
        if (kb == n_kb - 1) umma_commit(tfull0 + 8u * acc);
        if (++s == n_stages) { s = 0; ph ^= 1; }
      }
    }
  }
  __syncwarp();
}

template <int BN, int EPI>
__global__ void __launch_bounds__(kGemmThreads, 1)
k_gemm_tc(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int M, int N, int K,
          int a_rows, int kc, EpiArgs ea) {
  using Cfg = GemmCfg<BN>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  // a_rows < 128: the MMA still reads 128 rows from a_addr; rows a_rows.. are whatever follows in shared memory (this
  // stage's W, the next stage).  They feed accumulator rows >= m_lim only, which no epilogue stores.
  // kc consecutive k-blocks of A and of W per stage (gemm1_producer)
  const uint32_t a_chunk = (uint32_t)a_rows * (BK * 2);        // a_rows % 8 == 0: a multiple of the swizzle atom
  const uint32_t stage_bytes = (a_chunk + Cfg::B_BYTES) * kc;
  const int n_stages = min(Cfg::MAX_STAGES, Cfg::RING / (int)stage_bytes);
  const uint32_t bar_base = smem_base + Cfg::RING;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (Cfg::MAX_STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::MAX_STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::MAX_STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * Cfg::MAX_STAGES + 4);
  volatile uint32_t* tmem_slot_ptr =
      reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_lim = ea.m_active ? min(M, *ea.m_active) : M;
  const int n_m = (m_lim + BM - 1) / BM, n_n = N / BN;
  const int n_tiles = n_m * n_n, n_kb = K / (BK * kc);

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tmA);
    prefetch_tensormap(&tmB);
    for (int s = 0; s < n_stages; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull_bar(a), 1);
      mbar_init(tempty_bar(a), kEpiWarps);
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
  // dependency wait: per role (the producer sends out its first W tiles before it, gemm1_producer); everything
  // above overlapped the previous kernel's tail
  if (warp != 0) { pdl_wait(); pdl_trigger(); }

  if (warp == 0) {  // ---------------- TMA producer
    if (kc == 4) gemm1_producer<BN, 4>(&tmA, &tmB, smem_base, bar_base, a_chunk, n_stages, n_tiles, n_m, n_kb);
    else if (kc == 2) gemm1_producer<BN, 2>(&tmA, &tmB, smem_base, bar_base, a_chunk, n_stages, n_tiles, n_m, n_kb);
    else gemm1_producer<BN, 1>(&tmA, &tmB, smem_base, bar_base, a_chunk, n_stages, n_tiles, n_m, n_kb);
  } else if (warp == 1) {  // ---------------- MMA issuer
    // fp16 operands: A/B format bits 0 instead of 1 (bf16)
    const uint32_t idesc = ea.in_fp16 ? (make_idesc_bf16(BM, BN) & ~((1u << 7) | (1u << 10))) : make_idesc_bf16(BM, BN);
    if (kc == 4) gemm1_mma<BN, 4>(smem_base, bar_base, tmem_base, idesc, a_chunk, n_stages, n_tiles, n_kb);
    else if (kc == 2) gemm1_mma<BN, 2>(smem_base, bar_base, tmem_base, idesc, a_chunk, n_stages, n_tiles, n_kb);
    else gemm1_mma<BN, 1>(smem_base, bar_base, tmem_base, idesc, a_chunk, n_stages, n_tiles, n_kb);
  } else {  // ---------------- epilogue warps 2..9
    const int q = warp & 3;            // TMEM lane quarter this warp may access
    const int half = (warp - 2) >> 2;  // which half of the tile's columns
    float* scr = reinterpret_cast<float*>(smem_raw + (bar_base + 512u - smem_u32(smem_raw))) + (warp - 2) * kScrFloats;
    int it = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
      const int acc = it & 1;
      const uint32_t acc_ph = (it >> 1) & 1;
      const int m0 = (t % n_m) * BM, n0 = (t / n_m) * BN;
      const int r0 = m0 + q * 32;            // first row of this warp
      EpiPre pre;
      epilogue_pre<BN, EPI>(pre, ea, r0, n0, m_lim, N, lane, half);
      mbar_wait_idle(tfull_bar(acc), acc_ph);
      tc_fence_after();
      const uint32_t t_acc = tmem_base + ((uint32_t)(q * 32) << 16) + acc * BN;
      auto release = [&] {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty_bar(acc));
      };
      if constexpr (EPI == EPI_RESID || EPI == EPI_BIAS_F32) {
        if (!ea.gate) {  // the adaptive-norm variant's gated residual takes the general form in epilogue_tile
          epilogue_tile_resid<BN, EPI>(ea, scr, t_acc, r0, n0, m_lim, N, lane, half, release);
          continue;
        }
      }
      epilogue_tile<BN, EPI>(ea, pre, scr, t_acc, r0, n0, m_lim, N, lane, half, release);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

// Measurement aid, compiled in only with -DROSA_TRACE: clock64 at the phases of CTAs 0 and 64 of the last pair-kernel
// launch of each class [class = 2 * EPI + (K > 2048)][CTA 0 | CTA 64][slot].
#ifdef ROSA_TRACE
__device__ long long g_gemm_trace[16 * 2 * 16];
#define GT_TRACE(slot) do { if ((blockIdx.x == 0 || blockIdx.x == 64) && lane == 0) \
  g_gemm_trace[((2 * EPI + (K > 2048)) * 2 + (blockIdx.x != 0)) * 16 + (slot)] = clock64(); } while (0)
extern "C" int rosa_trace_gemm(long long* host) { return (int)cudaMemcpyFromSymbol(host, g_gemm_trace, sizeof(g_gemm_trace)); }
#else
#define GT_TRACE(slot) do { } while (0)
#endif

// ------------------------------------------------------------------ CTA-pair variant (cta_group::2)
// Pair tile 256 x BN: CTA r of the cluster holds A rows [m0 + 128 r, +128) and B rows
// [n0 + (BN/2) r, +BN/2) of every k-block; ONE tcgen05.mma (M = 256) issued by the leader reads
// both CTAs' shared memory and writes each CTA's 128 x BN half of D into that CTA's tensor memory.
// Per CTA and k-block that is 16 KB + BN*64 B from L2 for 128 x BN x 64 MACs: a third less than
// the single-CTA tile, which is what bounds the single-CTA kernel (profiles/r1_gemm_notes.md).
template <int BN>
struct Gemm2Cfg {
  static_assert(BN % 16 == 0 && BN >= 64 && BN <= 256, "pair tile width");
  static constexpr int A_BYTES = BM * BK * 2;
  static constexpr int B_BYTES = (BN / 2) * BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;  // a multiple of 1024 for every BN % 16 == 0
  static constexpr int FIXED = 1024 + 256 + kEpiWarps * kScrFloats * 4;
  static constexpr int FIT = (232448 - FIXED) / STAGE_BYTES;
  static constexpr int STAGES = FIT > 8 ? 8 : FIT;
  static constexpr int SMEM = STAGES * STAGE_BYTES + FIXED;
  static constexpr int ACC_STRIDE = BN <= 64 ? 64 : (BN <= 128 ? 128 : 256);  // columns between the two accumulators
  static constexpr int TMEM_COLS = 2 * ACC_STRIDE;
};

template <int BN, int EPI>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kGemmThreads, 1)
k_gemm_tc2(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, int M, int N, int K,
           EpiArgs ea) {
  using Cfg = Gemm2Cfg<BN>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + Cfg::STAGES * Cfg::STAGE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };                        // used in the leader
  auto empty_bar = [&](int s) { return bar_base + 8u * (Cfg::STAGES + s); };       // both CTAs
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::STAGES + a); };   // both CTAs
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * Cfg::STAGES + 2 + a); };  // leader
  const uint32_t tmem_slot = bar_base + 8u * (2 * Cfg::STAGES + 4);
  volatile uint32_t* tmem_slot_ptr =
      reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  if (warp == 0) GT_TRACE(0);
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int m_lim = ea.m_active ? min(M, *ea.m_active) : M;
  const int n_m = (m_lim + 2 * BM - 1) / (2 * BM), n_n = (N + BN - 1) / BN;  // the last column tile may hang over N
  const int n_tiles = n_m * n_n, n_kb = K / BK;
  // Tile order.  Default: the k-th tile of a pair is pair + k n_pairs with the ROW block running fastest, so the pairs that
  // run side by side share a W tile.  RoPE launches (QKV: two tiles per pair at B = 64, the second tile's epilogue is
  // exposed): a pair takes CONSECUTIVE tiles with the COLUMN tile (head) running fastest, i.e. heads of the same row block,
  // so the second tile's epilogue reuses the rows' norm scale and position instead of waiting for three dependent loads
  // (robot id -> prefix length -> cos / sin rows) after the first tile's epilogue.
  constexpr bool kHeadFastest = EPI == EPI_ROPE;
  const int tpp = (n_tiles + n_pairs - 1) / n_pairs;   // tiles per pair (the last pairs may get fewer, or none)
  auto tile_of = [&](int k) { return kHeadFastest ? (k < tpp ? pair * tpp + k : n_tiles) : pair + k * n_pairs; };
  auto tile_mb = [&](int t) { return kHeadFastest ? t / n_n : t % n_m; };
  auto tile_nb = [&](int t) { return kHeadFastest ? t % n_n : t / n_m; };

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tmA);
    prefetch_tensormap(&tmB);
    for (int s = 0; s < Cfg::STAGES; ++s) {
      mbar_init(full_bar(s), 2);   // one arrive.expect_tx per CTA of the pair
      mbar_init(empty_bar(s), 1);  // tcgen05.commit (multicast)
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull_bar(a), 1);   // tcgen05.commit (multicast)
      mbar_init(tempty_bar(a), 2 * kEpiWarps);  // epilogue warps of both CTAs
    }
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc_cg2(tmem_slot, Cfg::TMEM_COLS);
    tmem_relinquish_cg2();
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();  // the peer's barriers are initialised before anything is signalled on them
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  if (warp == 0) GT_TRACE(1);
  // Dependency wait: per role.  The producer first sends out the W tiles of its first ring-full of stages (weights do
  // not depend on the previous kernel; the A tiles of the same stages follow after the wait and complete the same
  // barriers); everyone else waits here.  Everything above overlapped the previous kernel's tail.
  if (warp != 0) { pdl_wait(); pdl_trigger(); }

  // The two issue loops are each ONE thread's dependent instruction stream: what they execute per k-block bounds the
  // K loop of every tile narrower than the tensor pipe's 2 BN cycles, so they run on one elected lane from start to
  // end (no per-k-block elect / warp sync) with the descriptors' constant parts hoisted.
  if (warp == 0) {  // ---------------- TMA producer (both CTAs; completion counted in the leader)
    const bool issuer = elect_one();
    const uint32_t lfull0 = mapa_shared(full_bar(0), 0);
    const int pre = tile_of(0) < n_tiles ? min(Cfg::STAGES, n_kb) : 0;   // stages whose W tile goes out before the wait
    if (issuer) {
      const int n0 = tile_nb(tile_of(0)) * BN + (int)rank * (BN / 2);
      for (int kb = 0; kb < pre; ++kb) {
        mbar_expect_tx_cluster(lfull0 + 8u * kb, Cfg::STAGE_BYTES);
        tma_load_2d_cg2(smem_base + kb * Cfg::STAGE_BYTES + Cfg::A_BYTES, &tmB, lfull0 + 8u * kb, kb * BK, n0);
      }
    }
    pdl_wait();
    pdl_trigger();
    GT_TRACE(2);
    if (issuer) {
      const int lane = 0;  // GT_TRACE
      (void)lane;
      int s = 0;
      uint32_t ph = 0;
      for (int k = 0, t; (t = tile_of(k)) < n_tiles; ++k) {
        const int m0 = tile_mb(t) * (2 * BM) + (int)rank * BM, n0 = tile_nb(t) * BN + (int)rank * (BN / 2);
        for (int kb = 0; kb < n_kb; ++kb) {
          const uint32_t lfull = lfull0 + 8u * s;
          const uint32_t a_dst = smem_base + s * Cfg::STAGE_BYTES;
          if (k == 0 && kb < pre) {   // first pass over the ring: stage free, W already on its way
            if (kb == 0) GT_TRACE(10);
            tma_load_2d_cg2(a_dst, &tmA, lfull, kb * BK, m0);
          } else {
            mbar_wait_idle(empty_bar(s), ph ^ 1);
            mbar_expect_tx_cluster(lfull, Cfg::STAGE_BYTES);
            tma_load_2d_cg2(a_dst, &tmA, lfull, kb * BK, m0);
            tma_load_2d_cg2(a_dst + Cfg::A_BYTES, &tmB, lfull, kb * BK, n0);
          }
          if (++s == Cfg::STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    if (rank == 0 && elect_one()) {  // ---------------- MMA issuer (leader CTA only)
      const int lane = 0;  // GT_TRACE
      (void)lane;
      const uint32_t idesc =
          ea.in_fp16 ? (make_idesc_bf16(2 * BM, BN) & ~((1u << 7) | (1u << 10))) : make_idesc_bf16(2 * BM, BN);
      const uint64_t desc_hi = make_sdesc_k128(0);   // all but the 14-bit start address
      const uint32_t base16 = (smem_base >> 4) & 0x3FFF;
      int s = 0, it = 0;
      uint32_t ph = 0;
      for (; tile_of(it) < n_tiles; ++it) {
        const int acc = it & 1;
        const uint32_t acc_ph = (it >> 1) & 1;
        mbar_wait(tempty_bar(acc), acc_ph ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * Cfg::ACC_STRIDE;
        for (int kb = 0; kb < n_kb; ++kb) {
          mbar_wait(full_bar(s), ph);
          tc_fence_after();
          if (it == 0 && kb == 0) GT_TRACE(3);
          if (kb == n_kb - 1) GT_TRACE(4);
          if (it == 0 && kb == n_kb - 1) GT_TRACE(9);
          if (it == 0 && kb == 8) GT_TRACE(13);
          const uint32_t a16 = base16 + s * (Cfg::STAGE_BYTES >> 4), b16 = a16 + (Cfg::A_BYTES >> 4);
#pragma unroll
          for (int kk = 0; kk < BK / 16; ++kk) {
            umma_bf16_cg2(d_tmem, desc_hi | (uint64_t)(a16 + kk * 2), desc_hi | (uint64_t)(b16 + kk * 2), idesc,
                          kk ? 1u : (uint32_t)(kb != 0));
          }
          umma_commit_cg2(empty_bar(s));
          if (kb == n_kb - 1) umma_commit_cg2(tfull_bar(acc));
          if (++s == Cfg::STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else {  // ---------------- epilogue warps 2..9 (both CTAs, each on its own 128 rows)
    const int q = warp & 3;
    const int half = (warp - 2) >> 2;
    float* scr = reinterpret_cast<float*>(smem_raw + (bar_base + 256u - smem_u32(smem_raw))) + (warp - 2) * kScrFloats;
    int it = 0, mb_prev = -1;
    EpiPre pre;
    for (int t; (t = tile_of(it)) < n_tiles; ++it) {
      const int acc = it & 1;
      const uint32_t acc_ph = (it >> 1) & 1;
      const int mb = tile_mb(t);
      const int m0 = mb * (2 * BM) + (int)rank * BM, n0 = tile_nb(t) * BN;
      const int r0 = m0 + q * 32;
      epilogue_pre<BN, EPI>(pre, ea, r0, n0, m_lim, N, lane, half, /*same_rows=*/mb == mb_prev);
      mb_prev = mb;
      mbar_wait_idle(tfull_bar(acc), acc_ph);
      tc_fence_after();
      const uint32_t t_acc = tmem_base + ((uint32_t)(q * 32) << 16) + acc * Cfg::ACC_STRIDE;
      auto release = [&] {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(mapa_shared(tempty_bar(acc), 0));
      };
      if (warp == 2) GT_TRACE(5);
      if (warp == 2 && it == 0) GT_TRACE(11);
      if constexpr (EPI == EPI_RESID || EPI == EPI_BIAS_F32) {
        if (!ea.gate) {  // the adaptive-norm variant's gated residual takes the general form in epilogue_tile
          epilogue_tile_resid<BN, EPI>(ea, scr, t_acc, r0, n0, m_lim, N, lane, half, release);
          continue;
        }
      }
      epilogue_tile<BN, EPI>(ea, pre, scr, t_acc, r0, n0, m_lim, N, lane, half, release);
      if (warp == 2) GT_TRACE(6);
      if (warp == 2 && it == 0) GT_TRACE(12);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) GT_TRACE(7);
  cluster_sync_all();  // the leader's MMAs read the peer's shared memory; nobody leaves early
  if (warp == 0) GT_TRACE(8);
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_cg2(tmem_base, Cfg::TMEM_COLS);
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

// SM count of the CURRENT device (cached per device: a process may hold experts on several GPUs)
int num_sms() {
  static int n[64] = {};
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64) dev = 0;
  if (!n[dev]) cudaDeviceGetAttribute(&n[dev], cudaDevAttrMultiProcessorCount, dev);
  return n[dev];
}
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: true the first time `flags` is asked on the current one
bool first_use_on_device(uint64_t& flags) {
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64) return true;
  const bool first = !((flags >> dev) & 1u);
  flags |= (uint64_t)1 << dev;
  return first;
}

bool tc_gemm_supported(int N, int K) { return N % 64 == 0 && K % 64 == 0 && N >= 64; }
// CTA pairs (256-row tiles) once there is more than one 128-row tile of tokens
static bool use_pair(int M) { return M > BM; }
bool tc_use_pair(int M) { return use_pair(M); }
// N tile of the EPI_BIAS_F32 / EPI_RESID launches.
// Single CTA (M <= 128): latency-bound (a serial K loop per tile), so narrower tiles are chosen until about
// half of the CTAs have a tile.
// CTA pairs: these GEMMs have few tiles (N = d), so whole rounds of tiles over the pairs decide the time:
// 13 row blocks x 4 tiles of 256 columns leave 22 of 74 pairs idle, 13 x 5 tiles of 208 do not.  The width
// is the candidate with the least rounds x (time per k-block + fixed cost per tile), where a k-block costs
// max(MMA time ~ 2 BN, operand feed ~ 288 + BN) cycles (the L2 -> shared-memory feed bounds narrow tiles;
// measured: profiles/r1_gemm_tile_width.md).
static const int kPairBn[] = {256, 224, 192, 160, 128, 96, 64};
static int resid_bn(int N, int M) {
  if (!use_pair(M)) {
    const int units = num_sms(), n_m = (M + BM - 1) / BM;
    for (int bn = 128; bn > 64; bn >>= 1)
      if (N % bn == 0 && n_m * (N / bn) * 2 >= units) return bn;
    return 64;
  }
  const int pairs = num_sms() / 2, n_m = (M + 2 * BM - 1) / (2 * BM);
  int best = 256;
  long best_cost = -1;
  for (int bn : kPairBn) {
    const int tiles = n_m * ((N + bn - 1) / bn);
    const long rounds = (tiles + pairs - 1) / pairs;
    const long per_kb = 2 * bn > 288 + bn ? 2 * bn : 288 + bn;
    const long cost = rounds * (per_kb * 32 + 4000);  // 32 k-blocks (K = 2048) as the reference depth
    if (best_cost < 0 || cost < best_cost) { best = bn; best_cost = cost; }
  }
  return best;
}
// sum-of-squares partials per row written by the residual / bias launches: one per 32 columns, whatever the tile width
int tc_ssq_parts(int N) { return N / 32; }
int tc_resid_bn(int N, int M) { return resid_bn(N, M); }

template <int BN, int EPI>
static cudaError_t launch_one(const op16* A, const op16* W, int M, int N, int K, const EpiArgs& a, cudaStream_t s) {
  using Cfg = GemmCfg<BN>;
  static uint64_t configured = 0;
  if (first_use_on_device(configured)) {
    cudaError_t e = cudaFuncSetAttribute(k_gemm_tc<BN, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM);
    if (e != cudaSuccess) return e;
  }
  CUtensorMap tmA, tmB;
  // one row block of fewer than 128 rows: load only those rows (rounded up to the swizzle's 8-row period)
  const int a_rows = M < BM ? (M + 7) / 8 * 8 : BM;
  // k-blocks per stage (gemm1_mma): 4, 2 or 1, as many as divide K and still leave three stages in the ring
  int kc = 1;
  while (kc < 4 && K % (BK * kc * 2) == 0 && Cfg::RING / ((a_rows * BK * 2 + Cfg::B_BYTES) * kc * 2) >= 3) kc *= 2;
  if (!make_tmap_2d(&tmA, A, (uint64_t)M, (uint64_t)K, (uint32_t)a_rows, a.in_fp16) ||
      !make_tmap_2d(&tmB, W, (uint64_t)N, (uint64_t)K, BN, a.in_fp16))
    return cudaErrorInvalidValue;
  const int tiles = ((M + BM - 1) / BM) * (N / BN);
  const int grid = tiles < num_sms() ? tiles : num_sms();
  return launch_k(k_gemm_tc<BN, EPI>, dim3(grid), dim3(kGemmThreads), Cfg::SMEM, s, tmA, tmB, M, N, K, a_rows, kc, a);
}

template <int BN, int EPI>
static cudaError_t launch_two(const op16* A, const op16* W, int M, int N, int K, const EpiArgs& a, cudaStream_t s) {
  using Cfg = Gemm2Cfg<BN>;
  static uint64_t configured = 0;
  if (first_use_on_device(configured)) {
    cudaError_t e = cudaFuncSetAttribute(k_gemm_tc2<BN, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM);
    if (e != cudaSuccess) return e;
  }
  CUtensorMap tmA, tmB;
  if (!make_tmap_2d(&tmA, A, (uint64_t)M, (uint64_t)K, BM, a.in_fp16) ||
      !make_tmap_2d(&tmB, W, (uint64_t)N, (uint64_t)K, BN / 2, a.in_fp16))
    return cudaErrorInvalidValue;
  const int tiles = ((M + 2 * BM - 1) / (2 * BM)) * ((N + BN - 1) / BN);
  const int pairs = tiles < num_sms() / 2 ? tiles : num_sms() / 2;
  return launch_k(k_gemm_tc2<BN, EPI>, dim3(2 * pairs), dim3(kGemmThreads), Cfg::SMEM, s, tmA, tmB, M, N, K, a);
}

template <int EPI>
static cudaError_t launch_by_n(const op16* A, const op16* W, int M, int N, int K, const EpiArgs& a, cudaStream_t s) {
  const bool pair = a.force_pair ? a.force_pair == 2 : use_pair(M);
  const int bn = a.force_bn ? a.force_bn : resid_bn(N, M);
  if (pair) {
    switch (bn) {
      case 256: return launch_two<256, EPI>(A, W, M, N, K, a, s);
      case 224: return launch_two<224, EPI>(A, W, M, N, K, a, s);
      case 192: return launch_two<192, EPI>(A, W, M, N, K, a, s);
      case 160: return launch_two<160, EPI>(A, W, M, N, K, a, s);
      case 128: return launch_two<128, EPI>(A, W, M, N, K, a, s);
      case 96: return launch_two<96, EPI>(A, W, M, N, K, a, s);
      case 64: return launch_two<64, EPI>(A, W, M, N, K, a, s);
      default: return cudaErrorNotSupported;
    }
  }
  if (N % bn) return cudaErrorNotSupported;   // the single-CTA kernel has no masked column tile
  if (bn == 256) return launch_one<256, EPI>(A, W, M, N, K, a, s);
  if (bn == 128) return launch_one<128, EPI>(A, W, M, N, K, a, s);
  if (bn == 64) return launch_one<64, EPI>(A, W, M, N, K, a, s);
  return cudaErrorNotSupported;
}

cudaError_t launch_gemm_tc(Epi epi, const op16* A, const op16* W, int M, int N, int K, const EpiArgs& a,
                           cudaStream_t s) {
  switch (epi) {
    case EPI_STORE_F32: return launch_by_n<EPI_STORE_F32>(A, W, M, N, K, a, s);
    case EPI_BIAS_F32: return launch_by_n<EPI_BIAS_F32>(A, W, M, N, K, a, s);
    case EPI_RESID: return launch_by_n<EPI_RESID>(A, W, M, N, K, a, s);
    case EPI_FINAL:
      if (N != 64) return cudaErrorNotSupported;
      return use_pair(M) ? launch_two<64, EPI_FINAL>(A, W, M, N, K, a, s) : launch_one<64, EPI_FINAL>(A, W, M, N, K, a, s);
    case EPI_ROPE:
      if (a.hd != 256 || N % 256) return cudaErrorNotSupported;
      return use_pair(M) ? launch_two<256, EPI_ROPE>(A, W, M, N, K, a, s) : launch_one<256, EPI_ROPE>(A, W, M, N, K, a, s);
    case EPI_GEGLU:
      if (a.gu_blk != 64 || N % 256) return cudaErrorNotSupported;
      // M <= 128: 128-column tiles (5 stages of 32 KB, twice the CTAs) halve the latency-bound K loop of a tile
      return use_pair(M) ? launch_two<256, EPI_GEGLU>(A, W, M, N, K, a, s)
                         : launch_one<128, EPI_GEGLU>(A, W, M, N, K, a, s);
  }
  return cudaErrorNotSupported;
}

}  // namespace rosa
