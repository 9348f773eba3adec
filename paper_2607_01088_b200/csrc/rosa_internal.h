// Internal declarations of librosa (not part of the ABI).  sm_100a only.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "rosa.h"
#include "rosa_debug.h"

typedef __nv_bfloat16 bf16;
typedef uint16_t op16;  // 16-bit GEMM operand storage: fp16 or bf16 bits, chosen per expert (Dims::fp16)

namespace rosa {

// Model dimensions in the paper/BASELINE notation.
struct Dims {
  int layers, d, nq, nkv, hd, F, H, A;
  int qkv_n;   // (nq + 2 nkv) * hd : packed [q heads | k heads | v heads]
  int q_n;     // nq * hd
  int gu_blk;  // gate/up interleave block: packed rows [b*2g, b*2g+g) = gate, next g = up
  int fp16;    // GEMM operands (weights + activations) held as fp16 (1) or bf16 (0); R19
  int ada;     // time conditioning by adaptive RMSNorm (reading R25) instead of the concatenated time MLP
  float rope_base, eps, pmin, pmax;
};

// Per-call device tables (internal batch order = robots sorted by n_steps, descending, so the
// active set of iteration k is the prefix [0, m_active[k]) of the token rows).
struct Tables {
  const int* ids;       // [B] robot id of internal position p
  const int* src;       // [B] index of p in the caller's noise/out arrays
  const float* t0;      // [B]
  const float* dt;      // [B]
  const int* nsteps;    // [B]
  const int* m_active;  // [max_steps] active token rows (= H * active robots) in iteration k
  // attention work lists (attn_tcgen05.cu): offs + attn_iter[k] = the n_cta + 1 segment offsets of iteration k
  const int* attn_iter;     // [max_steps]
  const int* attn_offs;
  const struct AttnSeg* attn_segs;
  const int* batch_dev;     // live robots of this call (<= batch, the graph's bucket)
  const bf16* const* rk;  // [max_robots * layers] prefix K pointer of (robot, layer)
  const bf16* const* rv;  // [max_robots * layers]
  const int* rlen;        // [max_robots]
  int batch;                // the captured graph's batch bucket: grids and row counts are sized for it
};

// One entry of a CTA's attention work list: key blocks [kb0, kb1) of item (robot position p, token tile tt).
// n_part >= 0: head segment (kb0 = 0): writes the output after merging the partials of CTAs part0 .. part0 + n_part - 1;
// n_part < 0: continuation: leaves its partial (O, m, l) in the scratch slot of its CTA.
// The record carries everything a role needs about the item (robot id, prefix length), so that walking the list
// costs one 32-byte load per segment, issued a segment ahead, instead of a chain of dependent table lookups.
struct AttnSeg {
  int32_t p, robot, len;
  int16_t tt, kb0, kb1, n_part, part0, pad0;
  int32_t pad1, pad2;
};
static_assert(sizeof(AttnSeg) == 32, "AttnSeg is copied to the device as 32-byte records");

// Caller pointers of the current call live in device memory so that a captured graph can be
// replayed for a different call (the kernels read them through this struct).
struct CallPtrs {
  const float* noise;  // [batch, H, A] caller order
  float* out;          // [batch, H, A] caller order
  float* vel;          // [nmax, batch, H, A] or null
  int batch_ext;
};

struct LayerWeights {
  op16 *wqkv, *wo, *wgu, *wdown;  // [qkv_n,d] [d,q_n] [2F,d] (interleaved) [d,F]; RMSNorm gains folded
                                  // into the columns of wqkv and wgu
};

// Epilogue selector shared by the CUDA-core path (separate elementwise kernels over an fp32
// scratch) and the tcgen05 path (fused into the GEMM).
enum Epi : int {
  EPI_STORE_F32 = 0,     // C fp32 = acc                     (debug GEMM)
  EPI_BIAS_F32 = 2,      // h fp32 = acc + bias[n]          (+ 16-bit copy and sum-of-squares partials)
  EPI_ROPE = 3,          // qkv bf16 = rope(r * acc) on q and k heads at pos = len + j; v = r * acc
  EPI_RESID = 4,         // h fp32 += acc                   (+ 16-bit copy and sum-of-squares partials)
  EPI_GEGLU = 5,         // out 16-bit [M, N/2] = gelu_tanh(r * gate) * (r * up) (interleaved columns)
  EPI_FINAL = 6          // a9 + a10: v = r * acc + b_out ; x += dt_p * v ; optional velocity export (N = 64 >= A)
};

struct EpiArgs {
  float* out_f32;         // EPI_STORE_F32 / BIAS_F32 / RESID
  void* out16;            // GEGLU: op16 (fp16 or bf16 per out_fp16); ROPE: bf16
  void* h16;              // BIAS_F32 / RESID (tcgen05 family): op16 copy of the new h, or null
  float* ssq_out;         // BIAS_F32 / RESID (tcgen05 family): [M, N / BN] partial sums of squares, or null
  const float* ssq_in;    // ROPE / GEGLU (tcgen05 family): partials of the A operand's rows, or null
  int n_part;             // partials per row in ssq_in
  float inv_d, eps;       // 1 / d_model, rms_eps
  int out_fp16;           // 16-bit output format: 1 = fp16, 0 = bf16
  int in_fp16;            // operand format of A and W
  const float* bias;      // BIAS_F32: [N]
  const float2* rope_tab; // ROPE: [max_pos, hd/2] (cos, sin)
  const int* ids;         // ROPE: Tables::ids
  const int* rlen;        // ROPE: Tables::rlen
  int H, hd, rope_cols;   // ROPE: columns [0, rope_cols) are rotated (q and k heads)
  int gu_blk;             // GEGLU
  int ld_out;             // leading dimension (elements) of the output
  const int* m_active;    // device pointer to the active row count of this iteration (or null)
  // EPI_FINAL
  float* x;               // [M, A] current actions (internal robot order)
  const CallPtrs* cp;     // velocity export pointer + caller batch
  const float* dt;        // Tables::dt
  const int* src;         // Tables::src
  int A, k_iter;
  int force_bn;           // BIAS_F32 / RESID: N tile to use (0 = chosen from N and M)
  const float* gate;      // RESID, adaptive-norm variant: h += gate[row / H][col] * acc (null = 1); rows gate_ld floats apart
  int gate_ld;
  int force_pair;         // rosa_debug_gemm only: 0 = kernel chosen by M (the path), 1 = single-CTA kernel, 2 = CTA-pair kernel
};

// ---- launchers (each checks nothing; callers validated shapes) -------------------------
// simple CUDA-core family
void launch_gemm_naive(const op16* A, const op16* W, float* C, int M, int N, int K, int fp16,
                       const int* m_active, cudaStream_t s);
void launch_epilogue(Epi epi, const float* C, int M, int N, const EpiArgs& a, cudaStream_t s);
void launch_attn_simple(const Dims& dm, const Tables& tb, int layer, const bf16* qkv, op16* o,
                        int k_iter, int max_len, cudaStream_t s);
// common elementwise kernels
void launch_gather_x(float* x, const CallPtrs* cp, const Tables& tb, int HA, cudaStream_t s);
void launch_scatter_x(const CallPtrs* cp, const float* x, const Tables& tb, int HA, cudaStream_t s);
void launch_timevec(float* tvec, const bf16* w_t1, const float* b_t1, const Dims& dm,
                    const Tables& tb, int nsteps_max, cudaStream_t s);
void launch_tau16(op16* a16, const Dims& dm, const Tables& tb, int nsteps_max, cudaStream_t s);
// adaptive-norm variant (reading R25)
void launch_swish16(op16* out, const float* in, size_t n, int fp16, cudaStream_t s);
void launch_embed_lin(float* h, const float* x, const float* w_inT, const float* b_in, const Dims& dm, const Tables& tb,
                      int k_iter, int M, cudaStream_t s);
void launch_adarms(op16* out, const float* h, const float* mod, int mod_ld, const Dims& dm, const Tables& tb, int k_iter,
                   int M, cudaStream_t s);
void launch_embed1(op16* z, const float* x, const float* wca, const float* bca, const float* tvec_k,
                   const Dims& dm, const Tables& tb, int k_iter, int M, cudaStream_t s);
void launch_rmsnorm(op16* out, const float* h, const Dims& dm, const Tables& tb, int k_iter, int M,
                    cudaStream_t s);
void launch_final(float* x, const CallPtrs* cp, const float* h, const float* g, const bf16* w_out,
                  const float* b_out, const Dims& dm, const Tables& tb, int k_iter, int M,
                  cudaStream_t s);
void launch_f32_to_bf16(bf16* dst, const float* src, size_t n, cudaStream_t s);
// tcgen05 family (gemm_tcgen05.cu)
bool tc_gemm_supported(int N, int K);
int tc_resid_bn(int N, int M);  // N tile of the BIAS_F32 / RESID launches
int tc_ssq_parts(int N);       // sum-of-squares partials per row written by the BIAS_F32 / RESID launches (one per 32 columns)
// A [M,K] row-major, W [N,K] row-major, both fp16 or both bf16 (EpiArgs::in_fp16)
cudaError_t launch_gemm_tc(Epi epi, const op16* A, const op16* W, int M, int N, int K,
                           const EpiArgs& a, cudaStream_t s);

bool tc_use_pair(int M);

// tcgen05 attention (attn_tcgen05.cu)
bool tc_attn_supported(const Dims& dm);
size_t tc_attn_map_bytes();  // sizeof(CUtensorMap)
bool tc_attn_make_prefix_maps(void* out2_host, const bf16* k, const bf16* v, int len, const Dims& dm);
size_t tc_attn_part_bytes(int n_cta);  // scratch for the partial results of items cut between CTAs
int tc_attn_tiles(const Dims& dm);     // token tiles (items) per robot
int attn_build_list(const Dims& dm, int n_active, const int* len, int n_cta, std::vector<AttnSeg>& segs, int* offs);
cudaError_t launch_attn_tc(const Dims& dm, const Tables& tb, int layer, const bf16* qkv, op16* o, int k_iter,
                           int M, const void* d_kv_maps, void* part, int* part_flag, int n_cta, cudaStream_t s);

void set_error(const std::string& msg);

// Kernel launch with the programmatic-stream-serialization attribute (PDL; ROSA_PDL=0 turns it off).
// Only for kernels that call pdl_wait() before touching global data produced or consumed by earlier kernels.
bool pdl_enabled();
template <typename... KArgs, typename... Args>
inline cudaError_t launch_k(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl_enabled() ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

}  // namespace rosa
