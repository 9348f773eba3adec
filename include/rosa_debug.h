/* rosa_debug.h — measurement and unit-test hooks of librosa.  Not needed to USE the library (rosa.h is the
 * boundary); bench.py and the tests call these through the same ctypes binding.
 * Citations as in rosa.h. */
#ifndef ROSA_DEBUG_H_
#define ROSA_DEBUG_H_

#include "rosa.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernel launches (graph nodes) the last denoise call issued, and which kernel family runs
 * (0 = shape-generic CUDA-core kernels, 1 = tcgen05). */
rosa_status_t rosa_last_launch_count(rosa_expert_t *e, int64_t *n_kernels);
rosa_status_t rosa_kernel_family(rosa_expert_t *e, int32_t *family);
/* CUDA graphs captured so far by this expert.  A call replays the graph of its batch BUCKET (next power of two,
 * at most max_batch) and its largest n_steps; a capture happens only the first time a (bucket, n) pair is seen. */
rosa_status_t rosa_debug_graph_captures(rosa_expert_t *e, int64_t *n_captures);

/* Kernel classes of the hot path, for rosa_profile_batch. */
typedef enum {
  ROSA_KC_GATHER_SCATTER = 0, /* x gather at call start / scatter at call end */
  ROSA_KC_TIMEVEC = 1,        /* a1, time half of W_1 (hoisted, once per call) */
  ROSA_KC_INPROJ = 2,         /* a1, W_in x + b_in */
  ROSA_KC_GEMM_EMBED = 3,     /* a1, the two d x d GEMMs of the time MLP */
  ROSA_KC_RMSNORM = 4,        /* a2 */
  ROSA_KC_GEMM_QKV = 5,       /* a3 + a4 */
  ROSA_KC_ATTN = 6,           /* a5 */
  ROSA_KC_GEMM_O = 7,         /* a6 */
  ROSA_KC_GEMM_GATEUP = 8,    /* a7 */
  ROSA_KC_GEMM_DOWN = 9,      /* a8 */
  ROSA_KC_FINAL = 10,         /* a9 + a10 */
  ROSA_KC_COUNT = 11
} rosa_kernel_class_t;

/* Measurement aid for bench.py (SURVEY 8(d) "evidence per kernel"): runs the same call as
 * rosa_denoise_batch_ex, NOT through the CUDA graph, with a CUDA event recorded on `stream`
 * between consecutive launches, synchronises, and returns per kernel class the summed device
 * time in milliseconds (ms_out [host] float[ROSA_KC_COUNT]) and the number of launches
 * (launches_out [host] int32[ROSA_KC_COUNT]).  Results are identical to the graphed call. */
rosa_status_t rosa_profile_batch(rosa_expert_t *e, int32_t batch, const int32_t *robot_ids,
                                 const float *noise, const float *t_start, const float *dt,
                                 const int32_t *n_steps, float *out_actions, void *stream,
                                 float *ms_out, int32_t *launches_out);
const char *rosa_kernel_class_name(int32_t cls); /* "" if out of range */

/* Kernel unit-test hook for the GEMMs with their fused residual / bias epilogues (steps a1, a6, a8).
 *   acc[M,N] = A[M,K] * W[N,K]^T       A, W: 16-bit [dev] operands, bf16 (fp16 = 0) or fp16 (fp16 = 1)
 *   epi = 0  C = acc                                       (C [dev] float32 [M,N])
 *   epi = 2  C = acc + bias[n]                             (bias [dev] float32 [N])
 *   epi = 4  C = C + acc                                   (C holds the residual on entry)
 * For epi 2 and 4, when h16 / ssq are not NULL the kernel also writes what the path's fused RMSNorm needs:
 * h16 [dev] [M,N] = the 16-bit copy of the new C, and ssq [dev] float32 [M, N/32] = the sum of squares of each
 * 32-column group of the new C.  family 1 = tcgen05/TMA kernels (K % 64 == 0, N % 64 == 0), family 0 = the
 * CUDA-core GEMM (epi 0 only).  pair = 1 forces the CTA-pair kernel (256-row tiles), 0 the single-CTA kernel,
 * -1 the library's own choice; bn = N-tile width to force (pair: 64..256 in steps of 32; single: 64, 128, 256)
 * or 0 for the library's choice.  ROSA_ERR_UNSUPPORTED for a combination the kernels do not have. */
rosa_status_t rosa_debug_gemm(int32_t family, int32_t epi, int32_t pair, int32_t bn, int32_t fp16, int32_t M,
                              int32_t N, int32_t K, const void *A, const void *W, float *C, const float *bias,
                              void *h16, float *ssq, void *stream);

/* Host logic of the attention kernel's work split, testable without a device (no expert, no CUDA call).
 * The attention step (a5) of n_robots robots with prefix lengths len[] is cut into per-CTA runs of SEGMENTS
 * (robot, token tile, key blocks [kb0, kb1)); see attn_tcgen05.cu.  Writes offs_out[n_cta + 1] (segment index
 * ranges per CTA) and up to cap records of 8 int32 {robot, tile, kb0, kb1, n_part, part0, 0, 0} to segs_out;
 * returns the number of segments or a negative rosa_status_t (ROSA_ERR_CAPACITY if cap is too small). */
int32_t rosa_debug_attn_plan(int32_t horizon, int32_t n_robots, const int32_t *len, int32_t n_cta,
                             int32_t *offs_out, int32_t *segs_out, int32_t cap);

#ifdef __cplusplus
}
#endif
#endif /* ROSA_DEBUG_H_ */
