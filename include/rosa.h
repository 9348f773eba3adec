/* rosa.h — C ABI of librosa: inter-robot batched action-model inference on one B200.
 *
 * What the calls mean (citations: PAPER.md = /root/reference/PAPER.md, the ROSA paper;
 * BJ = BASELINE.json north_star / configs; R# = readings listed in DESIGN.md):
 *
 *   The paper's GPU worker hosts ONE model and serves a batch of per-robot inference
 *   requests with a scheduler-chosen discrete batch size ("each GPU worker
 *   [is dedicated] to a single model", :352 server configuration = (model, batch size,
 *   #robots), :527 "System 1 action models use a discrete batch size").  The System-1
 *   output is an action chunk.  The model itself is a black box in the paper
 *   (PAPER.md:346-348); here it is the pi0-style flow-matching action expert of BJ:
 *   N Euler steps x <- x + dt*v(x,t); v is a pre-norm GQA transformer over each robot's H
 *   action tokens that attend to that robot's cached VLM-prefix K/V (ragged lengths) and to
 *   the block's own action tokens (DESIGN.md section 1 gives the full algorithm).
 *
 * All entry points return rosa_status_t (except rosa_last_error / rosa_version); nothing is
 * thrown across the ABI.  Arguments are validated before any launch.  There is no CPU
 * fallback: without a CUDA device every compute entry point returns ROSA_ERR_CUDA.
 * Pointers are marked [host] or [dev].  The library is not thread-safe per expert handle.
 * Measurement and unit-test hooks (per-class timing, the GEMM unit test, host-side planners) are declared in
 * rosa_debug.h; they are exported by the same library and are not needed to use it.
 */
#ifndef ROSA_H_
#define ROSA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rosa_expert rosa_expert_t; /* opaque: owns device weights, workspaces, CUDA graphs */

typedef enum {
  ROSA_OK = 0,
  ROSA_ERR_INVALID_ARG = -1,   /* NULL pointer, out-of-range size, duplicate robot id, n_steps < 1 ... */
  ROSA_ERR_UNBOUND_ROBOT = -2, /* a robot id in the batch has no prefix K/V bound */
  ROSA_ERR_CAPACITY = -3,      /* batch > max_batch, robot >= max_robots, len > max_prefix_len */
  ROSA_ERR_CUDA = -4,          /* CUDA runtime/driver error (message in rosa_last_error) */
  ROSA_ERR_UNSUPPORTED = -5    /* shape the kernels do not cover (see rosa_expert_create) */
} rosa_status_t;

typedef enum { ROSA_F32 = 0, ROSA_BF16 = 1 } rosa_dtype_t;

/* Model + capacity description (BJ configs 0/1; R3 time-embedding periods, R5 eps, R7 rope base). */
typedef struct {
  int32_t layers, d_model, n_q_heads, n_kv_heads, head_dim, ffn, horizon, action_dim;
  int32_t max_robots;     /* robot ids are 0 .. max_robots-1 */
  int32_t max_batch;      /* largest batch one rosa_denoise_batch call may carry */
  int32_t max_prefix_len; /* largest prefix length L_i that may be bound */
  int32_t max_steps;      /* largest n_steps[i] per call */
  float rope_base;        /* 10000 */
  float rms_eps;          /* 1e-6 */
  float time_min_period;  /* 4e-3 */
  float time_max_period;  /* 4.0  */
  int32_t time_conditioning; /* 0: time concatenated into the embedding MLP (pi0-style, BJ cfg0; the path of
                              * every BASELINE.json config).  1: adaptive RMSNorm (pi0.5-style, PAPER.md:438,
                              * DESIGN.md reading R25): cond = swish(W_t2 swish(W_t1 tau(t) + b_t1) + b_t2),
                              * h0 = W_in x + b_in, every norm y = h rsqrt(mean h^2 + eps)(1 + scale) + shift
                              * with (scale, shift, gate) = W_mod cond + b_mod, h += gate * sublayer(y).
                              * Needs the tcgen05 shapes (head_dim 256), else ROSA_ERR_UNSUPPORTED. */
} rosa_expert_config_t;

/* Weights.  Every matrix is [out_features, in_features] row-major (R10); q/k/v rows are
 * head-major ([head, head_dim]).  dtype applies to all tensors; on_device says whether the
 * pointers are device (1) or host (0) pointers.  Per-layer members are [host] arrays of
 * `layers` pointers.  Shapes: w_in [d,A] b_in [d]; w_t1 [d,2d] (columns 0..d-1 multiply the
 * sinusoidal time embedding, d..2d-1 the projected action, R2) b_t1 [d]; w_t2 [d,d] b_t2 [d];
 * w_out [A,d] b_out [A]; g_final [d]; per layer g_attn [d], wq [nq*hd,d], wk [nkv*hd,d],
 * wv [nkv*hd,d], wo [d,nq*hd], g_mlp [d], w_gate [F,d], w_up [F,d], w_down [d,F].
 * time_conditioning == 1 only (ignored otherwise): w_t1 is [d,d]; w_mod_* [3d,d] and b_mod_* [3d], rows
 * ordered scale | shift | gate, one pair per norm (per layer: attention, MLP; and the final norm);
 * g_attn, g_mlp, g_final are not read.
 * Loading a trained checkpoint: the conventions here are the ones of DESIGN.md section 2, not of any particular
 * code base - w_t1's columns are [time | action] (a model that concatenates [action | time] needs its two column
 * blocks swapped), and the RMSNorm gain multiplies as g (a "1 + g" parameterisation needs 1 added to the stored
 * gains). */
typedef struct {
  rosa_dtype_t dtype;
  int32_t on_device;
  const void *w_in, *b_in, *w_t1, *b_t1, *w_t2, *b_t2, *w_out, *b_out, *g_final;
  const void *const *g_attn, *const *wq, *const *wk, *const *wv, *const *wo;
  const void *const *g_mlp, *const *w_gate, *const *w_up, *const *w_down;
  const void *const *w_mod_attn, *const *b_mod_attn, *const *w_mod_mlp, *const *b_mod_mlp;
  const void *w_mod_final, *b_mod_final;
} rosa_weights_t;

/* Create an expert on the current CUDA device (every later call on this expert must be made with that device
 * current, else ROSA_ERR_INVALID_ARG).  Copies and repacks every weight into library-owned 16-bit device storage
 * (the caller may free its copies on return).
 * Operand format (R19', R26): the weight GEMMs run on fp16 operands with fp32 accumulation by default
 * (bf16-valued weights convert exactly above 6.1e-5; smaller ones become fp16 subnormals with <= 3e-8 absolute error);
 * the residual stream is fp32, and its 16-bit operand copy SATURATES at +-65504: a model whose un-normalised residual
 * leaves the fp16 range is clipped there (finite, never inf / NaN).  The environment variable ROSA_GEMM_DTYPE=bf16
 * (read here) selects bf16 operands instead: the range of fp32, at about five times the operand rounding error.
 * q, k, v, the softmax numerators and the prefix cache are bf16 in either mode.
 * Constraints (else ROSA_ERR_UNSUPPORTED): d_model, ffn, n_q_heads*head_dim multiples of 64;
 * head_dim even, <= 256; n_q_heads % n_kv_heads == 0; action_dim <= 64; horizon <= 64.
 * The environment variable ROSA_KERNELS=simple forces the shape-generic CUDA-core kernels
 * (debugging aid); by default the tcgen05 kernels run whenever the shape qualifies. */
rosa_status_t rosa_expert_create(const rosa_expert_config_t *cfg, const rosa_weights_t *w,
                                 rosa_expert_t **out);
rosa_status_t rosa_expert_destroy(rosa_expert_t *e);

/* Bind robot's per-layer prefix K/V cache (the VLM prefill output; BJ cfg1:
 * "[L,1,256] bf16, K pre-rotated").  k_layers/v_layers: [host] arrays of `layers` [dev]
 * pointers, each [len, n_kv_heads, head_dim] contiguous, 16-byte aligned.
 * dtype ROSA_BF16: the pointers are BORROWED (kept alive by the caller until unbind/re-bind/
 * destroy); a packed ragged buffer is bound by passing base + cu_seqlens[i]*n_kv*hd (BJ cfg2).
 * dtype ROSA_F32: values are converted, synchronously, into library-owned bf16 storage (kept until destroy).
 * len == 0 is legal (self-attention only, R8).  Re-binding replaces the entry.
 * Ordering: bind returns without waiting for the device.  The robot's table entries (pointers, length, tensor maps)
 * are updated by copies on a library stream that runs AFTER every rosa_denoise_batch* call enqueued before the
 * bind, and the next rosa_denoise_batch* call waits for them on its own stream: calls enqueued before a bind see
 * the old binding, calls made after it the new one.  The DATA behind borrowed pointers is the caller's: it must be
 * complete, in stream order, before the first call that uses it, and must stay untouched until the last call that
 * was enqueued with that binding has finished.  unbind only marks the robot unbound on the host. */
rosa_status_t rosa_prefix_kv_bind(rosa_expert_t *e, int32_t robot, const void *const *k_layers,
                                  const void *const *v_layers, int32_t len, rosa_dtype_t dtype);
rosa_status_t rosa_prefix_kv_unbind(rosa_expert_t *e, int32_t robot);

/* The step before the loop (the VLM backbone processes the observation before the action head runs;
 * SURVEY.md 8(f) item 4; reading R29): produce one robot's prefix K/V cache from the backbone's NORMALISED
 * hidden states of its `len` prefix tokens, per layer l:
 *     K_l = RoPE(n_l W_pk,l^T, positions 0..len-1)   ("K pre-rotated", BJ cfg1; R7),     V_l = n_l W_pv,l^T
 * hidden_layers / wk_layers / wv_layers / k_out_layers / v_out_layers: [host] arrays of `layers` [dev] pointers,
 * 16-byte aligned, all bf16: hidden [len, d_prefix], wk / wv [n_kv_heads*head_dim, d_prefix] row-major, outputs
 * [len, n_kv_heads, head_dim] contiguous - exactly what rosa_prefix_kv_bind(..., ROSA_BF16) borrows.  Nothing is
 * bound: bind the outputs afterwards (in stream order before the first call that uses them).  The backbone that
 * produces the hidden states is outside this library.  Asynchronous on `stream`; needs the tcgen05 kernels
 * (head_dim 256) and d_prefix % 64 == 0, else ROSA_ERR_UNSUPPORTED; len <= max_prefix_len, else ROSA_ERR_CAPACITY. */
rosa_status_t rosa_prefix_kv_produce(rosa_expert_t *e, int32_t d_prefix, const void *const *hidden_layers,
                                     const void *const *wk_layers, const void *const *wv_layers, int32_t len,
                                     void *const *k_out_layers, void *const *v_out_layers, void *stream);

/* One batched denoise call (BJ north_star (1); PAPER.md:293/:527 discrete batch).
 * Robot i is integrated from t_start[i] (NULL = 1.0 for all) to 0 in n_steps[i] uniform Euler
 * steps, dt_i = -t_start[i]/n_steps[i] (R1).  The call runs max_i n_steps[i] iterations;
 * robot i is active in iteration k iff k < n_steps[i]; afterwards its x is untouched (R16).
 *   robot_ids   [host] int32 [batch], distinct, each bound
 *   noise       [dev]  float32 [batch, H, A]  (x at t_start)
 *   out_actions [dev]  float32 [batch, H, A]  (may alias noise)
 *   stream      cudaStream_t (NULL = legacy default stream)
 * Asynchronous on `stream`; the [host] arrays are consumed before return. */
rosa_status_t rosa_denoise_batch(rosa_expert_t *e, int32_t batch, const int32_t *robot_ids,
                                 const float *noise, const float *t_start, const int32_t *n_steps,
                                 float *out_actions, void *stream);

/* Same with an explicit per-robot dt (continuous-batching use, BJ cfg3 / R15: a caller may
 * advance a robot part of the way, t_end = t_start + n*dt) and an optional export of the
 * per-step velocities: out_velocity [dev] float32 [max_i n_steps, batch, H, A] or NULL;
 * rows of robots inactive in iteration k are written as 0. */
rosa_status_t rosa_denoise_batch_ex(rosa_expert_t *e, int32_t batch, const int32_t *robot_ids,
                                    const float *noise, const float *t_start, const float *dt,
                                    const int32_t *n_steps, float *out_actions,
                                    float *out_velocity, void *stream);

/* End-to-end convenience: noise and out_actions are [host] float32 buffers; the call copies
 * noise host->device, runs rosa_denoise_batch_ex, copies the actions back and synchronises
 * `stream` before returning (the robot-facing request/response of PAPER.md:58). */
rosa_status_t rosa_denoise_batch_host(rosa_expert_t *e, int32_t batch, const int32_t *robot_ids,
                                      const float *noise_host, const float *t_start,
                                      const float *dt, const int32_t *n_steps,
                                      float *out_actions_host, void *stream);

/* Allocation-free linear layer, for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid it).  One GEMM of the path's kind with its fp32 epilogue,
 *     acc[M,N] = A[M,K] * W[N,K]^T      A, W: 16-bit [dev] operands, row-major, bf16 (fp16 = 0) or fp16 (fp16 = 1)
 *     epi = 0: C = acc      epi = 2: C = acc + bias[n] (bias [dev] float32 [N])      epi = 4: C = C + acc
 * with C [dev] float32 [M,N], through the shape-generic CUDA-core kernels (any M, N, K >= 1; not a speed path).
 * The fp32 product passes through a scratch matrix that is a file-scope device array of the library
 * (ROSA_NOALLOC_MAX_ELEMS floats = 4 MiB, held by every GPU that loads the library until exit): the call makes no
 * cudaMalloc / cudaFree and calls no allocating routine; M * N beyond the limit returns ROSA_ERR_CAPACITY.
 * Asynchronous on `stream`.  All calls share the scratch: calls that may overlap on the GPU (different streams
 * with no ordering between them) race on it - serialise them.  Needs no expert. */
#define ROSA_NOALLOC_MAX_ELEMS (1 << 20)
rosa_status_t rosa_linear_noalloc(int32_t epi, int32_t fp16, int32_t M, int32_t N, int32_t K, const void *A,
                                  const void *W, const float *bias, float *C, void *stream);

const char *rosa_last_error(void); /* thread-local, never NULL */
int32_t rosa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ROSA_H_ */
