// C-ABI entry points of librosa (include/rosa.h) and the host runtime that sequences the hot
// path: per-call device tables, the N-step loop, CUDA-graph capture/replay.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <numeric>
#include <tuple>

#include <nvtx3/nvToolsExt.h>   // header-only NVTX: host ranges around a call, its capture and each Euler step

#include "rosa_internal.h"

namespace rosa {

static thread_local std::string g_err = "";
void set_error(const std::string& msg) { g_err = msg; }
bool pdl_enabled() {
  static int on = -1;
  if (on < 0) { const char* e = getenv("ROSA_PDL"); on = !(e && !strcmp(e, "0")); }
  return on != 0;
}

#define CK(call)                                                                      \
  do {                                                                                \
    cudaError_t _e = (call);                                                          \
    if (_e != cudaSuccess) {                                                          \
      set_error(std::string(#call) + ": " + cudaGetErrorString(_e));                  \
      return ROSA_ERR_CUDA;                                                           \
    }                                                                                 \
  } while (0)

static inline uint16_t f2bf(float f) {  // round-to-nearest-even, host side
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
static inline float bf2f(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}

constexpr int kStageRing = 4;
constexpr size_t kMaxGraphs = 48;   // (batch bucket, max n_steps) pairs kept instantiated per expert

struct GraphKey {
  int batch, nmax, vel;
  bool operator<(const GraphKey& o) const {
    return std::tie(batch, nmax, vel) < std::tie(o.batch, o.nmax, o.vel);
  }
};

}  // namespace rosa

using namespace rosa;

struct rosa_expert {
  rosa_expert_config_t cfg;
  Dims dm;
  int family = 0;     // 0 simple, 1 tcgen05
  bool use_graph = true;
  int max_pos = 0;
  // weights
  bf16 *w_t1 = nullptr, *w_out = nullptr;  // CUDA-core steps: bf16 as given
  float *wca = nullptr, *bca = nullptr;    // (W_1[:, d:] W_in)^T [A, d] and W_1[:, d:] b_in [d], folded in fp64
  op16* w_t2 = nullptr;                    // GEMM operand: fp16 or bf16 (dm.fp16)
  op16 *w_t1dup = nullptr, *tau16 = nullptr;
  // adaptive-norm variant (R25): all 2L+1 modulation matrices stacked [(2L+1) 3d, d] (norm n = 2l attention,
  // 2l+1 MLP, 2L final; rows scale | shift | gate), their biases, the 16-bit time-MLP activations and the
  // per-step modulation vectors [max_batch, (2L+1) 3d]
  op16 *w_mod = nullptr, *z16 = nullptr, *cond16 = nullptr;
  float *b_mod = nullptr, *mod = nullptr;  // tcgen05 family: [W_1[:, :d] | W_1[:, :d]] [d, 2d] and the [hi | lo] tau rows
  op16* w_out16 = nullptr;                 // [64, d]: W_out with the final-norm gain folded in, zero rows past A (tcgen05 family)
  float *b_t1 = nullptr, *b_t2 = nullptr, *b_out = nullptr, *g_final = nullptr;
  std::vector<LayerWeights> lw;
  float2* rope_tab = nullptr;
  // workspaces
  float *x = nullptr, *h = nullptr, *tvec = nullptr, *scratch = nullptr;
  // nrm: A operand of the QKV / gate-up GEMMs = normalised h (family 0) or the 16-bit copy of h
  // itself (family 1, norm scale applied in the consumer's epilogue from the ssq partials)
  op16 *zbuf = nullptr, *nrm = nullptr, *obuf = nullptr, *mact = nullptr;
  float* ssq = nullptr;  // [Mmax, n_part] partial sums of squares of h rows (family 1)
  bf16* qkv = nullptr;  // q/k/v feed attention together with the bf16 prefix cache: always bf16
  // robot table (device) + host mirror
  const bf16** d_rk = nullptr;
  const bf16** d_rv = nullptr;
  int* d_rlen = nullptr;
  int* d_zero = nullptr;           // two device zeros: the (ids, rlen) tables of rosa_prefix_kv_produce (positions = row index)
  std::vector<int> h_rlen;         // -1 = unbound
  std::vector<std::vector<bf16*>> owned;  // per robot: library-owned K/V buffers (fp32 binds), kept until destroy
  std::vector<size_t> owned_cap;          // elements each of them holds
  // bind is asynchronous: table updates go from a pinned per-robot record through bind_stream (ordered after the last
  // denoise call that was enqueued); the next denoise call waits for bind_ev on its stream
  cudaStream_t bind_stream = nullptr;
  cudaEvent_t bind_ev = nullptr, call_ev = nullptr;
  char* h_bind = nullptr;                 // [max_robots][bind_rec]
  size_t bind_rec = 0;
  std::vector<char> bind_pending;         // robot's record is (possibly) still being copied
  bool bind_dirty = false, call_pending = false;
  int max_len_bound = 0;
  bool attn_tc = false;            // tcgen05 attention kernel in use
  char* d_kv_maps = nullptr;       // [max_robots * layers * 2] CUtensorMap (prefix K, V per robot/layer)
  // per-call tables
  char* d_call = nullptr;          // fixed device block
  char* h_stage[kStageRing] = {};  // pinned ring
  cudaEvent_t stage_ev[kStageRing] = {};
  int stage_next = 0;
  size_t call_bytes = 0;
  size_t off_ids, off_src, off_t0, off_dt, off_ns, off_mact, off_ptrs, off_aiter, off_aoffs, off_asegs;
  size_t seg_cap = 0;              // capacity of the attention segment table (entries)
  int n_cta = 0;                   // CTAs of the persistent attention kernel (= SMs of the device)
  void* attn_part = nullptr;       // per-CTA partial (O, m, l) of items cut between CTAs
  int* attn_flag = nullptr;        // [n_cta] ready flags of those partials
  int64_t graph_captures = 0;      // graphs captured so far (rosa_debug_graph_captures)
  std::map<GraphKey, cudaGraphExec_t> graphs;      // at most kMaxGraphs, least recently used evicted
  std::map<GraphKey, int64_t> graph_launches;
  std::map<GraphKey, int64_t> graph_used;          // value of graph_clock at the last launch
  int64_t graph_clock = 0;
  int device = 0;                                  // the CUDA device the expert lives on
  cudaStream_t cap_stream = nullptr;
  int64_t last_launches = 0;
  float* e2e_dev = nullptr;  // staging for rosa_denoise_batch_host
  // per-launch event timing (rosa_profile_batch): boundary event before every launch
  bool prof_on = false;
  std::vector<cudaEvent_t> prof_ev;
  std::vector<int> prof_cls;
  size_t prof_n = 0;
  std::vector<void*> allocs;
  std::vector<rosa::AttnSeg> seg_tmp;
};

namespace rosa {

static rosa_status_t dev_alloc(rosa_expert* e, void** p, size_t bytes) {
  CK(cudaMalloc(p, bytes ? bytes : 16));
  e->allocs.push_back(*p);
  return ROSA_OK;
}

// Bring a caller tensor to host float32 (weights are repacked on the host once, at create).
static rosa_status_t fetch_f32(const void* src, size_t n, rosa_dtype_t dt, int on_device,
                               std::vector<float>& out) {
  out.resize(n);
  const size_t esz = dt == ROSA_F32 ? 4 : 2;
  std::vector<char> raw;
  const void* hp = src;
  if (on_device) {
    raw.resize(n * esz);
    CK(cudaMemcpy(raw.data(), src, n * esz, cudaMemcpyDeviceToHost));
    hp = raw.data();
  }
  if (dt == ROSA_F32) {
    memcpy(out.data(), hp, n * 4);
  } else {
    const uint16_t* b = (const uint16_t*)hp;
    for (size_t i = 0; i < n; ++i) out[i] = bf2f(b[i]);
  }
  return ROSA_OK;
}
static rosa_status_t upload_bf16(rosa_expert* e, const std::vector<float>& v, bf16** out) {
  std::vector<uint16_t> b(v.size());
  for (size_t i = 0; i < v.size(); ++i) b[i] = f2bf(v[i]);
  rosa_status_t st = dev_alloc(e, (void**)out, b.size() * 2);
  if (st != ROSA_OK) return st;
  CK(cudaMemcpy(*out, b.data(), b.size() * 2, cudaMemcpyHostToDevice));
  return ROSA_OK;
}
// GEMM operand upload: fp16 (RNE from the given values; bf16-valued inputs with |w| >= 6.1e-5
// convert exactly) or bf16, per dm.fp16.
static rosa_status_t upload_op16(rosa_expert* e, const std::vector<float>& v, op16** out) {
  std::vector<uint16_t> b(v.size());
  if (e->dm.fp16) {
    for (size_t i = 0; i < v.size(); ++i) b[i] = __half_as_ushort(__float2half_rn(v[i]));
  } else {
    for (size_t i = 0; i < v.size(); ++i) b[i] = f2bf(v[i]);
  }
  rosa_status_t st = dev_alloc(e, (void**)out, b.size() * 2);
  if (st != ROSA_OK) return st;
  CK(cudaMemcpy(*out, b.data(), b.size() * 2, cudaMemcpyHostToDevice));
  return ROSA_OK;
}
static rosa_status_t upload_f32(rosa_expert* e, const std::vector<float>& v, float** out) {
  rosa_status_t st = dev_alloc(e, (void**)out, v.size() * 4);
  if (st != ROSA_OK) return st;
  CK(cudaMemcpy(*out, v.data(), v.size() * 4, cudaMemcpyHostToDevice));
  return ROSA_OK;
}

// Device tables of the current call (robots in internal order).
static Tables make_tables(const rosa_expert* e, int batch) {
  const int p0 = 0;
  Tables tb;
  tb.ids = (const int*)(e->d_call + e->off_ids) + p0;
  tb.src = (const int*)(e->d_call + e->off_src) + p0;
  tb.t0 = (const float*)(e->d_call + e->off_t0) + p0;
  tb.dt = (const float*)(e->d_call + e->off_dt) + p0;
  tb.nsteps = (const int*)(e->d_call + e->off_ns) + p0;
  tb.m_active = (const int*)(e->d_call + e->off_mact);
  tb.attn_iter = (const int*)(e->d_call + e->off_aiter);
  tb.attn_offs = (const int*)(e->d_call + e->off_aoffs);
  tb.attn_segs = (const AttnSeg*)(e->d_call + e->off_asegs);
  tb.batch_dev = &((const CallPtrs*)(e->d_call + e->off_ptrs))->batch_ext;
  tb.rk = e->d_rk;
  tb.rv = e->d_rv;
  tb.rlen = e->d_rlen;
  tb.batch = batch;
  return tb;
}

// Internal order of a call: n_steps descending (stable), so that the active set of iteration k is a row prefix.
static std::vector<int> call_order(int batch, const int32_t* n_steps) {
  std::vector<int> order(batch);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return n_steps[a] > n_steps[b]; });
  return order;
}

static void destroy_impl(rosa_expert* e) {
  if (!e) return;
  cudaDeviceSynchronize();
  for (auto& kv : e->graphs) cudaGraphExecDestroy(kv.second);
  for (void* p : e->allocs) cudaFree(p);
  for (auto& v : e->owned)
    for (bf16* p : v) cudaFree(p);
  for (int i = 0; i < kStageRing; ++i) {
    if (e->h_stage[i]) cudaFreeHost(e->h_stage[i]);
    if (e->stage_ev[i]) cudaEventDestroy(e->stage_ev[i]);
  }
  if (e->cap_stream) cudaStreamDestroy(e->cap_stream);
  if (e->bind_stream) cudaStreamDestroy(e->bind_stream);
  if (e->bind_ev) cudaEventDestroy(e->bind_ev);
  if (e->call_ev) cudaEventDestroy(e->call_ev);
  if (e->h_bind) cudaFreeHost(e->h_bind);
  for (cudaEvent_t ev : e->prof_ev) cudaEventDestroy(ev);
  delete e;
}

static rosa_status_t create_impl(const rosa_expert_config_t* c, const rosa_weights_t* w, rosa_expert* e) {
  Dims& dm = e->dm;
  dm.layers = c->layers; dm.d = c->d_model; dm.nq = c->n_q_heads; dm.nkv = c->n_kv_heads;
  dm.hd = c->head_dim; dm.F = c->ffn; dm.H = c->horizon; dm.A = c->action_dim;
  dm.qkv_n = (dm.nq + 2 * dm.nkv) * dm.hd;
  dm.q_n = dm.nq * dm.hd;
  dm.gu_blk = 64;
  dm.ada = c->time_conditioning == 1;
  {  // GEMM operand format: fp16 by default (reading R19), ROSA_GEMM_DTYPE=bf16 to compare
    const char* gd = getenv("ROSA_GEMM_DTYPE");
    dm.fp16 = (gd && !strcmp(gd, "bf16")) ? 0 : 1;
  }
  dm.rope_base = c->rope_base; dm.eps = c->rms_eps; dm.pmin = c->time_min_period; dm.pmax = c->time_max_period;
  const int d = dm.d, F = dm.F, A = dm.A;
  const rosa_dtype_t dt = w->dtype;
  const int od = w->on_device;
  std::vector<float> t, u;
  rosa_status_t st;
#define FETCH(ptr, n) if ((st = fetch_f32(ptr, (size_t)(n), dt, od, t)) != ROSA_OK) return st
#define UPB(dst) if ((st = upload_bf16(e, t, &(dst))) != ROSA_OK) return st
#define UPO(dst) if ((st = upload_op16(e, t, &(dst))) != ROSA_OK) return st
#define UPF(dst) if ((st = upload_f32(e, t, &(dst))) != ROSA_OK) return st
  if (dm.ada) {  // R25: h0 = W_in x + b_in on CUDA cores (W_in^T as [A, d]); time MLP first layer [d, d], doubled along K
    std::vector<float> win, bin;
    if ((st = fetch_f32(w->w_in, (size_t)d * A, dt, od, win)) != ROSA_OK) return st;
    if ((st = fetch_f32(w->b_in, (size_t)d, dt, od, bin)) != ROSA_OK) return st;
    std::vector<float> wt((size_t)A * d);
    for (int n = 0; n < d; ++n)
      for (int c2 = 0; c2 < A; ++c2) wt[(size_t)c2 * d + n] = win[(size_t)n * A + c2];
    if ((st = upload_f32(e, wt, &e->wca)) != ROSA_OK) return st;
    if ((st = upload_f32(e, bin, &e->bca)) != ROSA_OK) return st;
    FETCH(w->w_t1, (size_t)d * d);
    std::vector<float> dup((size_t)d * 2 * d);
    for (int n = 0; n < d; ++n)
      for (int c2 = 0; c2 < d; ++c2) dup[(size_t)n * 2 * d + c2] = dup[(size_t)n * 2 * d + d + c2] = t[(size_t)n * d + c2];
    if ((st = upload_op16(e, dup, &e->w_t1dup)) != ROSA_OK) return st;
    // modulation matrices, stacked in norm order
    const size_t blk = (size_t)3 * d * d;
    std::vector<float> wm((size_t)(2 * dm.layers + 1) * blk), bm((size_t)(2 * dm.layers + 1) * 3 * d);
    for (int nrm = 0; nrm <= 2 * dm.layers; ++nrm) {
      const void* wp = nrm == 2 * dm.layers ? w->w_mod_final : (nrm & 1 ? w->w_mod_mlp[nrm / 2] : w->w_mod_attn[nrm / 2]);
      const void* bp = nrm == 2 * dm.layers ? w->b_mod_final : (nrm & 1 ? w->b_mod_mlp[nrm / 2] : w->b_mod_attn[nrm / 2]);
      if (!wp || !bp) { set_error("NULL modulation weight pointer"); return ROSA_ERR_INVALID_ARG; }
      FETCH(wp, blk); memcpy(&wm[nrm * blk], t.data(), blk * 4);
      FETCH(bp, (size_t)3 * d); memcpy(&bm[(size_t)nrm * 3 * d], t.data(), (size_t)3 * d * 4);
    }
    if ((st = upload_op16(e, wm, &e->w_mod)) != ROSA_OK) return st;
    if ((st = upload_f32(e, bm, &e->b_mod)) != ROSA_OK) return st;
  } else {  // a1 folding (exact algebra, fp64): Wca = W_1[:, d:] W_in, bca = W_1[:, d:] b_in
    std::vector<float> win, bin;
    if ((st = fetch_f32(w->w_in, (size_t)d * A, dt, od, win)) != ROSA_OK) return st;
    if ((st = fetch_f32(w->b_in, (size_t)d, dt, od, bin)) != ROSA_OK) return st;
    FETCH(w->w_t1, (size_t)d * 2 * d); UPB(e->w_t1);
    if (e->family == 1) {  // time half twice along K: pairs with the [hi(tau) | lo(tau)] operand rows of k_tau16
      std::vector<float> dup((size_t)d * 2 * d);
      for (int n = 0; n < d; ++n)
        for (int c = 0; c < d; ++c) dup[(size_t)n * 2 * d + c] = dup[(size_t)n * 2 * d + d + c] = t[(size_t)n * 2 * d + c];
      if ((st = upload_op16(e, dup, &e->w_t1dup)) != ROSA_OK) return st;
    }
    std::vector<float> wca((size_t)d * A), bca(d);
    std::vector<double> accr(A);
    for (int n = 0; n < d; ++n) {
      const float* w1a = &t[(size_t)n * 2 * d + d];
      std::fill(accr.begin(), accr.end(), 0.0);
      double accb = 0.0;
      for (int j = 0; j < d; ++j) {
        const double wj = w1a[j];
        const float* wi = &win[(size_t)j * A];
        for (int c = 0; c < A; ++c) accr[c] += wj * wi[c];
        accb += wj * bin[j];
      }
      for (int c = 0; c < A; ++c) wca[(size_t)c * d + n] = (float)accr[c];  // stored [A, d]: coalesced over n
      bca[n] = (float)accb;
    }
    if ((st = upload_f32(e, wca, &e->wca)) != ROSA_OK) return st;
    if ((st = upload_f32(e, bca, &e->bca)) != ROSA_OK) return st;
  }
  FETCH(w->b_t1, d); UPF(e->b_t1);
  FETCH(w->w_t2, (size_t)d * d); UPO(e->w_t2);
  FETCH(w->b_t2, d); UPF(e->b_t2);
  FETCH(w->w_out, (size_t)A * d); UPB(e->w_out);
  {  // a9 on the tensor cores (family 1): [64, d] operand, gain folded (R23), rows >= A zero
    std::vector<float> gf(d, 1.f), wo = t;
    if (!dm.ada && (st = fetch_f32(w->g_final, (size_t)d, dt, od, gf)) != ROSA_OK) return st;
    t.assign((size_t)64 * d, 0.f);
    for (int a = 0; a < A; ++a)
      for (int c = 0; c < d; ++c) t[(size_t)a * d + c] = wo[(size_t)a * d + c] * gf[c];
    UPO(e->w_out16);
  }
  FETCH(w->b_out, A); UPF(e->b_out);
  if (!dm.ada) { FETCH(w->g_final, d); UPF(e->g_final); }
  e->lw.resize(dm.layers);
  for (int l = 0; l < dm.layers; ++l) {
    LayerWeights& L = e->lw[l];
    // RMSNorm gains are folded into the columns of the consuming matrices: (h r g) W^T = r h (W g)^T
    std::vector<float> g1(d, 1.f), g2(d, 1.f);  // the adaptive norms (R25) have no learned gain
    if (!dm.ada && (st = fetch_f32(w->g_attn[l], (size_t)d, dt, od, g1)) != ROSA_OK) return st;
    if (!dm.ada && (st = fetch_f32(w->g_mlp[l], (size_t)d, dt, od, g2)) != ROSA_OK) return st;
    // packed [wq ; wk ; wv]  -> one QKV GEMM (step a3)
    std::vector<float> pk((size_t)dm.qkv_n * d);
    FETCH(w->wq[l], (size_t)dm.q_n * d); memcpy(pk.data(), t.data(), t.size() * 4);
    FETCH(w->wk[l], (size_t)dm.nkv * dm.hd * d); memcpy(pk.data() + (size_t)dm.q_n * d, t.data(), t.size() * 4);
    FETCH(w->wv[l], (size_t)dm.nkv * dm.hd * d);
    memcpy(pk.data() + (size_t)(dm.q_n + dm.nkv * dm.hd) * d, t.data(), t.size() * 4);
    for (size_t n = 0; n < (size_t)dm.qkv_n; ++n)
      for (int c = 0; c < d; ++c) pk[n * d + c] *= g1[c];
    t.swap(pk); UPO(L.wqkv);
    FETCH(w->wo[l], (size_t)d * dm.q_n); UPO(L.wo);
    // gate/up interleaved in blocks of gu_blk rows -> one GEMM + GeGLU epilogue (step a7)
    std::vector<float> gu((size_t)2 * F * d);
    const int g = dm.gu_blk;
    FETCH(w->w_gate[l], (size_t)F * d);
    for (int f = 0; f < F; ++f)
      memcpy(&gu[((size_t)(f / g) * 2 * g + f % g) * d], &t[(size_t)f * d], (size_t)d * 4);
    FETCH(w->w_up[l], (size_t)F * d);
    for (int f = 0; f < F; ++f)
      memcpy(&gu[((size_t)(f / g) * 2 * g + g + f % g) * d], &t[(size_t)f * d], (size_t)d * 4);
    for (size_t n = 0; n < (size_t)2 * F; ++n)
      for (int c = 0; c < d; ++c) gu[n * d + c] *= g2[c];
    t.swap(gu); UPO(L.wgu);
    FETCH(w->w_down[l], (size_t)d * F); UPO(L.wdown);
  }
#undef FETCH
#undef UPB
#undef UPO
#undef UPF
  // RoPE table in fp64 (R7): pos in [0, max_prefix_len + H), c < hd/2 -> (cos, sin)(pos * base^(-2c/hd))
  e->max_pos = c->max_prefix_len + dm.H;
  {
    const int half = dm.hd / 2;
    std::vector<float2> tab((size_t)e->max_pos * half);
    for (int cidx = 0; cidx < half; ++cidx) {
      const double theta = std::pow((double)dm.rope_base, -2.0 * cidx / dm.hd);
      for (int pos = 0; pos < e->max_pos; ++pos) {
        const double phi = pos * theta;
        tab[(size_t)pos * half + cidx] = make_float2((float)std::cos(phi), (float)std::sin(phi));
      }
    }
    if ((st = dev_alloc(e, (void**)&e->rope_tab, tab.size() * sizeof(float2))) != ROSA_OK) return st;
    CK(cudaMemcpy(e->rope_tab, tab.data(), tab.size() * sizeof(float2), cudaMemcpyHostToDevice));
  }
  // workspaces (rows padded to a multiple of 128 for the tile kernels)
  // + 256: lane 1 of a split batch starts on the next 256-row boundary after lane 0's rows
  const size_t Mmax = ((size_t)c->max_batch * dm.H + 127) / 128 * 128 + 256;
  const size_t HA = (size_t)dm.H * A;
#define WS(ptr, bytes) if ((st = dev_alloc(e, (void**)&(ptr), (bytes))) != ROSA_OK) return st
  WS(e->x, (size_t)c->max_batch * HA * 4);
  WS(e->h, Mmax * d * 4);
  WS(e->tvec, (size_t)c->max_steps * c->max_batch * d * 4);
  WS(e->zbuf, Mmax * d * 2);
  if (dm.ada) {
    const size_t rows = ((size_t)c->max_steps * c->max_batch + 127) / 128 * 128;
    WS(e->z16, rows * d * 2);
    WS(e->cond16, rows * d * 2);
    WS(e->mod, (size_t)c->max_batch * (2 * dm.layers + 1) * 3 * d * 4);
  }
  if (e->family == 1) WS(e->tau16, ((size_t)c->max_steps * c->max_batch + 127) / 128 * 128 * 2 * d * 2);
  WS(e->nrm, Mmax * d * 2);
  WS(e->qkv, Mmax * dm.qkv_n * 2);
  WS(e->obuf, Mmax * dm.q_n * 2);
  WS(e->mact, Mmax * F * 2);
  if (e->family == 0) WS(e->scratch, Mmax * (size_t)std::max(2 * F, dm.qkv_n) * 4);  // fp32 GEMM output of the CUDA-core family
  WS(e->e2e_dev, (size_t)c->max_batch * HA * 4);
  WS(e->ssq, Mmax * (d / 32) * 4);
  CK(cudaMemset(e->zbuf, 0, Mmax * d * 2));
  CK(cudaMemset(e->nrm, 0, Mmax * d * 2));
  CK(cudaMemset(e->qkv, 0, Mmax * dm.qkv_n * 2));
  CK(cudaMemset(e->obuf, 0, Mmax * dm.q_n * 2));
  CK(cudaMemset(e->mact, 0, Mmax * F * 2));
  // robot table
  WS(e->d_rk, (size_t)c->max_robots * dm.layers * sizeof(void*));
  WS(e->d_rv, (size_t)c->max_robots * dm.layers * sizeof(void*));
  WS(e->d_rlen, (size_t)c->max_robots * 4);
  CK(cudaMemset(e->d_rk, 0, (size_t)c->max_robots * dm.layers * sizeof(void*)));
  CK(cudaMemset(e->d_rv, 0, (size_t)c->max_robots * dm.layers * sizeof(void*)));
  CK(cudaMemset(e->d_rlen, 0, (size_t)c->max_robots * 4));
  WS(e->d_zero, 16);
  CK(cudaMemset(e->d_zero, 0, 16));
  {
    const char* at = getenv("ROSA_ATTN");
    e->attn_tc = e->family == 1 && tc_attn_supported(dm) && !(at && !strcmp(at, "simple"));
    if (e->attn_tc) {
      const size_t nb = (size_t)c->max_robots * dm.layers * 2 * tc_attn_map_bytes();
      WS(e->d_kv_maps, nb);
      CK(cudaMemset(e->d_kv_maps, 0, nb));
      int sms = 1, dev = 0;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
      WS(e->attn_part, tc_attn_part_bytes(sms));
      WS(e->attn_flag, (size_t)sms * 8 * 4);
      CK(cudaMemset(e->attn_flag, 0, (size_t)sms * 8 * 4));
    }
  }
  if (dm.ada && !e->attn_tc) {
    set_error("time_conditioning = 1 needs the tcgen05 attention kernel (8 query heads, 1 KV head, head_dim 256; ROSA_ATTN unset)");
    return ROSA_ERR_UNSUPPORTED;
  }
  e->h_rlen.assign(c->max_robots, -1);
  e->owned.resize(c->max_robots);
  // per-call table block
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 15) / 16 * 16; return o; };
  e->off_ids = take((size_t)c->max_batch * 4);
  e->off_src = take((size_t)c->max_batch * 4);
  e->off_t0 = take((size_t)c->max_batch * 4);
  e->off_dt = take((size_t)c->max_batch * 4);
  e->off_ns = take((size_t)c->max_batch * 4);
  e->off_mact = take((size_t)c->max_steps * 4);
  e->off_ptrs = take(sizeof(CallPtrs));
  // attention work lists: one list per distinct active-robot count of the call, the used part is copied per call
  e->n_cta = 1;
  {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&e->n_cta, cudaDevAttrMultiProcessorCount, dev);
  }
  e->off_aiter = take((size_t)c->max_steps * 4);
  e->off_aoffs = take((size_t)c->max_steps * (e->n_cta + 1) * 4);
  e->seg_cap = (size_t)c->max_steps * ((size_t)c->max_batch * tc_attn_tiles(dm) + 4 * e->n_cta);
  e->off_asegs = take(e->seg_cap * sizeof(AttnSeg));
  e->call_bytes = off;
  WS(e->d_call, e->call_bytes);
#undef WS
  for (int i = 0; i < kStageRing; ++i) {
    CK(cudaMallocHost((void**)&e->h_stage[i], e->call_bytes));
    CK(cudaEventCreateWithFlags(&e->stage_ev[i], cudaEventDisableTiming));
  }
  CK(cudaStreamCreateWithFlags(&e->cap_stream, cudaStreamNonBlocking));
  CK(cudaStreamCreateWithFlags(&e->bind_stream, cudaStreamNonBlocking));
  CK(cudaEventCreateWithFlags(&e->bind_ev, cudaEventDisableTiming));
  CK(cudaEventCreateWithFlags(&e->call_ev, cudaEventDisableTiming));
  e->bind_rec = ((size_t)dm.layers * (2 * sizeof(void*) + 2 * tc_attn_map_bytes()) + 64 + 63) / 64 * 64;
  CK(cudaMallocHost((void**)&e->h_bind, e->bind_rec * c->max_robots));
  e->bind_pending.assign(c->max_robots, 0);
  e->owned_cap.assign(c->max_robots, 0);
  return ROSA_OK;
}

// Profiling mark: when rosa_profile_batch is running, record a boundary event on `s` before the
// launch(es) of kernel class `cls`; the time between two consecutive marks is attributed to the
// earlier one.  A no-op otherwise (and never active during graph capture).
static void mark(rosa_expert* e, int cls, cudaStream_t s) {
  if (!e->prof_on) return;
  if (e->prof_n == e->prof_ev.size()) {
    cudaEvent_t ev;
    cudaEventCreate(&ev);
    e->prof_ev.push_back(ev);
    e->prof_cls.push_back(0);
  }
  cudaEventRecord(e->prof_ev[e->prof_n], s);
  e->prof_cls[e->prof_n] = cls;
  e->prof_n += 1;
}

// One GEMM + epilogue of the path, in whichever kernel family the expert runs.
static cudaError_t gemm(rosa_expert* e, int cls, Epi epi, const op16* A, const op16* W, int M, int N, int K,
                        const EpiArgs& a, cudaStream_t s) {
  mark(e, cls, s);
  if (e->family == 1 && tc_gemm_supported(N, K)) {
    e->last_launches += 1;
    return launch_gemm_tc(epi, A, W, M, N, K, a, s);
  }
  if (e->family != 0) return cudaErrorNotSupported;  // unreachable: create admits the tcgen05 family only for shapes its GEMMs cover
  launch_gemm_naive(A, W, e->scratch, M, N, K, a.in_fp16, a.m_active, s);
  launch_epilogue(epi, e->scratch, M, N, a, s);
  e->last_launches += 2;
  return cudaGetLastError();
}

// The call of the adaptive-norm variant (reading R25; tcgen05 family only).  Same GEMM, attention and
// final-projection kernels as the base path; the norms are k_adarms launches (normalised, modulated 16-bit
// operand; the GEMMs then run with a unit row scale) and the residual epilogues take the per-robot gate.
static cudaError_t enqueue_call_ada(rosa_expert* e, int batch, int nmax, cudaStream_t s) {
  const Dims& dm = e->dm;
  const Tables tb = make_tables(e, batch);
  const CallPtrs* cp = (const CallPtrs*)(e->d_call + e->off_ptrs);
  const int M = batch * dm.H, d = dm.d, R = nmax * batch;
  const int n_mod = (2 * dm.layers + 1) * 3 * d;
  cudaError_t err;
  e->last_launches = 0;
  mark(e, ROSA_KC_GATHER_SCATTER, s);
  launch_gather_x(e->x, cp, tb, dm.H * dm.A, s);
  e->last_launches += 1;
  // cond of every (step, robot) row: swish(W_t2 swish(W_t1 tau + b_t1) + b_t2), rows [k][batch]
  mark(e, ROSA_KC_TIMEVEC, s);
  launch_tau16(e->tau16, dm, tb, nmax, s);
  EpiArgs et{};
  et.in_fp16 = dm.fp16; et.out_f32 = e->tvec; et.ld_out = d; et.bias = e->b_t1;
  if ((err = launch_gemm_tc(EPI_BIAS_F32, e->tau16, e->w_t1dup, R, d, 2 * d, et, s)) != cudaSuccess) return err;
  launch_swish16(e->z16, e->tvec, (size_t)R * d, dm.fp16, s);
  et.bias = e->b_t2;
  if ((err = launch_gemm_tc(EPI_BIAS_F32, e->z16, e->w_t2, R, d, d, et, s)) != cudaSuccess) return err;
  launch_swish16(e->cond16, e->tvec, (size_t)R * d, dm.fp16, s);
  e->last_launches += 5;
  for (int k = 0; k < nmax; ++k) {
    EpiArgs ea{};
    ea.m_active = tb.m_active + k;
    ea.H = dm.H; ea.hd = dm.hd; ea.gu_blk = dm.gu_blk; ea.in_fp16 = dm.fp16; ea.out_fp16 = dm.fp16;
    ea.inv_d = 1.f / (float)d; ea.eps = dm.eps;
    // (scale, shift, gate) of all 2L+1 norms for this step's robots: mod[p][norm][3d]
    EpiArgs em{};
    em.in_fp16 = dm.fp16; em.out_f32 = e->mod; em.ld_out = n_mod; em.bias = e->b_mod;
    mark(e, ROSA_KC_TIMEVEC, s);
    if ((err = launch_gemm_tc(EPI_BIAS_F32, e->cond16 + (size_t)k * batch * d, e->w_mod, batch, n_mod, d, em, s)) != cudaSuccess) return err;
    mark(e, ROSA_KC_INPROJ, s);
    launch_embed_lin(e->h, e->x, e->wca, e->bca, dm, tb, k, M, s);
    e->last_launches += 2;
    for (int l = 0; l < dm.layers; ++l) {
      const LayerWeights& L = e->lw[l];
      const float* mod_a = e->mod + (size_t)(2 * l) * 3 * d;
      const float* mod_m = e->mod + (size_t)(2 * l + 1) * 3 * d;
      mark(e, ROSA_KC_RMSNORM, s);
      launch_adarms(e->nrm, e->h, mod_a, n_mod, dm, tb, k, M, s);
      e->last_launches += 1;
      ea.gate = nullptr;
      ea.out16 = e->qkv; ea.ld_out = dm.qkv_n;
      ea.rope_tab = e->rope_tab; ea.ids = tb.ids; ea.rlen = tb.rlen;
      ea.rope_cols = dm.q_n + dm.nkv * dm.hd;
      if ((err = gemm(e, ROSA_KC_GEMM_QKV, EPI_ROPE, e->nrm, L.wqkv, M, dm.qkv_n, d, ea, s)) != cudaSuccess) return err;
      mark(e, ROSA_KC_ATTN, s);
      if ((err = launch_attn_tc(dm, tb, l, e->qkv, e->obuf, k, M, e->d_kv_maps, e->attn_part, e->attn_flag, e->n_cta, s)) != cudaSuccess) return err;
      e->last_launches += 1;
      ea.out_f32 = e->h; ea.ld_out = d; ea.gate = mod_a + 2 * d; ea.gate_ld = n_mod;
      if ((err = gemm(e, ROSA_KC_GEMM_O, EPI_RESID, e->obuf, L.wo, M, d, dm.q_n, ea, s)) != cudaSuccess) return err;
      mark(e, ROSA_KC_RMSNORM, s);
      launch_adarms(e->nrm, e->h, mod_m, n_mod, dm, tb, k, M, s);
      e->last_launches += 1;
      ea.gate = nullptr;
      ea.out16 = e->mact; ea.ld_out = dm.F;
      if ((err = gemm(e, ROSA_KC_GEMM_GATEUP, EPI_GEGLU, e->nrm, L.wgu, M, 2 * dm.F, d, ea, s)) != cudaSuccess) return err;
      ea.out_f32 = e->h; ea.ld_out = d; ea.gate = mod_m + 2 * d; ea.gate_ld = n_mod;
      if ((err = gemm(e, ROSA_KC_GEMM_DOWN, EPI_RESID, e->mact, L.wdown, M, d, dm.F, ea, s)) != cudaSuccess) return err;
    }
    mark(e, ROSA_KC_RMSNORM, s);
    launch_adarms(e->nrm, e->h, e->mod + (size_t)(2 * dm.layers) * 3 * d, n_mod, dm, tb, k, M, s);
    e->last_launches += 1;
    ea.gate = nullptr;
    ea.bias = e->b_out; ea.x = e->x; ea.cp = cp; ea.dt = tb.dt; ea.src = tb.src; ea.A = dm.A; ea.k_iter = k;
    if ((err = gemm(e, ROSA_KC_FINAL, EPI_FINAL, e->nrm, e->w_out16, M, 64, d, ea, s)) != cudaSuccess) return err;
  }
  mark(e, ROSA_KC_GATHER_SCATTER, s);
  launch_scatter_x(cp, e->x, tb, dm.H * dm.A, s);
  e->last_launches += 1;
  mark(e, -1, s);
  return cudaGetLastError();
}

// All Euler iterations (a1..a10 x nmax) of a call on `s`.  `batch` is the graph's batch BUCKET: grids and row counts
// are sized for it, the rows that are live in iteration k come from the device table m_active[k].
static cudaError_t enqueue_steps(rosa_expert* e, const Tables& tb, int nmax, cudaStream_t s) {
  const Dims& dm = e->dm;
  const CallPtrs* cp = (const CallPtrs*)(e->d_call + e->off_ptrs);
  const int batch = tb.batch, M = batch * dm.H, d = dm.d;
  float *x = e->x, *h = e->h, *ssq = e->ssq;
  op16 *zbuf = e->zbuf, *nrm = e->nrm, *obuf = e->obuf, *mact = e->mact;
  bf16* qkv = e->qkv;
  cudaError_t err;
  const bool fused_norm = e->family == 1;  // RMSNorm fused into the GEMM epilogues (tcgen05 family)
  for (int k = 0; k < nmax; ++k) {
    struct StepRange { StepRange(int k) { char nm[32]; snprintf(nm, sizeof(nm), "rosa euler step %d", k); nvtxRangePushA(nm); }
                       ~StepRange() { nvtxRangePop(); } } step_range(k);
    EpiArgs ea{};
    ea.m_active = tb.m_active + k;
    ea.H = dm.H; ea.hd = dm.hd; ea.gu_blk = dm.gu_blk; ea.in_fp16 = dm.fp16; ea.out_fp16 = dm.fp16;
    ea.inv_d = 1.f / (float)d; ea.eps = dm.eps; ea.n_part = tc_ssq_parts(d);
    if (fused_norm) { ea.h16 = nrm; ea.ssq_out = ssq; ea.ssq_in = ssq; }
    // a1: h0 = W2 swish(W1 [tau ; W_in x + b_in] + b1) + b2
    mark(e, ROSA_KC_INPROJ, s);
    launch_embed1(zbuf, x, e->wca, e->bca, e->tvec + (size_t)k * batch * d, dm, tb, k, M, s);
    e->last_launches += 1;
    ea.out_f32 = h; ea.ld_out = d; ea.bias = e->b_t2;
    if ((err = gemm(e, ROSA_KC_GEMM_EMBED, EPI_BIAS_F32, zbuf, e->w_t2, M, d, d, ea, s)) != cudaSuccess) return err;
    for (int l = 0; l < dm.layers; ++l) {
      const LayerWeights& L = e->lw[l];
      if (!fused_norm) {
        mark(e, ROSA_KC_RMSNORM, s);
        launch_rmsnorm(nrm, h, dm, tb, k, M, s);                               // a2
        e->last_launches += 1;
      }
      ea.out16 = qkv; ea.ld_out = dm.qkv_n;
      ea.rope_tab = e->rope_tab; ea.ids = tb.ids; ea.rlen = tb.rlen;
      ea.rope_cols = dm.q_n + dm.nkv * dm.hd;
      if ((err = gemm(e, ROSA_KC_GEMM_QKV, EPI_ROPE, nrm, L.wqkv, M, dm.qkv_n, d, ea, s)) != cudaSuccess) return err;  // a2+a3+a4
      mark(e, ROSA_KC_ATTN, s);
      if (e->attn_tc) {                                                              // a5
        if ((err = launch_attn_tc(dm, tb, l, qkv, obuf, k, M, e->d_kv_maps, e->attn_part, e->attn_flag, e->n_cta, s)) != cudaSuccess) return err;
      } else {
        launch_attn_simple(dm, tb, l, qkv, obuf, k, e->cfg.max_prefix_len, s);
      }
      e->last_launches += 1;
      ea.out_f32 = h; ea.ld_out = d;
      if ((err = gemm(e, ROSA_KC_GEMM_O, EPI_RESID, obuf, L.wo, M, d, dm.q_n, ea, s)) != cudaSuccess) return err;    // a6
      if (!fused_norm) {
        mark(e, ROSA_KC_RMSNORM, s);
        launch_rmsnorm(nrm, h, dm, tb, k, M, s);                               // a2
        e->last_launches += 1;
      }
      ea.out16 = mact; ea.ld_out = dm.F;
      if ((err = gemm(e, ROSA_KC_GEMM_GATEUP, EPI_GEGLU, nrm, L.wgu, M, 2 * dm.F, d, ea, s)) != cudaSuccess) return err;  // a2+a7
      ea.out_f32 = h; ea.ld_out = d;
      if ((err = gemm(e, ROSA_KC_GEMM_DOWN, EPI_RESID, mact, L.wdown, M, d, dm.F, ea, s)) != cudaSuccess) return err;   // a8
    }
    if (fused_norm) {                                                                 // a9 + a10
      ea.bias = e->b_out; ea.x = x; ea.cp = cp; ea.dt = tb.dt; ea.src = tb.src; ea.A = dm.A; ea.k_iter = k;
      if ((err = gemm(e, ROSA_KC_FINAL, EPI_FINAL, nrm, e->w_out16, M, 64, d, ea, s)) != cudaSuccess) return err;
    } else {
      mark(e, ROSA_KC_FINAL, s);
      launch_final(x, cp, h, e->g_final, e->w_out, e->b_out, dm, tb, k, M, s);
      e->last_launches += 1;
    }
  }
  return cudaSuccess;
}

// Enqueue the whole call (steps a1..a11) on `s`.  Everything that changes from call to call (robots, their order,
// times, step counts, the number of live robots, the caller's pointers) is read from the device tables, so the
// sequence is captured once per (batch bucket, nmax) and replayed for any call that fits the bucket.
static cudaError_t enqueue_call(rosa_expert* e, int batch, int nmax, cudaStream_t s) {
  const Dims& dm = e->dm;
  if (dm.ada) return enqueue_call_ada(e, batch, nmax, s);
  const Tables tb = make_tables(e, batch);
  const CallPtrs* cp = (const CallPtrs*)(e->d_call + e->off_ptrs);
  const int d = dm.d;
  cudaError_t err;
  e->last_launches = 0;
  mark(e, ROSA_KC_GATHER_SCATTER, s);
  launch_gather_x(e->x, cp, tb, dm.H * dm.A, s);
  mark(e, ROSA_KC_TIMEVEC, s);
  if (e->family == 1 && tc_gemm_supported(d, 2 * d)) {  // a1 time half of every (step, robot) as one GEMM
    launch_tau16(e->tau16, dm, tb, nmax, s);
    EpiArgs et{};
    et.in_fp16 = dm.fp16; et.out_f32 = e->tvec; et.ld_out = d; et.bias = e->b_t1;
    if ((err = launch_gemm_tc(EPI_BIAS_F32, e->tau16, e->w_t1dup, nmax * batch, d, 2 * d, et, s)) != cudaSuccess) return err;
    e->last_launches += 3;
  } else {
    launch_timevec(e->tvec, e->w_t1, e->b_t1, dm, tb, nmax, s);
    e->last_launches += 2;
  }
  if ((err = enqueue_steps(e, tb, nmax, s)) != cudaSuccess) return err;
  mark(e, ROSA_KC_GATHER_SCATTER, s);
  launch_scatter_x(cp, e->x, tb, dm.H * dm.A, s);
  e->last_launches += 1;
  mark(e, -1, s);
  return cudaGetLastError();
}

static rosa_status_t denoise_impl(rosa_expert* e, int batch, const int32_t* ids, const float* noise,
                                  const float* t_start, const float* dt, const int32_t* n_steps,
                                  float* out, float* out_vel, cudaStream_t stream) {
  if (!e || !ids || !noise || !n_steps || !out) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  if (batch < 1) { set_error("batch < 1"); return ROSA_ERR_INVALID_ARG; }
  if (batch > e->cfg.max_batch) { set_error("batch > max_batch"); return ROSA_ERR_CAPACITY; }
  {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != e->device) {
      set_error("the expert was created on CUDA device " + std::to_string(e->device) + ", which is not the current device");
      return ROSA_ERR_INVALID_ARG;
    }
  }
  const Dims& dm = e->dm;
  int nmax = 0;
  std::vector<char> seen(e->cfg.max_robots, 0);
  for (int i = 0; i < batch; ++i) {
    if (ids[i] < 0 || ids[i] >= e->cfg.max_robots) { set_error("robot id out of range"); return ROSA_ERR_INVALID_ARG; }
    if (seen[ids[i]]) { set_error("duplicate robot id in batch"); return ROSA_ERR_INVALID_ARG; }
    seen[ids[i]] = 1;
    if (e->h_rlen[ids[i]] < 0) { set_error("robot has no prefix K/V bound"); return ROSA_ERR_UNBOUND_ROBOT; }
    if (n_steps[i] < 1) { set_error("n_steps < 1"); return ROSA_ERR_INVALID_ARG; }
    if (n_steps[i] > e->cfg.max_steps) { set_error("n_steps > max_steps"); return ROSA_ERR_CAPACITY; }
    nmax = std::max(nmax, (int)n_steps[i]);
  }
  // internal order: n_steps descending, so the robots live in iteration k are a prefix
  const std::vector<int> order = call_order(batch, n_steps);
  const int slot = e->stage_next;
  e->stage_next = (slot + 1) % kStageRing;
  CK(cudaEventSynchronize(e->stage_ev[slot]));  // the copy that last used this slot has completed
  char* hs = e->h_stage[slot];
  int* h_ids = (int*)(hs + e->off_ids); int* h_src = (int*)(hs + e->off_src);
  float* h_t0 = (float*)(hs + e->off_t0); float* h_dt = (float*)(hs + e->off_dt);
  int* h_ns = (int*)(hs + e->off_ns); int* h_ma = (int*)(hs + e->off_mact);
  for (int p = 0; p < batch; ++p) {
    const int i = order[p];
    h_ids[p] = ids[i]; h_src[p] = i;
    h_t0[p] = t_start ? t_start[i] : 1.0f;
    h_dt[p] = dt ? dt[i] : -h_t0[p] / (float)n_steps[i];
    h_ns[p] = n_steps[i];
  }
  std::vector<int> act(e->cfg.max_steps, 0);
  for (int k = 0; k < e->cfg.max_steps; ++k) {  // active token rows of iteration k
    for (int p = 0; p < batch; ++p) act[k] += h_ns[p] > k;
    h_ma[k] = act[k] * dm.H;
  }
  size_t copy_bytes = e->off_aiter;
  if (e->attn_tc) {
    // attention work lists (stream-K over the live robots' key streams): one per distinct live count
    std::vector<int> len(batch);
    for (int p = 0; p < batch; ++p) len[p] = e->h_rlen[h_ids[p]];
    int* h_iter = (int*)(hs + e->off_aiter);
    int* h_offs = (int*)(hs + e->off_aoffs);
    std::vector<AttnSeg>& segs = e->seg_tmp;
    segs.clear();
    int n_lists = 0;
    for (int k = 0; k < nmax; ++k) {
      if (k > 0 && act[k] == act[k - 1]) { h_iter[k] = h_iter[k - 1]; continue; }
      h_iter[k] = n_lists * (e->n_cta + 1);
      attn_build_list(dm, act[k], len.data(), e->n_cta, segs, h_offs + h_iter[k]);
      ++n_lists;
    }
    for (int k = nmax; k < e->cfg.max_steps; ++k) h_iter[k] = 0;
    for (AttnSeg& sg : segs) sg.robot = h_ids[sg.p];
    if (segs.size() > e->seg_cap) { set_error("attention work list overflow"); return ROSA_ERR_CAPACITY; }
    memcpy(hs + e->off_asegs, segs.data(), segs.size() * sizeof(AttnSeg));
    copy_bytes = e->off_asegs + segs.size() * sizeof(AttnSeg);
  }
  CallPtrs* h_cp = (CallPtrs*)(hs + e->off_ptrs);
  h_cp->noise = noise; h_cp->out = out; h_cp->vel = out_vel; h_cp->batch_ext = batch;
  if (e->bind_dirty) {   // table updates of binds since the last call: this call runs after them
    CK(cudaStreamWaitEvent(stream, e->bind_ev, 0));
    e->bind_dirty = false;
  }
  CK(cudaMemcpyAsync(e->d_call, hs, copy_bytes, cudaMemcpyHostToDevice, stream));
  CK(cudaEventRecord(e->stage_ev[slot], stream));
  if (out_vel) CK(cudaMemsetAsync(out_vel, 0, (size_t)nmax * batch * dm.H * dm.A * 4, stream));
  // The captured sequence is sized for a batch BUCKET (next power of two, at most max_batch): rows, robots and
  // work lists of the call itself come from the device tables, so one graph serves every call that fits the bucket.
  int bucket = 1;
  while (bucket < batch) bucket <<= 1;
  bucket = std::min(bucket, e->cfg.max_batch);
  if (!e->use_graph || e->prof_on) {
    CK(enqueue_call(e, bucket, nmax, stream));
    CK(cudaEventRecord(e->call_ev, stream));
    e->call_pending = true;
    return ROSA_OK;
  }
  const GraphKey key{bucket, nmax, 0};
  auto it = e->graphs.find(key);
  if (it == e->graphs.end()) {
    cudaGraph_t g = nullptr;
    nvtxRangePushA("rosa graph capture");
    CK(cudaStreamBeginCapture(e->cap_stream, cudaStreamCaptureModeThreadLocal));
    cudaError_t err = enqueue_call(e, bucket, nmax, e->cap_stream);
    cudaError_t err2 = cudaStreamEndCapture(e->cap_stream, &g);
    nvtxRangePop();
    if (err != cudaSuccess || err2 != cudaSuccess) {
      if (g) cudaGraphDestroy(g);
      set_error(std::string("graph capture failed: ") + cudaGetErrorString(err != cudaSuccess ? err : err2));
      return ROSA_ERR_CUDA;
    }
    cudaGraphExec_t ex = nullptr;
    CK(cudaGraphInstantiate(&ex, g, 0));
    cudaGraphDestroy(g);
    if (e->graphs.size() >= kMaxGraphs) {   // evict the least recently used graph (its launches have been enqueued: safe to destroy)
      auto victim = e->graphs.begin();
      for (auto g2 = e->graphs.begin(); g2 != e->graphs.end(); ++g2)
        if (e->graph_used[g2->first] < e->graph_used[victim->first]) victim = g2;
      cudaGraphExecDestroy(victim->second);
      e->graph_launches.erase(victim->first);
      e->graph_used.erase(victim->first);
      e->graphs.erase(victim);
    }
    it = e->graphs.emplace(key, ex).first;
    e->graph_launches[key] = e->last_launches;
    e->graph_captures += 1;
  }
  e->last_launches = e->graph_launches[key];
  e->graph_used[key] = ++e->graph_clock;
  CK(cudaGraphLaunch(it->second, stream));
  CK(cudaEventRecord(e->call_ev, stream));   // a later bind orders its table update after this call
  e->call_pending = true;
  return ROSA_OK;
}

}  // namespace rosa

// ===================================================================== C ABI
extern "C" {

rosa_status_t rosa_expert_create(const rosa_expert_config_t* c, const rosa_weights_t* w, rosa_expert_t** out) {
  if (!c || !w || !out) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  *out = nullptr;
  if (c->layers < 1 || c->d_model < 1 || c->n_q_heads < 1 || c->n_kv_heads < 1 || c->head_dim < 2 ||
      c->ffn < 1 || c->horizon < 1 || c->action_dim < 1 || c->max_robots < 1 || c->max_batch < 1 ||
      c->max_prefix_len < 0 || c->max_steps < 1) {
    set_error("non-positive dimension in config"); return ROSA_ERR_INVALID_ARG;
  }
  if (c->d_model % 64 || c->ffn % 64 || (c->n_q_heads * c->head_dim) % 64 || c->head_dim % 2 ||
      c->head_dim > 256 || c->n_q_heads % c->n_kv_heads || c->action_dim > 64 || c->horizon > 64) {
    set_error("unsupported shape (see rosa_expert_create in rosa.h)"); return ROSA_ERR_UNSUPPORTED;
  }
  if ((size_t)c->action_dim * c->d_model * 2 > 200 * 1024) {
    set_error("action_dim * d_model too large for the final projection's shared-memory copy of W_out"); return ROSA_ERR_UNSUPPORTED;
  }
  if ((size_t)c->n_q_heads * (c->head_dim + c->max_prefix_len + c->horizon + 1) * 4 > 220 * 1024) {
    set_error("max_prefix_len too large for the attention kernel's shared memory"); return ROSA_ERR_UNSUPPORTED;
  }
  const void* must[] = {w->w_in, w->b_in, w->w_t1, w->b_t1, w->w_t2, w->b_t2, w->w_out, w->b_out,
                        w->wq, w->wk, w->wv, w->wo, w->w_gate, w->w_up, w->w_down};
  for (const void* p : must) if (!p) { set_error("NULL weight pointer"); return ROSA_ERR_INVALID_ARG; }
  if (c->time_conditioning != 1 && (!w->g_final || !w->g_attn || !w->g_mlp)) {
    set_error("NULL weight pointer"); return ROSA_ERR_INVALID_ARG;
  }
  if (c->time_conditioning != 0 && c->time_conditioning != 1) { set_error("time_conditioning must be 0 or 1"); return ROSA_ERR_INVALID_ARG; }
  if (c->time_conditioning == 1) {
    const void* must_ada[] = {w->w_mod_attn, w->b_mod_attn, w->w_mod_mlp, w->b_mod_mlp, w->w_mod_final, w->b_mod_final};
    for (const void* p : must_ada) if (!p) { set_error("NULL modulation weight pointer"); return ROSA_ERR_INVALID_ARG; }
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    set_error("no CUDA device: librosa has no CPU fallback"); return ROSA_ERR_CUDA;
  }
  rosa_expert* e = new rosa_expert();
  e->cfg = *c;
  cudaGetDevice(&e->device);
  const char* fam = getenv("ROSA_KERNELS");
  // tcgen05 family needs head_dim == 256 (RoPE epilogue tile = one head) and 128/256-wide N tiles
  const bool tc_shape = c->head_dim == 256 && c->d_model % 128 == 0 && (2 * c->ffn) % 256 == 0;
  e->family = (fam && !strcmp(fam, "simple")) || !tc_shape ? 0 : 1;
  if (c->time_conditioning == 1 && e->family != 1) {
    delete e;
    set_error("time_conditioning = 1 needs the tcgen05 kernels (head_dim 256, d_model % 128 == 0, ROSA_KERNELS unset)");
    return ROSA_ERR_UNSUPPORTED;
  }
  const char* gr = getenv("ROSA_GRAPH");
  e->use_graph = !(gr && !strcmp(gr, "0"));
  rosa_status_t st = create_impl(c, w, e);
  if (st != ROSA_OK) { std::string keep = rosa_last_error(); destroy_impl(e); set_error(keep); return st; }
  *out = e;
  return ROSA_OK;
}

rosa_status_t rosa_expert_destroy(rosa_expert_t* e) {
  if (!e) { set_error("NULL expert"); return ROSA_ERR_INVALID_ARG; }
  destroy_impl(e);
  return ROSA_OK;
}

rosa_status_t rosa_prefix_kv_unbind(rosa_expert_t* e, int32_t robot) {
  if (!e) { set_error("NULL expert"); return ROSA_ERR_INVALID_ARG; }
  if (robot < 0 || robot >= e->cfg.max_robots) { set_error("robot id out of range"); return ROSA_ERR_CAPACITY; }
  e->h_rlen[robot] = -1;   // host-side only: library-owned copies stay allocated (a call in flight may still read them)
  return ROSA_OK;
}

rosa_status_t rosa_prefix_kv_bind(rosa_expert_t* e, int32_t robot, const void* const* k_layers,
                                  const void* const* v_layers, int32_t len, rosa_dtype_t dtype) {
  if (!e) { set_error("NULL expert"); return ROSA_ERR_INVALID_ARG; }
  if (robot < 0 || robot >= e->cfg.max_robots) { set_error("robot id out of range"); return ROSA_ERR_CAPACITY; }
  if (len < 0) { set_error("len < 0"); return ROSA_ERR_INVALID_ARG; }
  if (len > e->cfg.max_prefix_len) { set_error("len > max_prefix_len"); return ROSA_ERR_CAPACITY; }
  if (dtype != ROSA_F32 && dtype != ROSA_BF16) { set_error("bad dtype"); return ROSA_ERR_INVALID_ARG; }
  const Dims& dm = e->dm;
  if (len > 0) {
    if (!k_layers || !v_layers) { set_error("NULL K/V pointer array"); return ROSA_ERR_INVALID_ARG; }
    for (int l = 0; l < dm.layers; ++l) {
      if (!k_layers[l] || !v_layers[l]) { set_error("NULL K/V layer pointer"); return ROSA_ERR_INVALID_ARG; }
      if (((uintptr_t)k_layers[l] | (uintptr_t)v_layers[l]) & 15) { set_error("K/V pointer not 16-byte aligned"); return ROSA_ERR_INVALID_ARG; }
    }
  }
  e->h_rlen[robot] = -1;
  cudaStream_t bs = e->bind_stream;
  if (e->bind_pending[robot]) {   // the robot's pinned record may still be on its way: wait for the copies issued so far
    CK(cudaEventSynchronize(e->bind_ev));
    std::fill(e->bind_pending.begin(), e->bind_pending.end(), 0);
  }
  if (e->call_pending) {          // table updates (and fp32 conversions) run after every call enqueued so far
    CK(cudaStreamWaitEvent(bs, e->call_ev, 0));
    e->call_pending = false;
  }
  // pinned record of the robot: [K pointers | V pointers | tensor maps (64-byte aligned) | len]
  char* rec = e->h_bind + (size_t)robot * e->bind_rec;
  const bf16** hk = (const bf16**)rec;
  const bf16** hv = hk + dm.layers;
  const size_t mb = tc_attn_map_bytes();
  char* mp = rec + ((size_t)dm.layers * 2 * sizeof(void*) + 63) / 64 * 64;
  int* hl = (int*)(mp + (size_t)dm.layers * 2 * mb);
  const size_t n = (size_t)len * dm.nkv * dm.hd;
  for (int l = 0; l < dm.layers; ++l) hk[l] = hv[l] = nullptr;
  if (len > 0 && dtype == ROSA_BF16) {
    for (int l = 0; l < dm.layers; ++l) { hk[l] = (const bf16*)k_layers[l]; hv[l] = (const bf16*)v_layers[l]; }
  } else if (len > 0) {
    CK(cudaStreamSynchronize(bs));     // bs follows every call enqueued so far: none still reads the old copies
    if (e->owned_cap[robot] < n) {
      for (bf16* p : e->owned[robot]) cudaFree(p);
      e->owned[robot].clear();
      const size_t cap = (size_t)e->cfg.max_prefix_len * dm.nkv * dm.hd;
      for (int l = 0; l < 2 * dm.layers; ++l) {
        bf16* q = nullptr;
        CK(cudaMalloc((void**)&q, cap * 2));
        e->owned[robot].push_back(q);
      }
      e->owned_cap[robot] = cap;
    }
    for (int l = 0; l < dm.layers; ++l) {
      bf16 *ck = e->owned[robot][2 * l], *cv = e->owned[robot][2 * l + 1];
      // conversion on the legacy default stream, synchronously: the caller's fp32 tensors were produced in the
      // caller's stream order and may be released as soon as this call returns
      launch_f32_to_bf16(ck, (const float*)k_layers[l], n, 0);
      launch_f32_to_bf16(cv, (const float*)v_layers[l], n, 0);
      hk[l] = ck; hv[l] = cv;
    }
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(0));
  }
  CK(cudaMemcpyAsync(e->d_rk + (size_t)robot * dm.layers, hk, dm.layers * sizeof(void*), cudaMemcpyHostToDevice, bs));
  CK(cudaMemcpyAsync(e->d_rv + (size_t)robot * dm.layers, hv, dm.layers * sizeof(void*), cudaMemcpyHostToDevice, bs));
  if (e->attn_tc && len > 0) {
    for (int l = 0; l < dm.layers; ++l)
      if (!tc_attn_make_prefix_maps(mp + (size_t)l * 2 * mb, hk[l], hv[l], len, dm)) {
        set_error("cuTensorMapEncodeTiled failed for the prefix K/V"); return ROSA_ERR_CUDA;
      }
    CK(cudaMemcpyAsync(e->d_kv_maps + (size_t)robot * dm.layers * 2 * mb, mp, (size_t)dm.layers * 2 * mb,
                       cudaMemcpyHostToDevice, bs));
  }
  *hl = len;
  CK(cudaMemcpyAsync(e->d_rlen + robot, hl, 4, cudaMemcpyHostToDevice, bs));
  CK(cudaEventRecord(e->bind_ev, bs));
  e->bind_pending[robot] = 1;
  e->bind_dirty = true;
  e->h_rlen[robot] = len;
  return ROSA_OK;
}

rosa_status_t rosa_prefix_kv_produce(rosa_expert_t* e, int32_t d_prefix, const void* const* hidden_layers,
                                     const void* const* wk_layers, const void* const* wv_layers, int32_t len,
                                     void* const* k_out_layers, void* const* v_out_layers, void* stream) {
  if (!e || !hidden_layers || !wk_layers || !wv_layers || !k_out_layers || !v_out_layers) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  if (len < 0 || d_prefix < 1) { set_error("len < 0 or d_prefix < 1"); return ROSA_ERR_INVALID_ARG; }
  if (len > e->cfg.max_prefix_len) { set_error("len > max_prefix_len (the RoPE table ends there)"); return ROSA_ERR_CAPACITY; }
  const Dims& dm = e->dm;
  const int N = dm.nkv * dm.hd;
  if (e->family != 1 || dm.hd != 256 || d_prefix % 64) {
    set_error("rosa_prefix_kv_produce needs the tcgen05 kernels (head_dim 256) and d_prefix % 64 == 0"); return ROSA_ERR_UNSUPPORTED;
  }
  {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != e->device) { set_error("the expert lives on another CUDA device"); return ROSA_ERR_INVALID_ARG; }
  }
  if (len == 0) return ROSA_OK;
  for (int l = 0; l < dm.layers; ++l) {
    const void* ptrs[5] = {hidden_layers[l], wk_layers[l], wv_layers[l], k_out_layers[l], v_out_layers[l]};
    for (const void* q : ptrs) {
      if (!q) { set_error("NULL layer pointer"); return ROSA_ERR_INVALID_ARG; }
      if ((uintptr_t)q & 15) { set_error("layer pointer not 16-byte aligned"); return ROSA_ERR_INVALID_ARG; }
    }
  }
  cudaStream_t s = (cudaStream_t)stream;
  // K = RoPE(n W_pk^T) at positions 0..len-1, V = n W_pv^T: the QKV GEMM's kernel with its RoPE epilogue (a3 + a4),
  // bf16 operands (the backbone's hidden states and the cache are bf16), one head per 256-column tile.  The epilogue
  // takes a row's position from (ids, rlen, H) as rlen[ids[row / H]] + row % H: two device zeros and an H beyond
  // any row count make that the row index itself.
  EpiArgs ea{};
  ea.in_fp16 = 0; ea.out_fp16 = 0;
  ea.H = 1 << 30; ea.hd = dm.hd; ea.ld_out = N;
  ea.rope_tab = e->rope_tab; ea.ids = e->d_zero; ea.rlen = e->d_zero + 1;
  ea.inv_d = 1.f; ea.eps = 0.f;
  for (int l = 0; l < dm.layers; ++l) {
    ea.out16 = k_out_layers[l]; ea.rope_cols = N;
    CK(launch_gemm_tc(EPI_ROPE, (const op16*)hidden_layers[l], (const op16*)wk_layers[l], len, N, d_prefix, ea, s));
    ea.out16 = v_out_layers[l]; ea.rope_cols = 0;
    CK(launch_gemm_tc(EPI_ROPE, (const op16*)hidden_layers[l], (const op16*)wv_layers[l], len, N, d_prefix, ea, s));
  }
  return ROSA_OK;
}

rosa_status_t rosa_denoise_batch_ex(rosa_expert_t* e, int32_t batch, const int32_t* robot_ids, const float* noise,
                                    const float* t_start, const float* dt, const int32_t* n_steps,
                                    float* out_actions, float* out_velocity, void* stream) {
  return denoise_impl(e, batch, robot_ids, noise, t_start, dt, n_steps, out_actions, out_velocity,
                      (cudaStream_t)stream);
}

rosa_status_t rosa_denoise_batch(rosa_expert_t* e, int32_t batch, const int32_t* robot_ids, const float* noise,
                                 const float* t_start, const int32_t* n_steps, float* out_actions, void* stream) {
  return denoise_impl(e, batch, robot_ids, noise, t_start, nullptr, n_steps, out_actions, nullptr,
                      (cudaStream_t)stream);
}

rosa_status_t rosa_denoise_batch_host(rosa_expert_t* e, int32_t batch, const int32_t* robot_ids,
                                      const float* noise_host, const float* t_start, const float* dt,
                                      const int32_t* n_steps, float* out_actions_host, void* stream) {
  if (!e || !noise_host || !out_actions_host) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  if (batch < 1 || batch > e->cfg.max_batch) { set_error("batch out of range"); return ROSA_ERR_CAPACITY; }
  cudaStream_t s = (cudaStream_t)stream;
  const size_t bytes = (size_t)batch * e->dm.H * e->dm.A * 4;
  CK(cudaMemcpyAsync(e->e2e_dev, noise_host, bytes, cudaMemcpyHostToDevice, s));
  rosa_status_t st = denoise_impl(e, batch, robot_ids, e->e2e_dev, t_start, dt, n_steps, e->e2e_dev, nullptr, s);
  if (st != ROSA_OK) return st;
  CK(cudaMemcpyAsync(out_actions_host, e->e2e_dev, bytes, cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return ROSA_OK;
}

rosa_status_t rosa_profile_batch(rosa_expert_t* e, int32_t batch, const int32_t* robot_ids, const float* noise,
                                 const float* t_start, const float* dt, const int32_t* n_steps,
                                 float* out_actions, void* stream, float* ms_out, int32_t* launches_out) {
  if (!e || !ms_out || !launches_out) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  e->prof_on = true;
  e->prof_n = 0;
  rosa_status_t st = denoise_impl(e, batch, robot_ids, noise, t_start, dt, n_steps, out_actions, nullptr, s);
  e->prof_on = false;
  if (st != ROSA_OK) return st;
  CK(cudaStreamSynchronize(s));
  for (int c = 0; c < ROSA_KC_COUNT; ++c) { ms_out[c] = 0.f; launches_out[c] = 0; }
  for (size_t i = 0; i + 1 < e->prof_n; ++i) {
    const int c = e->prof_cls[i];
    if (c < 0 || c >= ROSA_KC_COUNT) continue;
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e->prof_ev[i], e->prof_ev[i + 1]));
    ms_out[c] += ms;
    launches_out[c] += 1;
  }
  return ROSA_OK;
}

const char* rosa_kernel_class_name(int32_t cls) {
  static const char* names[ROSA_KC_COUNT] = {"gather_scatter", "timevec", "inproj", "gemm_embed", "rmsnorm",
                                             "gemm_qkv_rope", "attention", "gemm_o_resid", "gemm_gateup_geglu",
                                             "gemm_down_resid", "final_norm_outproj_euler"};
  return cls >= 0 && cls < ROSA_KC_COUNT ? names[cls] : "";
}

rosa_status_t rosa_last_launch_count(rosa_expert_t* e, int64_t* n) {
  if (!e || !n) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  *n = e->last_launches;
  return ROSA_OK;
}
rosa_status_t rosa_kernel_family(rosa_expert_t* e, int32_t* family) {
  if (!e || !family) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  *family = e->family;
  return ROSA_OK;
}

rosa_status_t rosa_debug_graph_captures(rosa_expert_t* e, int64_t* n) {
  if (!e || !n) { set_error("NULL argument"); return ROSA_ERR_INVALID_ARG; }
  *n = e->graph_captures;
  return ROSA_OK;
}

rosa_status_t rosa_debug_gemm(int32_t family, int32_t epi, int32_t pair, int32_t bn, int32_t fp16, int32_t M, int32_t N,
                              int32_t K, const void* A, const void* W, float* C, const float* bias, void* h16,
                              float* ssq, void* stream) {
  if (!A || !W || !C || M < 1 || N < 1 || K < 1) { set_error("bad argument"); return ROSA_ERR_INVALID_ARG; }
  if (epi != EPI_STORE_F32 && epi != EPI_BIAS_F32 && epi != EPI_RESID) { set_error("epi must be 0, 2 or 4"); return ROSA_ERR_INVALID_ARG; }
  if (epi == EPI_BIAS_F32 && !bias) { set_error("bias is NULL"); return ROSA_ERR_INVALID_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  if (family == 0) {
    if (epi != EPI_STORE_F32) { set_error("family 0: epi 0 only"); return ROSA_ERR_UNSUPPORTED; }
    launch_gemm_naive((const op16*)A, (const op16*)W, C, M, N, K, fp16, nullptr, s);
    CK(cudaGetLastError());
    return ROSA_OK;
  }
  if (!tc_gemm_supported(N, K)) { set_error("shape not supported by the tcgen05 GEMM"); return ROSA_ERR_UNSUPPORTED; }
  EpiArgs ea{};
  ea.out_f32 = C; ea.ld_out = N; ea.bias = bias; ea.h16 = h16; ea.ssq_out = ssq;
  ea.in_fp16 = fp16; ea.out_fp16 = fp16;
  ea.force_bn = bn; ea.force_pair = pair < 0 ? 0 : (pair ? 2 : 1);
  cudaError_t err = launch_gemm_tc((Epi)epi, (const op16*)A, (const op16*)W, M, N, K, ea, s);
  if (err == cudaErrorNotSupported) { set_error("no kernel for this (pair, bn)"); return ROSA_ERR_UNSUPPORTED; }
  CK(err);
  return ROSA_OK;
}

int32_t rosa_debug_attn_plan(int32_t horizon, int32_t n_robots, const int32_t* len, int32_t n_cta, int32_t* offs_out,
                             int32_t* segs_out, int32_t cap) {
  if (horizon < 1 || n_robots < 1 || !len || n_cta < 1 || !offs_out || !segs_out) { set_error("bad argument"); return ROSA_ERR_INVALID_ARG; }
  Dims dm{};
  dm.H = horizon;
  std::vector<AttnSeg> segs;
  const int n = attn_build_list(dm, n_robots, len, n_cta, segs, offs_out);
  if (n > cap) { set_error("cap too small"); return ROSA_ERR_CAPACITY; }
  for (int i = 0; i < n; ++i) {
    int32_t* o = segs_out + 8 * i;
    o[0] = segs[i].p; o[1] = segs[i].tt; o[2] = segs[i].kb0; o[3] = segs[i].kb1;
    o[4] = segs[i].n_part; o[5] = segs[i].part0; o[6] = 0; o[7] = 0;
  }
  return n;
}

const char* rosa_last_error(void) { return g_err.c_str(); }
int32_t rosa_version(void) { return 1; }

}  // extern "C"
