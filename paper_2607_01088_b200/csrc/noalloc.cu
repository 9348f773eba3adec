// rosa_linear_noalloc (include/rosa.h): one linear layer of the path, C = epi(A W^T), for callers that cannot
// call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).
//
// It is the CUDA-core GEMM family's pair of kernels (kernels_simple.cu: k_gemm_naive writes the fp32 product into a
// scratch matrix, k_epilogue applies bias / residual and writes the result; in an expert that scratch is a
// cudaMalloc'ed workspace) with the scratch in a FILE-SCOPE DEVICE ARRAY instead: nothing is allocated, by this
// entry point or by anything it calls.  Every GPU that loads the library holds the array (4 MiB) until exit.
//
// The array's name is a host-side stand-in in host code, not a device address: its address on the CURRENT device is
// looked up once per device with cudaGetSymbolAddress and that pointer is what the kernels get.
// All calls share the array and it keeps the last call's contents.  Nothing has to start at zero (the GEMM kernel
// overwrites every element of the [M, N] product before the epilogue reads it), but two calls that overlap on the
// GPU - different streams without an ordering between them - race on it: serialise them.
#include "rosa_internal.h"

namespace rosa {

// fp32 [M, N] product of one call; M * N <= ROSA_NOALLOC_MAX_ELEMS (rosa.h)
static __device__ __align__(256) float g_noalloc_scratch[ROSA_NOALLOC_MAX_ELEMS];

// device address of the array on the current device (set-up: once per device, with that device current)
static cudaError_t noalloc_scratch_ptr(float** out) {
  static float* ptrs[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  if (!ptrs[dev]) {
    float* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    ptrs[dev] = p;
  }
  *out = ptrs[dev];
  return cudaSuccess;
}

}  // namespace rosa

using namespace rosa;

extern "C" rosa_status_t rosa_linear_noalloc(int32_t epi, int32_t fp16, int32_t M, int32_t N, int32_t K, const void* A,
                                             const void* W, const float* bias, float* C, void* stream) {
  if (!A || !W || !C || M < 1 || N < 1 || K < 1) { set_error("rosa_linear_noalloc: NULL pointer or non-positive size"); return ROSA_ERR_INVALID_ARG; }
  if (epi != EPI_STORE_F32 && epi != EPI_BIAS_F32 && epi != EPI_RESID) { set_error("rosa_linear_noalloc: epi must be 0 (store), 2 (+ bias) or 4 (+= residual)"); return ROSA_ERR_INVALID_ARG; }
  if (epi == EPI_BIAS_F32 && !bias) { set_error("rosa_linear_noalloc: bias is NULL"); return ROSA_ERR_INVALID_ARG; }
  if ((int64_t)M * (int64_t)N > (int64_t)ROSA_NOALLOC_MAX_ELEMS) {
    set_error("rosa_linear_noalloc: M * N = " + std::to_string((int64_t)M * N) + " exceeds the static scratch of " +
              std::to_string((int64_t)ROSA_NOALLOC_MAX_ELEMS) + " elements (ROSA_NOALLOC_MAX_ELEMS); split the rows or use an expert");
    return ROSA_ERR_CAPACITY;
  }
  float* scratch = nullptr;
  cudaError_t e = noalloc_scratch_ptr(&scratch);
  if (e != cudaSuccess) { set_error(std::string("rosa_linear_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e)); return ROSA_ERR_CUDA; }
  cudaStream_t s = (cudaStream_t)stream;
  launch_gemm_naive((const op16*)A, (const op16*)W, scratch, M, N, K, fp16 ? 1 : 0, nullptr, s);
  EpiArgs ea{};
  ea.out_f32 = C; ea.ld_out = N; ea.bias = bias;
  launch_epilogue((Epi)epi, scratch, M, N, ea, s);
  e = cudaGetLastError();
  if (e != cudaSuccess) { set_error(std::string("rosa_linear_noalloc: launch: ") + cudaGetErrorString(e)); return ROSA_ERR_CUDA; }
  return ROSA_OK;
}
