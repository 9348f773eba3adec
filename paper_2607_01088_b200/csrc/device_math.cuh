// Scalar device math shared by every kernel of librosa (readings R3, R6).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace rosa {

// Programmatic dependent launch: every kernel of the call is launched with the attribute (rosa_internal.h
// launch_k), so its prologue overlaps the tail of the previous kernel.  pdl_wait() returns when the
// previous kernel in the stream has completed and its writes are visible; nothing that depends on or
// overwrites earlier kernels' data may happen before it.  pdl_trigger() lets the next kernel start launching.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// 16-bit GEMM operand conversions (fp16 or bf16 bits, warp-uniform selector)
__device__ __forceinline__ uint16_t f2op(float v, int fp16) {
  return fp16 ? __half_as_ushort(__float2half_rn(v)) : __bfloat16_as_ushort(__float2bfloat16_rn(v));
}
__device__ __forceinline__ float op2f(uint16_t b, int fp16) {
  return fp16 ? __half2float(__ushort_as_half(b)) : __bfloat162float(__ushort_as_bfloat16(b));
}
__device__ __forceinline__ uint32_t pack_op2(float lo, float hi, int fp16) {
  if (fp16) {
    __half2 v = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
  }
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
// swish(z) = z / (1 + e^-z)
__device__ __forceinline__ float swish_f(float z) { return __fdividef(z, 1.f + __expf(-z)); }
// GELU, tanh form (R6): 0.5 z (1 + tanh(sqrt(2/pi) (z + 0.044715 z^3)))
// tanh(u) = 1 - 2/(1 + e^{2u}) keeps full fp32 accuracy for the range that matters.
__device__ __forceinline__ float gelu_tanh_f(float z) {
  const float u = 0.7978845608028654f * fmaf(0.044715f * z * z, z, z);
  const float t = 1.f - __fdividef(2.f, 1.f + __expf(2.f * u));
  return 0.5f * z * (1.f + t);
}

}  // namespace rosa
