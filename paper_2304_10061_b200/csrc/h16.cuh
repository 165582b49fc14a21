// 16-bit storage helpers of the 16-bit operand modes (precision 2: bf16, precision 4: fp16; allegro_model::hfmt = 1 / 0).
// Tensors that are GEMM operands in those modes (a_k, x^L, s^L, z-bar, omega-bar, w0-bar) and the pre-activations kept for SiLU'
// are stored as 16-bit; the producers outside the GEMM (first two-body layer, tensor-track kernels) store through these.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

__device__ __forceinline__ uint16_t h16_from_float(float v, int fmt) {
  if (fmt == 0) { __half h = __float2half_rn(v); return *reinterpret_cast<uint16_t*>(&h); }
  __nv_bfloat16 b = __float2bfloat16_rn(v);
  return *reinterpret_cast<uint16_t*>(&b);
}
__device__ __forceinline__ uint2 h16_pack4(float4 v, int fmt) {
  uint2 o;
  o.x = (uint32_t)h16_from_float(v.x, fmt) | ((uint32_t)h16_from_float(v.y, fmt) << 16);
  o.y = (uint32_t)h16_from_float(v.z, fmt) | ((uint32_t)h16_from_float(v.w, fmt) << 16);
  return o;
}
// store one value / four consecutive values at ELEMENT offset `off` of a tensor whose elements are 16-bit (fmt >= 0) or fp32
__device__ __forceinline__ void h16_store(void* base, size_t off, float v, int fmt) {
  if (fmt < 0) reinterpret_cast<float*>(base)[off] = v;
  else reinterpret_cast<uint16_t*>(base)[off] = h16_from_float(v, fmt);
}
__device__ __forceinline__ void h16_store4(void* base, size_t off, float4 v, int fmt) {
  if (fmt < 0) *reinterpret_cast<float4*>(reinterpret_cast<float*>(base) + off) = v;
  else *reinterpret_cast<uint2*>(reinterpret_cast<uint16_t*>(base) + off) = h16_pack4(v, fmt);
}
