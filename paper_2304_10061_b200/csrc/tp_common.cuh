// Warp-level helpers shared by the tensor-track kernels (tp_kernels.cu, tp2_kernels.cu).
#pragma once
#include <cuda_runtime.h>

#define TP_FULLMASK 0xffffffffu

__device__ __forceinline__ float tp_wsum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(TP_FULLMASK, v, o);
  return v;
}

// Sum each of 8 per-lane values over the 32 lanes with 9 shuffles (halving butterfly): on return the
// lane holds the total of value index ((lane>>4)&1)*4 + ((lane>>3)&1)*2 + ((lane>>2)&1).
__device__ __forceinline__ float tp_reduce8(const float* v, int lane) {
  float a[4], b[2], c;
  const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float send = h16 ? v[i] : v[i + 4], keep = h16 ? v[i + 4] : v[i];
    a[i] = keep + __shfl_xor_sync(TP_FULLMASK, send, 16);
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    float send = h8 ? a[i] : a[i + 2], keep = h8 ? a[i + 2] : a[i];
    b[i] = keep + __shfl_xor_sync(TP_FULLMASK, send, 8);
  }
  {
    float send = h4 ? b[0] : b[1], keep = h4 ? b[1] : b[0];
    c = keep + __shfl_xor_sync(TP_FULLMASK, send, 4);
  }
  c += __shfl_xor_sync(TP_FULLMASK, c, 2);
  c += __shfl_xor_sync(TP_FULLMASK, c, 1);
  return c;
}

// yrow[base + k] (+)= sum over lanes of p[k], k < D, for the first `nvalid` values (deterministic order).
// INIT: plain store instead of accumulation (first writer of this Y-bar row in the step).
template <int D, bool INIT>
__device__ __forceinline__ void tp_ybar_rows(float* yrow, const float* p, int base, int nvalid, int lane) {
  const int sel = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
#pragma unroll
  for (int k0 = 0; k0 + 8 <= D; k0 += 8) {
    float r = tp_reduce8(p + k0, lane);
    if ((lane & 3) == 0 && k0 + sel < nvalid) {
      if (INIT) yrow[base + k0 + sel] = r; else yrow[base + k0 + sel] += r;
    }
  }
#pragma unroll
  for (int k = (D / 8) * 8; k < D; ++k) {
    float s = tp_wsum(p[k]);
    if (lane == 0 && k < nvalid) {
      if (INIT) yrow[base + k] = s; else yrow[base + k] += s;
    }
  }
}

__device__ __forceinline__ void tp_cp16(float* smem_dst, const float* gsrc) {
  unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void tp_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void tp_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ROWS rows of 32 floats (128 B): smem dst row r at dst + 32 r, global row r at src + r * rstride
template <int ROWS>
__device__ __forceinline__ void tp_cp_rows(float* dst, const float* src, int rstride, int lane) {
#pragma unroll
  for (int i0 = 0; i0 < ROWS * 8; i0 += 32) {
    int i = i0 + lane;
    if (i < ROWS * 8) tp_cp16(dst + (i >> 3) * 32 + (i & 7) * 4, src + (size_t)(i >> 3) * rstride + (i & 7) * 4);
  }
}

// Same copy with the per-lane source offsets (in floats) hoisted out of the edge loop:
//   off[it] = row * rstride + 4 * (chunk within the row), for chunk i = 32 it + lane; destination offset = 4 i.
template <int ROWS>
__device__ __forceinline__ void tp_row_offsets(int* off, int rstride, int lane) {
#pragma unroll
  for (int it = 0; it < (ROWS * 8 + 31) / 32; ++it) {
    int i = it * 32 + lane;
    off[it] = (i >> 3) * rstride + (i & 7) * 4;
  }
}
template <int ROWS>
__device__ __forceinline__ void tp_cp_rows_pre(float* dst, const float* src, const int* off, int lane) {
#pragma unroll
  for (int it = 0; it < (ROWS * 8 + 31) / 32; ++it) {
    if (it * 32 + lane < ROWS * 8) tp_cp16(dst + (it * 32 + lane) * 4, src + off[it]);
  }
}

#ifndef TP_FFMA2
#define TP_FFMA2 1
#endif
__device__ __forceinline__ float2 tp_fma2(float2 a, float2 b, float2 c) {
#if TP_FFMA2
  return __ffma2_rn(a, b, c);
#else
  return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y));
#endif
}
