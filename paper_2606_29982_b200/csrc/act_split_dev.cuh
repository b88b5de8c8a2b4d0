// act_split_dev.cuh — the e4m3 decode kernel's activation split (expert_fp8.cu): one 128-wide block of a bf16
// row -> a / s = hi + lo (both e4m3) with the block's fp32 scale s = amax / 448.  One warp per block, 4 values
// per lane.  Shared by k_act_split (expert_fp8.cu) and the one-CTA decision kernel (decide.cu), which splits x
// itself in steps of <= 16 tokens while it waits for the router GEMM.
#pragma once
#include "caee_internal.cuh"

// two floats -> two e4m3 codes (low byte = a), round to nearest even, saturating
__device__ __forceinline__ uint16_t caee_cvt_e4m3x2(float a, float b) {
  uint16_t r;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(b), "f"(a));
  return r;
}
// two e4m3 codes -> two floats (exact)
__device__ __forceinline__ float2 caee_e4m3x2_to_float2(uint16_t v) {
  uint32_t h2;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"(v));
  return __half22float2(*reinterpret_cast<__half2*>(&h2));
}
// a/s as hi + lo (both e4m3), for a pair of values
__device__ __forceinline__ void caee_split_pair(float a, float b, float inv_s, uint16_t& hi, uint16_t& lo) {
  const float va = a * inv_s, vb = b * inv_s;
  hi = caee_cvt_e4m3x2(va, vb);
  const float2 h = caee_e4m3x2_to_float2(hi);
  lo = caee_cvt_e4m3x2(va - h.x, vb - h.y);
}

// block b of x (128 consecutive elements) by one warp
__device__ __forceinline__ void caee_act_split_block(const __nv_bfloat16* __restrict__ x, uint8_t* __restrict__ hi,
                                                     uint8_t* __restrict__ lo, float* __restrict__ scale, size_t b, int lane) {
  const uint2 u = *reinterpret_cast<const uint2*>(x + b * 128 + lane * 4);
  const float v0 = __uint_as_float(u.x << 16), v1 = __uint_as_float(u.x & 0xffff0000u);
  const float v2 = __uint_as_float(u.y << 16), v3 = __uint_as_float(u.y & 0xffff0000u);
  float m = fmaxf(fmaxf(fabsf(v0), fabsf(v1)), fmaxf(fabsf(v2), fabsf(v3)));
#pragma unroll
  for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  const float s = m > 0.f ? m * (1.0f / 448.0f) : 1.0f;
  const float inv = 1.0f / s;
  uint16_t h01, l01, h23, l23;
  caee_split_pair(v0, v1, inv, h01, l01);
  caee_split_pair(v2, v3, inv, h23, l23);
  *reinterpret_cast<uint32_t*>(hi + b * 128 + lane * 4) = (uint32_t)h01 | ((uint32_t)h23 << 16);
  *reinterpret_cast<uint32_t*>(lo + b * 128 + lane * 4) = (uint32_t)l01 | ((uint32_t)l23 << 16);
  if (lane == 0) scale[b] = s;
}
