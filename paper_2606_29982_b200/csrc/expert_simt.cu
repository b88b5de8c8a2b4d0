// expert_simt.cu — S7 grouped SwiGLU FFN on the plain fp32 ALUs (E_e(t)).
//
// This is the expert path for fp32 weights (BASELINE.json config 1, tolerance 1e-4 x RMS,
// which rules out the tensor cores' tf32/bf16 inputs) and a cross-check for the tcgen05
// path on bf16 / e4m3 weights.  One warp per weight row, tokens of the run in register
// chunks, fp32 accumulate, h kept in fp32.  Runs come from the device-side work list, so
// pruned experts cost nothing: their rows are never touched.
#include "caee_internal.cuh"

namespace {

constexpr int TCH = 4;      // tokens per register chunk
constexpr int WARPS = 8;    // rows per block

struct f4 { float v[4]; };

template <typename T> __device__ __forceinline__ f4 ld4(const T* p, size_t i);
template <> __device__ __forceinline__ f4 ld4<float>(const float* p, size_t i) {
  float4 a = *reinterpret_cast<const float4*>(p + i);
  return {{a.x, a.y, a.z, a.w}};
}
template <> __device__ __forceinline__ f4 ld4<__nv_bfloat16>(const __nv_bfloat16* p, size_t i) {
  uint2 a = *reinterpret_cast<const uint2*>(p + i);
  return {{__uint_as_float(a.x << 16), __uint_as_float(a.x & 0xffff0000u), __uint_as_float(a.y << 16),
           __uint_as_float(a.y & 0xffff0000u)}};
}
// e4m3 -> fp32, exact: via the f16x2 conversion (every e4m3 value is an f16 value)
template <> __device__ __forceinline__ f4 ld4<uint8_t>(const uint8_t* p, size_t i) {
  uint32_t a = *reinterpret_cast<const uint32_t*>(p + i);
  uint32_t lo, hi;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(lo) : "h"((uint16_t)(a & 0xffffu)));
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(hi) : "h"((uint16_t)(a >> 16)));
  __half2 l2 = *reinterpret_cast<__half2*>(&lo), h2 = *reinterpret_cast<__half2*>(&hi);
  return {{__low2float(l2), __high2float(l2), __low2float(h2), __high2float(h2)}};
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// h[row, i] = silu(W_g[i,:] . x) * (W_u[i,:] . x) for the tokens of run blockIdx.y
template <typename WT, typename XT>
__global__ void __launch_bounds__(WARPS * 32) k_simt_gateup(caee_worklist wl, const void* const* __restrict__ wg,
                                                            const void* const* __restrict__ wu,
                                                            const float* const* __restrict__ sg,
                                                            const float* const* __restrict__ su, const XT* __restrict__ x,
                                                            float* __restrict__ hbuf, int H, int I) {
  const int r = blockIdx.y;
  if (r >= wl.meta[1]) return;
  const int lane = threadIdx.x & 31, i = blockIdx.x * WARPS + (threadIdx.x >> 5);
  if (i >= I) return;
  const int e = wl.run_expert[r], start = wl.run_start[r], n = wl.run_n[r], hrow = wl.run_hrow[r];
  const WT* g = static_cast<const WT*>(wg[e]) + (size_t)i * H;
  const WT* u = static_cast<const WT*>(wu[e]) + (size_t)i * H;
  const int nbc = (H + 127) / 128;
  const float* sgr = (sizeof(WT) == 1 && sg && sg[e]) ? sg[e] + (size_t)(i / 128) * nbc : nullptr;
  const float* sur = (sizeof(WT) == 1 && su && su[e]) ? su[e] + (size_t)(i / 128) * nbc : nullptr;
  for (int n0 = 0; n0 < n; n0 += TCH) {
    int tok[TCH];
#pragma unroll
    for (int q = 0; q < TCH; ++q) tok[q] = wl.ent_tok[start + min(n0 + q, n - 1)];
    float ag[TCH] = {}, au[TCH] = {};
    for (int h = lane * 4; h < H; h += 128) {
      f4 a = ld4<WT>(g, h), b = ld4<WT>(u, h);
      if (sgr) {
        float s1 = sgr[h / 128], s2 = sur[h / 128];
#pragma unroll
        for (int c = 0; c < 4; ++c) { a.v[c] *= s1; b.v[c] *= s2; }
      }
#pragma unroll
      for (int q = 0; q < TCH; ++q) {
        f4 xv = ld4<XT>(x, (size_t)tok[q] * H + h);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          ag[q] = fmaf(a.v[c], xv.v[c], ag[q]);
          au[q] = fmaf(b.v[c], xv.v[c], au[q]);
        }
      }
    }
#pragma unroll
    for (int q = 0; q < TCH; ++q) {
      float gq = warp_sum(ag[q]), uq = warp_sum(au[q]);
      if (lane == 0 && n0 + q < n) hbuf[(size_t)(hrow + n0 + q) * I + i] = gq / (1.0f + expf(-gq)) * uq;
    }
  }
}

// o[dst, r_out] = W_d[r_out,:] . h[row,:]
template <typename WT>
__global__ void __launch_bounds__(WARPS * 32) k_simt_down(caee_worklist wl, const void* const* __restrict__ wd,
                                                          const float* const* __restrict__ sd,
                                                          const float* __restrict__ hbuf, float* __restrict__ obuf, int H,
                                                          int I) {
  const int r = blockIdx.y;
  if (r >= wl.meta[1]) return;
  const int lane = threadIdx.x & 31, ro = blockIdx.x * WARPS + (threadIdx.x >> 5);
  if (ro >= H) return;
  const int e = wl.run_expert[r], start = wl.run_start[r], n = wl.run_n[r], hrow = wl.run_hrow[r];
  const WT* w = static_cast<const WT*>(wd[e]) + (size_t)ro * I;
  const int nbc = (I + 127) / 128;
  const float* sr = (sizeof(WT) == 1 && sd && sd[e]) ? sd[e] + (size_t)(ro / 128) * nbc : nullptr;
  for (int n0 = 0; n0 < n; n0 += TCH) {
    float acc[TCH] = {};
    for (int i = lane * 4; i < I; i += 128) {
      f4 a = ld4<WT>(w, i);
      if (sr) {
        float s1 = sr[i / 128];
#pragma unroll
        for (int c = 0; c < 4; ++c) a.v[c] *= s1;
      }
#pragma unroll
      for (int q = 0; q < TCH; ++q) {
        f4 hv = ld4<float>(hbuf, (size_t)(hrow + min(n0 + q, n - 1)) * I + i);
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[q] = fmaf(a.v[c], hv.v[c], acc[q]);
      }
    }
#pragma unroll
    for (int q = 0; q < TCH; ++q) {
      float v = warp_sum(acc[q]);
      if (lane == 0 && n0 + q < n) caee_o_base(wl, obuf, wl.ent_tok[start + n0 + q])[(size_t)wl.ent_dst[start + n0 + q] * H + ro] = v;
    }
  }
}

template <typename WT>
void launch(caee_ctx* c, const void* x, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  dim3 g1(caee_ceil_div(d.I, WARPS), c->wl.max_runs), g2(caee_ceil_div(d.H, WARPS), c->wl.max_runs);
  if (d.act_dtype == CAEE_F32)
    k_simt_gateup<WT, float><<<g1, WARPS * 32, 0, st>>>(c->wl, c->wg, c->wu, c->sg, c->su, (const float*)x, c->hbuf_f32,
                                                        d.H, d.I);
  else
    k_simt_gateup<WT, __nv_bfloat16><<<g1, WARPS * 32, 0, st>>>(c->wl, c->wg, c->wu, c->sg, c->su,
                                                                (const __nv_bfloat16*)x, c->hbuf_f32, d.H, d.I);
  k_simt_down<WT><<<g2, WARPS * 32, 0, st>>>(c->wl, c->wd, c->sd, c->hbuf_f32, c->obuf, d.H, d.I);
}

}  // namespace

void caee_launch_expert_simt(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  (void)T;
  c->n_launches += 2;
  switch (c->d.w_dtype) {
    case CAEE_F32: launch<float>(c, x, st); break;
    case CAEE_BF16: launch<__nv_bfloat16>(c, x, st); break;
    default: launch<uint8_t>(c, x, st); break;
  }
}
