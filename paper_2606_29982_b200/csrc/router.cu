// router.cu — S0 router scores and S1 group-limited top-k + gates (router
// form per DESIGN.md reading R1).  Plain fp32 ALUs: E <= 512 and the GEMV is a few MB.
//
//  k_router_logits : split-K partial logits  partial[ks][t][e] = sum_{h in chunk ks} x[t,h] W_r[e,h]
//                    (fixed summation order => deterministic scores)
//  k_route_topk    : one warp per token: reduce partials, activation, selection, gates.
#include "caee_internal.cuh"
#include "warp_select.cuh"

namespace {

constexpr int TT = 32, TE = 32, KC = 32;

template <typename XT>
__device__ __forceinline__ float ld_act(const XT* p, size_t i);
template <>
__device__ __forceinline__ float ld_act<float>(const float* p, size_t i) { return p[i]; }
template <>
__device__ __forceinline__ float ld_act<__nv_bfloat16>(const __nv_bfloat16* p, size_t i) {
  return __bfloat162float(p[i]);
}

template <typename XT>
__global__ void __launch_bounds__(256) k_router_logits(const XT* __restrict__ x, const float* __restrict__ Wr,
                                                       float* __restrict__ partial, int T, int H, int E, int Hs) {
  __shared__ float xs[KC][TT + 1];
  __shared__ float ws[KC][TE + 1];
  const int e0 = blockIdx.x * TE, t0 = blockIdx.y * TT, ks = blockIdx.z;
  const int h_lo = ks * Hs, h_hi = min(H, h_lo + Hs);
  const int tid = threadIdx.x;
  const int ty = tid >> 4, tx = tid & 15;  // 16 x 16 threads, 2 x 2 outputs each
  float acc[2][2] = {{0.f, 0.f}, {0.f, 0.f}};
  const int lr = tid >> 3, lc = (tid & 7) * 4;  // loader: row 0..31, 4 consecutive h
  for (int h0 = h_lo; h0 < h_hi; h0 += KC) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int h = h0 + lc + j;
      int t = t0 + lr, e = e0 + lr;
      xs[lc + j][lr] = (t < T && h < h_hi) ? ld_act<XT>(x, (size_t)t * H + h) : 0.f;
      ws[lc + j][lr] = (e < E && h < h_hi) ? Wr[(size_t)e * H + h] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < KC; ++kk) {
      float a0 = xs[kk][ty * 2], a1 = xs[kk][ty * 2 + 1];
      float b0 = ws[kk][tx * 2], b1 = ws[kk][tx * 2 + 1];
      acc[0][0] = fmaf(a0, b0, acc[0][0]);
      acc[0][1] = fmaf(a0, b1, acc[0][1]);
      acc[1][0] = fmaf(a1, b0, acc[1][0]);
      acc[1][1] = fmaf(a1, b1, acc[1][1]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      int t = t0 + ty * 2 + i, e = e0 + tx * 2 + j;
      if (t < T && e < E) partial[((size_t)ks * T + t) * E + e] = acc[i][j];
    }
}

template <int NV>
__global__ void __launch_bounds__(128) k_route_topk(const float* __restrict__ partial, int ksplit,
                                                    const float* __restrict__ b_logit,
                                                    const float* __restrict__ scores_in,
                                                    const float* __restrict__ corr_bias, float* __restrict__ scores_out,
                                                    int32_t* __restrict__ idx, float* __restrict__ gate, int T, int E, int k,
                                                    int n_group, int topk_group, int score_fn, int norm_topk) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t >= T) return;
  float s[NV], sp[NV];
  if (scores_in) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int e = lane + 32 * i;
      s[i] = e < E ? scores_in[(size_t)t * E + e] : 0.f;
    }
  } else {
    float l[NV];
    float mx = -INFINITY;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int e = lane + 32 * i;
      float a = 0.f;
      if (e < E) {
        for (int ks = 0; ks < ksplit; ++ks) a += partial[((size_t)ks * T + t) * E + e];
        if (b_logit) a += b_logit[e];
        mx = fmaxf(mx, a);
      }
      l[i] = a;
    }
    if (score_fn == CAEE_SCORE_SIGMOID) {
#pragma unroll
      for (int i = 0; i < NV; ++i) s[i] = 1.0f / (1.0f + expf(-l[i]));
    } else {
#pragma unroll
      for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
      float den = 0.f;
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        int e = lane + 32 * i;
        s[i] = e < E ? expf(l[i] - mx) : 0.f;
        den += s[i];
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) den += __shfl_xor_sync(0xffffffffu, den, o);
#pragma unroll
      for (int i = 0; i < NV; ++i) s[i] = s[i] / den;
    }
  }
  if (scores_out) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int e = lane + 32 * i;
      if (e < E) scores_out[(size_t)t * E + e] = s[i];
    }
  }
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int e = lane + 32 * i;
    sp[i] = (corr_bias && e < E) ? __fadd_rn(s[i], corr_bias[e]) : s[i];
  }
  uint32_t ok = 0;
#pragma unroll
  for (int i = 0; i < NV; ++i)
    if (lane + 32 * i < E) ok |= 1u << i;
  if (n_group > 1 && topk_group < n_group) ok &= caee_group_mask<NV>(sp, ok, E, n_group, topk_group, lane);
  caee_warp_select<NV>(s, sp, ok, k, norm_topk, lane, idx + (size_t)t * k, gate + (size_t)t * k);
}

template <int NV>
void launch_topk(caee_ctx* c, const float* scores_in, int ksplit, int T, float* scores_out, int32_t* idx, float* gate,
                 cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  k_route_topk<NV><<<caee_ceil_div(T, 4), 128, 0, st>>>(c->partial, ksplit, c->b_logit, scores_in, c->corr_bias,
                                                         scores_out, idx, gate, T, d.E, d.k, d.n_group, d.topk_group,
                                                         d.score_fn, d.norm_topk);
}

}  // namespace

int caee_router_ksplit(const caee_ctx* c, int T) {
  const caee_layer_desc& d = c->d;
  int tiles = caee_ceil_div(d.E, TE) * caee_ceil_div(T, TT);
  int want = caee_ceil_div(2 * c->num_sms, tiles);
  int maxk = d.H / 256 > 0 ? d.H / 256 : 1;
  int ks = want < 1 ? 1 : (want > maxk ? maxk : want);
  return ks > c->ksplit_max ? c->ksplit_max : ks;
}

void caee_launch_router_logits(caee_ctx* c, const void* x, int T, int ksplit, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  int Hs = caee_ceil_div(caee_ceil_div(d.H, ksplit), KC) * KC;
  dim3 grid(caee_ceil_div(d.E, TE), caee_ceil_div(T, TT), ksplit);
  if (d.act_dtype == CAEE_F32)
    k_router_logits<float><<<grid, 256, 0, st>>>((const float*)x, c->Wr, c->partial, T, d.H, d.E, Hs);
  else
    k_router_logits<__nv_bfloat16><<<grid, 256, 0, st>>>((const __nv_bfloat16*)x, c->Wr, c->partial, T, d.H, d.E, Hs);
}

void caee_launch_route_topk(caee_ctx* c, const float* scores_in, int ksplit, int T, float* scores_out, int32_t* idx,
                            float* gate, cudaStream_t st) {
  int nv = caee_ceil_div(c->d.E, 32);
  if (nv <= 1) launch_topk<1>(c, scores_in, ksplit, T, scores_out, idx, gate, st);
  else if (nv <= 2) launch_topk<2>(c, scores_in, ksplit, T, scores_out, idx, gate, st);
  else if (nv <= 4) launch_topk<4>(c, scores_in, ksplit, T, scores_out, idx, gate, st);
  else if (nv <= 8) launch_topk<8>(c, scores_in, ksplit, T, scores_out, idx, gate, st);
  else launch_topk<16>(c, scores_in, ksplit, T, scores_out, idx, gate, st);
}
