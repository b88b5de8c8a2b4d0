// router.cu — S0 router scores and S1 group-limited top-k + gates (router
// form per DESIGN.md reading R1).  Plain fp32 ALUs: E <= 512 and the GEMV is a few MB.
//
//  k_router_logits : split-K partial logits  partial[ks][t][e] = sum_{h in chunk ks} x[t,h] W_r[e,h],
//                    reduced in ascending ks by the last CTA of each tile (deterministic scores)
//  k_route_topk    : one warp per token: activation, selection, gates (steps > 256 tokens and
//                    caee_route; decode-size steps run the same code inside k_decide, decide.cu).
#include "caee_internal.cuh"
#include "warp_select.cuh"

namespace {

constexpr int TE = 64, KC = 32, WS = TE + 4;   // expert tile, k chunk, padded smem row (keeps 16 B alignment)

template <typename XT>
__device__ __forceinline__ float4 ld_act4(const XT* p);
template <>
__device__ __forceinline__ float4 ld_act4<float>(const float* p) { return *reinterpret_cast<const float4*>(p); }
template <>
__device__ __forceinline__ float4 ld_act4<__nv_bfloat16>(const __nv_bfloat16* p) {
  const uint2 u = *reinterpret_cast<const uint2*>(p);
  return make_float4(__uint_as_float(u.x << 16), __uint_as_float(u.x & 0xffff0000u), __uint_as_float(u.y << 16),
                     __uint_as_float(u.y & 0xffff0000u));
}

// Split-K router GEMM  logit[t,e] = sum_h x[t,h] W_r[e,h]  (S0).
// Grid (E/64, T/TT, ksplit); CTA tile 64 experts x TT tokens, thread tile 4 x TT/16, fp32 FMAs in
// ascending h.  Each CTA writes its partial tile; the LAST CTA of a tile to finish (ticket
// counter) adds the ksplit partials in ascending ks and writes the logits, so the result
// does not depend on which CTA came last: scores are deterministic.
template <typename XT, int TT>
__global__ void __launch_bounds__(256) k_router_logits(const XT* __restrict__ x, const float* __restrict__ Wr,
                                                       float* __restrict__ partial, float* __restrict__ logits,
                                                       int* __restrict__ tile_ctr, int T, int H, int E, int Hs) {
  constexpr int TPT = TT / 16, XS = TT + 4;
  __shared__ __align__(16) float ws[KC][WS];
  __shared__ __align__(16) float xs[KC][XS];
  __shared__ int last_s;
  const int e0 = blockIdx.x * TE, t0 = blockIdx.y * TT, ks = blockIdx.z, ksplit = gridDim.z;
  const int h_lo = ks * Hs, h_hi = min(H, h_lo + Hs);
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  float acc[TPT][4];
#pragma unroll
  for (int i = 0; i < TPT; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  // loaders: W tile = 64 rows x 32 k = 512 float4 (2 per thread); x tile = TT rows x 32 k = TT*8 float4
  float4 wreg[2], xreg;
  auto load_tiles = [&](int h0) {
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const int i = tid + 256 * q, r = i >> 3, kq = (i & 7) * 4;
      const int e = e0 + r, h = h0 + kq;
      wreg[q] = (e < E && h < h_hi) ? *reinterpret_cast<const float4*>(Wr + (size_t)e * H + h) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (tid < TT * 8) {
      const int r = tid >> 3, kq = (tid & 7) * 4;
      const int t = t0 + r, h = h0 + kq;
      xreg = (t < T && h < h_hi) ? ld_act4<XT>(x + (size_t)t * H + h) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
  };
  auto store_tiles = [&]() {
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const int i = tid + 256 * q, r = i >> 3, kq = (i & 7) * 4;
      ws[kq][r] = wreg[q].x; ws[kq + 1][r] = wreg[q].y; ws[kq + 2][r] = wreg[q].z; ws[kq + 3][r] = wreg[q].w;
    }
    if (tid < TT * 8) {
      const int r = tid >> 3, kq = (tid & 7) * 4;
      xs[kq][r] = xreg.x; xs[kq + 1][r] = xreg.y; xs[kq + 2][r] = xreg.z; xs[kq + 3][r] = xreg.w;
    }
  };
  load_tiles(h_lo);
  for (int h0 = h_lo; h0 < h_hi; h0 += KC) {
    store_tiles();
    __syncthreads();
    if (h0 + KC < h_hi) load_tiles(h0 + KC);   // next chunk's global loads overlap this chunk's FMAs
#pragma unroll
    for (int kk = 0; kk < KC; ++kk) {
      const float4 w = *reinterpret_cast<const float4*>(&ws[kk][tx * 4]);
      float xv[TPT];
#pragma unroll
      for (int i = 0; i < TPT; ++i) xv[i] = xs[kk][ty * TPT + i];
#pragma unroll
      for (int i = 0; i < TPT; ++i) {
        acc[i][0] = fmaf(xv[i], w.x, acc[i][0]);
        acc[i][1] = fmaf(xv[i], w.y, acc[i][1]);
        acc[i][2] = fmaf(xv[i], w.z, acc[i][2]);
        acc[i][3] = fmaf(xv[i], w.w, acc[i][3]);
      }
    }
    __syncthreads();
  }
  float* out = ksplit == 1 ? logits : partial + (size_t)ks * T * E;
#pragma unroll
  for (int i = 0; i < TPT; ++i) {
    const int t = t0 + ty * TPT + i;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int e = e0 + tx * 4 + j;
      if (t < T && e < E) out[(size_t)t * E + e] = acc[i][j];
    }
  }
  if (ksplit == 1) return;
  // tile ticket: the last CTA to arrive reduces the tile (threadFenceReduction pattern)
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    int* ctr = tile_ctr + blockIdx.y * gridDim.x + blockIdx.x;
    const int prev = atomicAdd(ctr, 1);
    last_s = prev == ksplit - 1;
    if (last_s) *ctr = 0;   // ready for the next step
  }
  __syncthreads();
  if (!last_s) return;
  __threadfence();
  const int nt = min(TT, T - t0);
  for (int i = tid; i < nt * (TE / 4); i += 256) {
    const int t = t0 + i / (TE / 4), e = e0 + (i % (TE / 4)) * 4;
    if ((E & 3) == 0 && e + 3 < E) {
      float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
      for (int s = 0; s < ksplit; ++s) {
        const float4 v = __ldcg(reinterpret_cast<const float4*>(partial + ((size_t)s * T + t) * E + e));
        a.x += v.x; a.y += v.y; a.z += v.z; a.w += v.w;
      }
      *reinterpret_cast<float4*>(logits + (size_t)t * E + e) = a;
    } else {
      for (int j = 0; j < 4 && e + j < E; ++j) {
        float a = 0.f;
        for (int s = 0; s < ksplit; ++s) a += __ldcg(partial + ((size_t)s * T + t) * E + e + j);
        logits[(size_t)t * E + e + j] = a;
      }
    }
  }
}

template <int NV>
__global__ void __launch_bounds__(128) k_route_topk(const float* __restrict__ logits, const float* __restrict__ b_logit,
                                                    const float* __restrict__ scores_in,
                                                    const float* __restrict__ corr_bias, float* __restrict__ scores_out,
                                                    int32_t* __restrict__ idx, float* __restrict__ gate, int T, int E, int k,
                                                    int n_group, int topk_group, int score_fn, int norm_topk) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t >= T) return;
  float s[NV], bl[NV], cb[NV];
  caee_load_vec<NV>(b_logit, E, lane, bl);
  caee_load_vec<NV>(corr_bias, E, lane, cb);
  caee_token_scores<NV>(scores_in ? scores_in + (size_t)t * E : nullptr, logits ? logits + (size_t)t * E : nullptr,
                        b_logit != nullptr, bl, E, score_fn, lane, s);
  if (scores_out) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int e = lane + 32 * i;
      if (e < E) scores_out[(size_t)t * E + e] = s[i];
    }
  }
  caee_route_token<NV>(s, corr_bias != nullptr, cb, E, k, n_group, topk_group, norm_topk, lane, idx + (size_t)t * k, gate + (size_t)t * k);
}

template <int NV>
void launch_topk(caee_ctx* c, const float* scores_in, int T, float* scores_out, int32_t* idx, float* gate, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  k_route_topk<NV><<<caee_ceil_div(T, 4), 128, 0, st>>>(c->logits, c->b_logit, scores_in, c->corr_bias, scores_out, idx, gate,
                                                         T, d.E, d.k, d.n_group, d.topk_group, d.score_fn, d.norm_topk);
}

template <typename XT>
void launch_logits(caee_ctx* c, const XT* x, int T, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  int tt, ks;
  caee_router_shape(c, T, &tt, &ks);
  const int Hs = caee_ceil_div(caee_ceil_div(d.H, ks), KC) * KC;
  dim3 grid(caee_ceil_div(d.E, TE), caee_ceil_div(T, tt), ks);
  if (tt == 16) k_router_logits<XT, 16><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, c->logits, c->tile_ctr, T, d.H, d.E, Hs);
  else k_router_logits<XT, 32><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, c->logits, c->tile_ctr, T, d.H, d.E, Hs);
}

}  // namespace

// Token tile and split-K factor for a T-token step: about two CTAs per SM, K chunks >= 128.
void caee_router_shape(const caee_ctx* c, int T, int* tt, int* ksplit) {
  const caee_layer_desc& d = c->d;
  *tt = T <= 16 ? 16 : 32;
  const int tiles = caee_ceil_div(d.E, TE) * caee_ceil_div(T, *tt);
  const int want = caee_ceil_div(2 * c->num_sms, tiles);
  const int maxk = d.H / 128 > 0 ? d.H / 128 : 1;
  *ksplit = want < 1 ? 1 : (want > maxk ? maxk : want);
}

void caee_launch_router_logits(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  if (c->d.act_dtype == CAEE_F32) launch_logits<float>(c, (const float*)x, T, st);
  else launch_logits<__nv_bfloat16>(c, (const __nv_bfloat16*)x, T, st);
}

void caee_launch_route_topk(caee_ctx* c, const float* scores_in, int T, float* scores_out, int32_t* idx, float* gate,
                            cudaStream_t st) {
  int nv = caee_ceil_div(c->d.E, 32);
  if (nv <= 1) launch_topk<1>(c, scores_in, T, scores_out, idx, gate, st);
  else if (nv <= 2) launch_topk<2>(c, scores_in, T, scores_out, idx, gate, st);
  else if (nv <= 4) launch_topk<4>(c, scores_in, T, scores_out, idx, gate, st);
  else if (nv <= 8) launch_topk<8>(c, scores_in, T, scores_out, idx, gate, st);
  else launch_topk<16>(c, scores_in, T, scores_out, idx, gate, st);
}
