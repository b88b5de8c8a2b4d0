// router.cu — S0 router scores and S1 group-limited top-k + gates (router
// form per DESIGN.md reading R1).  Plain fp32 ALUs: E <= 512 and the GEMV is a few MB.
//
//  k_router_logits : split-K partial logits  partial[ks][t][e] = sum_{h in chunk ks} x[t,h] W_r[e,h];
//                    the consumer (caee_token_scores, warp_select.cuh) adds the partials of its token
//                    in ascending ks: deterministic scores, no reduction tail in this kernel
//  k_route_topk    : one warp per token: activation, selection, gates (steps > 256 tokens and
//                    caee_route; decode-size steps run the same code inside k_decide, decide.cu).
#include <cstring>
#include <mutex>

#include "caee_internal.cuh"
#include "warp_select.cuh"

namespace {

constexpr int TE = 64, KC = 32;          // expert tile, k elements per pipeline stage
constexpr int WROW = KC * 4 + 16;        // bytes of one W row in shared memory (16 B pad: conflict-free LDS.128)

template <typename XT> struct XTraits;
template <> struct XTraits<float> {
  static constexpr int kRow = KC * 4 + 16, kChunks = KC / 4, kStages = 3;
  static __device__ __forceinline__ void ld4(const uint8_t* p, float (&v)[4]) {
    const float4 f = *reinterpret_cast<const float4*>(p);
    v[0] = f.x; v[1] = f.y; v[2] = f.z; v[3] = f.w;
  }
};
template <> struct XTraits<__nv_bfloat16> {
  static constexpr int kRow = KC * 2 + 16, kChunks = KC / 8, kStages = 4;
  static __device__ __forceinline__ void ld4(const uint8_t* p, float (&v)[4]) {
    const uint2 u = *reinterpret_cast<const uint2*>(p);
    v[0] = __uint_as_float(u.x << 16); v[1] = __uint_as_float(u.x & 0xffff0000u);
    v[2] = __uint_as_float(u.y << 16); v[3] = __uint_as_float(u.y & 0xffff0000u);
  }
};

__device__ __forceinline__ void cp_async16(void* dst, const void* src, bool valid) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst);
  const uint32_t n = valid ? 16u : 0u;   // src-size 0: zero fill
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(n) : "memory");
}

// Split-K router GEMM  logit[t,e] = sum_h x[t,h] W_r[e,h]  (S0).
// Grid (E/64, T/TT, ksplit); CTA tile 64 experts x TT tokens, thread tile 4 x TT/16, fp32 FMAs in
// ascending h.  W_r and x tiles stream through a cp.async ring (3-4 stages in flight).  Each CTA
// writes its partial tile and is done.
template <typename XT, int TT>
__global__ void __launch_bounds__(256) k_router_logits(const XT* __restrict__ x, const float* __restrict__ Wr,
                                                       float* __restrict__ partial, int T, int H, int E, int Hs) {
  using XR = XTraits<XT>;
  constexpr int TPT = TT / 16, NS = TT >= 64 ? (sizeof(XT) == 4 ? 2 : 3) : XR::kStages;   // static shared memory stays below 48 KB
  constexpr int kStageBytes = TE * WROW + TT * XR::kRow;
  __shared__ __align__(16) uint8_t ring[NS * kStageBytes];
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the decision kernel may set itself up (it waits for this grid)
  const int e0 = blockIdx.x * TE, t0 = blockIdx.y * TT, ks = blockIdx.z;
  const int h_lo = ks * Hs, h_hi = min(H, h_lo + Hs);
  const int n_it = h_hi > h_lo ? (h_hi - h_lo + KC - 1) / KC : 0;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  float acc[TPT][4];
#pragma unroll
  for (int i = 0; i < TPT; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  auto issue = [&](int it) {
    if (it < n_it) {
      uint8_t* st = ring + (it % NS) * kStageBytes;
      const int h0 = h_lo + it * KC;
#pragma unroll
      for (int q = 0; q < 2; ++q) {   // W tile: 64 rows x 8 chunks of 4 floats
        const int i = tid + 256 * q, r = i >> 3, c = i & 7;
        const int e = e0 + r, h = h0 + c * 4;
        const bool ok = e < E && h < h_hi;
        cp_async16(st + r * WROW + c * 16, ok ? Wr + (size_t)e * H + h : Wr, ok);
      }
      if (tid < TT * XR::kChunks) {   // x tile: TT rows x kChunks chunks of 16 bytes
        const int r = tid / XR::kChunks, c = tid % XR::kChunks;
        const int t = t0 + r, h = h0 + c * (16 / (int)sizeof(XT));
        const bool ok = t < T && h < h_hi;
        cp_async16(st + TE * WROW + r * XR::kRow + c * 16, ok ? x + (size_t)t * H + h : x, ok);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
#pragma unroll
  for (int s = 0; s < NS - 1; ++s) issue(s);
  for (int it = 0; it < n_it; ++it) {
    asm volatile("cp.async.wait_group %0;" ::"n"(NS - 2) : "memory");
    __syncthreads();
    issue(it + NS - 1);   // refills the slot consumed in iteration it - 1
    const uint8_t* st = ring + (it % NS) * kStageBytes;
    const uint8_t* wrow = st + tx * WROW;
    const uint8_t* xrow = st + TE * WROW + (ty * TPT) * XR::kRow;
#pragma unroll
    for (int k4 = 0; k4 < KC / 4; ++k4) {
      float4 w[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) w[j] = *reinterpret_cast<const float4*>(wrow + j * 16 * WROW + k4 * 16);
#pragma unroll
      for (int i = 0; i < TPT; ++i) {
        float xv[4];
        XR::ld4(xrow + i * XR::kRow + k4 * 4 * (int)sizeof(XT), xv);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          acc[i][j] = fmaf(xv[0], w[j].x, acc[i][j]);
          acc[i][j] = fmaf(xv[1], w[j].y, acc[i][j]);
          acc[i][j] = fmaf(xv[2], w[j].z, acc[i][j]);
          acc[i][j] = fmaf(xv[3], w[j].w, acc[i][j]);
        }
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  // thread (tx, ty) holds experts e0 + tx + 16 j, tokens t0 + ty*TPT + i
  float* out = partial + (size_t)ks * T * E;
#pragma unroll
  for (int i = 0; i < TPT; ++i) {
    const int t = t0 + ty * TPT + i;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int e = e0 + tx + 16 * j;
      if (t < T && e < E) out[(size_t)t * E + e] = acc[i][j];
    }
  }
}

// The same partial logits for steps of at most 4 tokens, where the tile kernel above would spend its
// time on padding tokens: a bandwidth-shaped GEMV.  CTA tile 16 experts x TT tokens; a stage holds 128
// k of the 16 rows (8 KB, cp.async ring); thread (tx = expert, ty = one of 16 k-octets of the stage)
// multiplies its 8 k in ascending order; the 16 octet sums of an output are added in ascending ty
// through shared memory at the end (a fixed order).  Grid (E/16, ksplit): about one CTA per SM, and
// only ~8 partials for the decision kernel to add.
constexpr int SE = 16, SKC = 128, SWROW = SKC * 4 + 16, SNS = 4;
template <typename XT, int TT>
__global__ void __launch_bounds__(256) k_router_small(const XT* __restrict__ x, const float* __restrict__ Wr,
                                                      float* __restrict__ partial, int T, int H, int E, int Hs) {
  constexpr int kXRow = SKC * (int)sizeof(XT) + 16;
  constexpr int kStageBytes = SE * SWROW + TT * kXRow;
  __shared__ __align__(16) uint8_t ring[SNS * kStageBytes];
  __shared__ float red[16][TT][SE + 1];
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the decision kernel may set itself up (it waits for this grid)
  const int e0 = blockIdx.x * SE, ks = blockIdx.y;
  const int h_lo = ks * Hs, h_hi = min(H, h_lo + Hs);
  const int n_it = h_hi > h_lo ? (h_hi - h_lo + SKC - 1) / SKC : 0;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  float acc[TT];
#pragma unroll
  for (int t = 0; t < TT; ++t) acc[t] = 0.f;
  auto issue = [&](int it) {
    if (it < n_it) {
      uint8_t* st = ring + (it % SNS) * kStageBytes;
      const int h0 = h_lo + it * SKC;
#pragma unroll
      for (int q = 0; q < 2; ++q) {   // W tile: 16 rows x 32 chunks of 4 floats
        const int i = tid + 256 * q, r = i >> 5, c = i & 31;
        const int e = e0 + r, h = h0 + c * 4;
        const bool ok = e < E && h < h_hi;
        cp_async16(st + r * SWROW + c * 16, ok ? Wr + (size_t)e * H + h : Wr, ok);
      }
      constexpr int kXChunks = SKC * (int)sizeof(XT) / 16;
      if (tid < TT * kXChunks) {      // x tile: TT rows of 128 k
        const int r = tid / kXChunks, c = tid % kXChunks;
        const int t = r, h = h0 + c * (16 / (int)sizeof(XT));
        const bool ok = t < T && h < h_hi;
        cp_async16(st + SE * SWROW + r * kXRow + c * 16, ok ? x + (size_t)t * H + h : x, ok);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
#pragma unroll
  for (int s = 0; s < SNS - 1; ++s) issue(s);
  for (int it = 0; it < n_it; ++it) {
    asm volatile("cp.async.wait_group %0;" ::"n"(SNS - 2) : "memory");
    __syncthreads();
    issue(it + SNS - 1);
    const uint8_t* st = ring + (it % SNS) * kStageBytes;
    const float4 w0 = *reinterpret_cast<const float4*>(st + tx * SWROW + ty * 32);
    const float4 w1 = *reinterpret_cast<const float4*>(st + tx * SWROW + ty * 32 + 16);
#pragma unroll
    for (int t = 0; t < TT; ++t) {
      float xv[4], xw[4];
      const uint8_t* xr = st + SE * SWROW + t * kXRow + ty * 8 * (int)sizeof(XT);
      XTraits<XT>::ld4(xr, xv);
      XTraits<XT>::ld4(xr + 4 * (int)sizeof(XT), xw);
      float a = acc[t];
      a = fmaf(xv[0], w0.x, a); a = fmaf(xv[1], w0.y, a); a = fmaf(xv[2], w0.z, a); a = fmaf(xv[3], w0.w, a);
      a = fmaf(xw[0], w1.x, a); a = fmaf(xw[1], w1.y, a); a = fmaf(xw[2], w1.z, a); a = fmaf(xw[3], w1.w, a);
      acc[t] = a;
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
  for (int t = 0; t < TT; ++t) red[ty][t][tx] = acc[t];
  __syncthreads();
  if (tid < TT * SE) {
    const int t = tid / SE, e = tid % SE;
    float a = red[0][t][e];
#pragma unroll
    for (int q = 1; q < 16; ++q) a += red[q][t][e];
    if (t < T && e0 + e < E) partial[((size_t)ks * T + t) * E + e0 + e] = a;
  }
}

template <int NV>
__global__ void __launch_bounds__(128) k_route_topk(const float* __restrict__ logits, int n_part, const float* __restrict__ b_logit,
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
                        n_part, (size_t)T * E, b_logit != nullptr, bl, E, score_fn, lane, s);
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
  int tt, ks;
  caee_router_shape(c, T, &tt, &ks, nullptr);
  k_route_topk<NV><<<caee_ceil_div(T, 4), 128, 0, st>>>(c->partial, ks, c->b_logit, scores_in, c->corr_bias, scores_out, idx, gate,
                                                         T, d.E, d.k, d.n_group, d.topk_group, d.score_fn, d.norm_topk);
}

template <typename XT>
void launch_logits(caee_ctx* c, const XT* x, int T, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  int tt, ks, Hs;
  ++c->n_launches;
  caee_router_shape(c, T, &tt, &ks, &Hs);
  if (tt <= 4) {
    dim3 grid(caee_ceil_div(d.E, SE), ks);
    if (tt == 1) k_router_small<XT, 1><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, T, d.H, d.E, Hs);
    else if (tt == 2) k_router_small<XT, 2><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, T, d.H, d.E, Hs);
    else k_router_small<XT, 4><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, T, d.H, d.E, Hs);
    return;
  }
  dim3 grid(caee_ceil_div(d.E, TE), caee_ceil_div(T, tt), ks);
  if (tt == 16) k_router_logits<XT, 16><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, T, d.H, d.E, Hs);
  else if (tt == 64) k_router_logits<XT, 64><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, T, d.H, d.E, Hs);
  else k_router_logits<XT, 32><<<grid, 256, 0, st>>>(x, c->Wr, c->partial, T, d.H, d.E, Hs);
}

}  // namespace

// Token tile and split-K factor for a T-token step: about one CTA per SM for decode-size steps (every
// partial is read back by the step's decision kernel), two for larger ones; K chunks >= 128.  The
// split actually used is the number of non-empty chunks of Hs = ceil(H / ksplit) rounded up to the
// stage depth.  Steps of at most 4 tokens take the GEMV-shaped kernel (token tile 1, 2 or 4).
void caee_router_shape(const caee_ctx* c, int T, int* tt, int* ksplit, int* hs) {
  const caee_layer_desc& d = c->d;
  if (caee_router_uses_mma(c, T)) {   // prefill-size steps: tensor-core router (router_mma.cu), 128-token tiles
    int sps;
    caee_router_mma_shape(c, T, ksplit, &sps);
    *tt = 128;
    if (hs) *hs = sps * 64;
    return;
  }
  const bool small = T <= 4;
  *tt = small ? (T <= 1 ? 1 : (T <= 2 ? 2 : 4)) : (T <= 16 ? 16 : (T >= 1024 ? 64 : 32));   // prefill-size steps: 4 x 4 outputs per thread
  const int tiles = small ? caee_ceil_div(d.E, SE) : caee_ceil_div(d.E, TE) * caee_ceil_div(T, *tt);
  const int want = caee_ceil_div((small ? c->router_small_waves : (T <= 256 ? 1 : 2)) * c->num_sms, tiles);
  const int maxk = d.H / 128 > 0 ? d.H / 128 : 1;
  int ks = want < 1 ? 1 : (want > maxk ? maxk : want);
  const int kc = small ? SKC : KC;
  const int Hs = caee_ceil_div(caee_ceil_div(d.H, ks), kc) * kc;
  *ksplit = caee_ceil_div(d.H, Hs);
  if (hs) *hs = Hs;
}

caee_status caee_launch_router_logits(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  if (caee_router_uses_mma(c, T)) return caee_launch_router_mma(c, x, T, st);
  if (c->d.act_dtype == CAEE_F32) launch_logits<float>(c, (const float*)x, T, st);
  else launch_logits<__nv_bfloat16>(c, (const __nv_bfloat16*)x, T, st);
  return CAEE_OK;
}

void caee_launch_route_topk(caee_ctx* c, const float* scores_in, int T, float* scores_out, int32_t* idx, float* gate,
                            cudaStream_t st) {
  ++c->n_launches;
  int nv = caee_ceil_div(c->d.E, 32);
  if (nv <= 1) launch_topk<1>(c, scores_in, T, scores_out, idx, gate, st);
  else if (nv <= 2) launch_topk<2>(c, scores_in, T, scores_out, idx, gate, st);
  else if (nv <= 4) launch_topk<4>(c, scores_in, T, scores_out, idx, gate, st);
  else if (nv <= 8) launch_topk<8>(c, scores_in, T, scores_out, idx, gate, st);
  else launch_topk<16>(c, scores_in, T, scores_out, idx, gate, st);
}

// ------------------------------------------------------------------ caee_route_noalloc (include/caee.h)
// The split-K scratch of the router GEMM for callers that cannot allocate: one file-scope device array per GPU that
// loads the library.  In HOST code the name below is a host-side stand-in, not a device address: its device address
// is taken once per device with cudaGetSymbolAddress (that device current) and passed to the kernels as `partial`.
static __device__ __align__(256) float g_route_noalloc_partial[CAEE_ROUTE_NOALLOC_SCRATCH_FLOATS];

namespace {

constexpr int kNoAllocMaxDevices = 64;
struct NoAllocDevice {
  float* partial = nullptr;   // device address of g_route_noalloc_partial on this device
  int num_sms = 0;
  bool ready = false;
};
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];
std::mutex g_noalloc_mu;

struct CurrentDevice {   // makes `dev` current for the scope
  int prev = -1;
  explicit CurrentDevice(int dev) {
    cudaGetDevice(&prev);
    if (prev != dev) cudaSetDevice(dev);
    else prev = -1;
  }
  ~CurrentDevice() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

// set-up, once per device, with that device current; no allocation (the array came with the module)
caee_status noalloc_device(int dev, NoAllocDevice* out) {
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  NoAllocDevice& nd = g_noalloc_dev[dev];
  if (!nd.ready) {
    int major = 0, sms = 0;
    CAEE_CUDA(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return caee_fail(nullptr, CAEE_EUNSUPPORTED, "caee_route_noalloc: device %d is not an sm_100 device", dev);
    CAEE_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* ptr = nullptr;
    CAEE_CUDA(nullptr, cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_route_noalloc_partial));
    if (!ptr) return caee_fail(nullptr, CAEE_ECUDA, "caee_route_noalloc: cudaGetSymbolAddress returned NULL");
    nd.partial = ptr;
    nd.num_sms = sms;
    nd.ready = true;
  }
  *out = nd;
  return CAEE_OK;
}

}  // namespace

caee_status caee_route_noalloc(int32_t device, const void* x, int32_t act_dtype, const float* Wr, const float* b_logit,
                               const float* corr_bias, int32_t T, int32_t H, int32_t E, int32_t k, int32_t n_group,
                               int32_t topk_group, int32_t score_fn, int32_t norm_topk, float* scores, int32_t* idx,
                               float* gate, void* stream) {
  const char* me = "caee_route_noalloc";
  if (H < 8 || H % 8) return caee_fail(nullptr, CAEE_ESHAPE, "%s: H must be a positive multiple of 8", me);
  if (E < 1 || E > CAEE_MAX_E) return caee_fail(nullptr, CAEE_EINVAL, "%s: E must be in 1..%d", me, CAEE_MAX_E);
  if (k < 1 || k > E || k > 32) return caee_fail(nullptr, CAEE_EINVAL, "%s: k must be in 1..min(E,32)", me);
  if (n_group < 1 || n_group > 32 || E % n_group) return caee_fail(nullptr, CAEE_EINVAL, "%s: n_group must divide E and be <= 32", me);
  if (topk_group < 1 || topk_group > n_group) return caee_fail(nullptr, CAEE_EINVAL, "%s: topk_group must be in 1..n_group", me);
  if ((long long)topk_group * (E / n_group) < k) return caee_fail(nullptr, CAEE_EINVAL, "%s: topk_group*(E/n_group) < k", me);
  if (score_fn != CAEE_SCORE_SOFTMAX && score_fn != CAEE_SCORE_SIGMOID) return caee_fail(nullptr, CAEE_EINVAL, "%s: unknown score_fn", me);
  if (act_dtype != CAEE_F32 && act_dtype != CAEE_BF16) return caee_fail(nullptr, CAEE_EDTYPE, "%s: act_dtype must be F32 or BF16", me);
  if (T < 0) return caee_fail(nullptr, CAEE_EINVAL, "%s: T is negative", me);
  if (T > CAEE_ROUTE_NOALLOC_MAX_TOKENS)
    return caee_fail(nullptr, CAEE_ESHAPE, "%s: T=%d exceeds the no-allocation limit of %d tokens", me, T, CAEE_ROUTE_NOALLOC_MAX_TOKENS);
  if (T == 0) return CAEE_OK;
  if (!x || !Wr || !idx || !gate) return caee_fail(nullptr, CAEE_EINVAL, "%s: x, Wr, idx or gate is NULL", me);
  if (((uintptr_t)x | (uintptr_t)Wr) & 15) return caee_fail(nullptr, CAEE_EINVAL, "%s: x and Wr must be 16-byte aligned", me);
  int dev = device;
  if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return caee_fail(nullptr, CAEE_ECUDA, "%s: no current device", me);
  if (dev < 0 || dev >= kNoAllocMaxDevices) return caee_fail(nullptr, CAEE_EINVAL, "%s: device %d out of range", me, dev);
  CurrentDevice cur(dev);
  NoAllocDevice nd;
  caee_status rc = noalloc_device(dev, &nd);
  if (rc != CAEE_OK) return rc;

  // a host-only stand-in for the context the launchers read their shapes and pointers from (nothing is allocated;
  // wr_img stays NULL, so caee_router_shape picks the FMA kernels at every T)
  caee_ctx view;
  memset(&view.d, 0, sizeof view.d);
  view.d.H = H; view.d.E = E; view.d.k = k; view.d.n_group = n_group; view.d.topk_group = topk_group;
  view.d.score_fn = score_fn; view.d.norm_topk = norm_topk; view.d.act_dtype = act_dtype; view.d.device = dev;
  view.device = dev; view.num_sms = nd.num_sms;
  view.Wr = Wr; view.b_logit = b_logit; view.corr_bias = corr_bias;
  view.partial = nd.partial;
  int tt, ks;
  caee_router_shape(&view, T, &tt, &ks, nullptr);
  const size_t need = (size_t)ks * (size_t)T * (size_t)E;
  if (need > (size_t)CAEE_ROUTE_NOALLOC_SCRATCH_FLOATS)
    return caee_fail(nullptr, CAEE_ESHAPE, "%s: T=%d, E=%d with a %d-way split needs %zu scratch floats, the static array holds %d", me, T,
                     E, ks, need, CAEE_ROUTE_NOALLOC_SCRATCH_FLOATS);
  cudaStream_t st = (cudaStream_t)stream;
  if ((rc = caee_launch_router_logits(&view, x, T, st)) != CAEE_OK) return caee_fail(nullptr, rc, "%s: %s", me, view.err.c_str());
  caee_launch_route_topk(&view, nullptr, T, scores, idx, gate, st);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return caee_fail(nullptr, CAEE_ECUDA, "%s: launch failed: %s", me, cudaGetErrorString(e));
  return CAEE_OK;
}
