// combine.cu — S8 weighted combine:
//   y_t = routed_scale * sum_{j: K_final(t)_j valid} G(t)_j * o[t, j] + sum_s o[t, k+s]
// The expert kernels leave each (token, slot) output row in o[(t*(k+S) + slot), :] (fp32), so
// the sum runs in list order and y is deterministic.  Also fills caee_fwd_stats.
#include "caee_internal.cuh"
#include "worklist_dev.cuh"

namespace {

template <typename YT> __device__ __forceinline__ void st4(YT* p, float4 v);
template <> __device__ __forceinline__ void st4<float>(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
template <> __device__ __forceinline__ void st4<__nv_bfloat16>(__nv_bfloat16* p, float4 v) {
  __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
  uint2 u = {*reinterpret_cast<uint32_t*>(&a), *reinterpret_cast<uint32_t*>(&b)};
  *reinterpret_cast<uint2*>(p) = u;
}

template <typename YT>
__global__ void __launch_bounds__(256) k_combine(const float* __restrict__ obuf, const int32_t* __restrict__ idx,
                                                 const float* __restrict__ gate, YT* __restrict__ y, int H, int k, int S,
                                                 float routed_scale, int t_lo) {
  // K_final and the gates were complete before the expert kernel started: fetch them while it still runs
  __shared__ int s_idx[32];
  __shared__ float s_gate[32];
  const int t = t_lo + blockIdx.y, c = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (threadIdx.x < k) {
    const int e = idx[(size_t)t * k + threadIdx.x];
    s_idx[threadIdx.x] = e;
    s_gate[threadIdx.x] = e >= 0 ? gate[(size_t)t * k + threadIdx.x] : 0.f;
  }
  __syncthreads();
  asm volatile("griddepcontrol.wait;" ::: "memory");   // programmatic dependent launch: the expert kernel is done
  if (c >= H) return;
  const int KS = k + S;
  float4 acc = {0.f, 0.f, 0.f, 0.f};
  const float* orow = obuf + (size_t)t * KS * H + c;
#pragma unroll 4
  for (int j = 0; j < k; ++j) {
    if (s_idx[j] < 0) continue;            // an empty slot's row was never written
    const float g = s_gate[j];
    const float4 o = *reinterpret_cast<const float4*>(orow + (size_t)j * H);
    acc.x = fmaf(g, o.x, acc.x); acc.y = fmaf(g, o.y, acc.y); acc.z = fmaf(g, o.z, acc.z); acc.w = fmaf(g, o.w, acc.w);
  }
  acc.x *= routed_scale; acc.y *= routed_scale; acc.z *= routed_scale; acc.w *= routed_scale;
  for (int s = 0; s < S; ++s) {
    const float4 o = *reinterpret_cast<const float4*>(obuf + ((size_t)t * KS + k + s) * H + c);
    acc.x += o.x; acc.y += o.y; acc.z += o.z; acc.w += o.w;
  }
  st4<YT>(y + (size_t)t * H + c, acc);
}

__global__ void k_stats(caee_fwd_stats* st, const int64_t* scalars, const int64_t* load, const int32_t* meta, int D, int S,
                        int pruned, long long bytes_per_expert, int n_fetch) {
  caee_stats_fill(st, scalars, load, meta, D, S, pruned, bytes_per_expert, n_fetch, threadIdx.x, blockDim.x);
}

}  // namespace

// tokens [t_lo, t_hi) of the step (t_hi < 0: all T): an expert-parallel device combines its home tokens only
void caee_launch_combine(caee_ctx* c, int T, const int32_t* idx, const float* gate, void* y, cudaStream_t st, int t_lo, int t_hi) {
  const caee_layer_desc& d = c->d;
  if (t_hi < 0) t_hi = T;
  if (T <= 0 || t_hi <= t_lo) return;
  ++c->n_launches;
  dim3 grid(caee_ceil_div(d.H, 1024), t_hi - t_lo);
  if (c->pdl && !c->any_offload && d.act_dtype != CAEE_F32) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(256);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, k_combine<__nv_bfloat16>, (const float*)c->obuf, idx, gate, (__nv_bfloat16*)y, (int)d.H, (int)d.k, (int)d.S,
                       (float)d.routed_scale, t_lo);
    return;
  }
  if (d.act_dtype == CAEE_F32)
    k_combine<float><<<grid, 256, 0, st>>>(c->obuf, idx, gate, (float*)y, d.H, d.k, d.S, d.routed_scale, t_lo);
  else
    k_combine<__nv_bfloat16><<<grid, 256, 0, st>>>(c->obuf, idx, gate, (__nv_bfloat16*)y, d.H, d.k, d.S, d.routed_scale, t_lo);
}

long long caee_expert_bytes(const caee_ctx* c) {
  long long bpe = 3LL * c->d.H * c->d.I * (c->d.w_dtype == CAEE_F32 ? 4 : c->d.w_dtype == CAEE_BF16 ? 2 : 1);
  if (c->d.w_dtype == CAEE_E4M3) bpe += 3LL * ((c->d.H + 127) / 128) * ((c->d.I + 127) / 128) * 4;
  return bpe;
}

void caee_launch_stats(caee_ctx* c, caee_fwd_stats* stats, int pruned, int n_fetch, cudaStream_t st) {
  if (!stats) return;
  ++c->n_launches;
  const long long bpe = caee_expert_bytes(c);
  k_stats<<<1, 64, 0, st>>>(stats, c->scalars, c->load, c->wl.meta, c->d.D, c->d.S, pruned, bpe, n_fetch);
}
