// prune.cu — S2 activation set + importance, S3 cost lookup / F_cost, S4 cost-aware pruning
// and S5 compensation.
//
// The pruning decision is batch-global (x_e is per expert) and tiny
// (E <= 512), so one CTA takes it; integers everywhere (importance in units of 2^-40, costs
// in ns ticks) make the result independent of summation order.  Compensation is one warp per
// token again (warp_select.cuh).
#include "caee_internal.cuh"
#include "prune_dev.cuh"
#include "warp_select.cuh"

namespace {

constexpr int PRUNE_THREADS = 512;

struct PartLists {
  const int32_t* experts;   // [E] experts grouped by partition
  const int32_t* start;     // [D+1]
  int fast;                 // largest partition <= 32 experts: one warp per partition (caee_prune_decide_fast)
};

__global__ void __launch_bounds__(PRUNE_THREADS) k_prune(int mode, int flags, double theta, double eps, int T, int E, int k, int D,
                                                         const int32_t* __restrict__ idx, const float* __restrict__ gate,
                                                         const int64_t* __restrict__ w_eff, const int32_t* __restrict__ part,
                                                         const PartLists pl,
                                                         uint8_t* __restrict__ act_o, uint8_t* __restrict__ must_o,
                                                         uint8_t* __restrict__ keep_o, int64_t* __restrict__ I_o,
                                                         int64_t* __restrict__ load_o, int64_t* __restrict__ scalars) {
  __shared__ caee_prune_smem sm;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int e = tid; e < E; e += PRUNE_THREADS) { sm.I[e] = 0; sm.act[e] = 0; sm.must[e] = 0; }
  if (pl.fast) caee_prune_preload(sm, E, D, w_eff, part, pl.experts, pl.start);
  __syncthreads();
  for (int t = warp; t < T; t += PRUNE_THREADS / 32)
    caee_prune_token(mode, flags, theta, k, idx + (size_t)t * k, gate + (size_t)t * k, lane, sm.I, sm.act, sm.must);
  __syncthreads();
  if (pl.fast) caee_prune_decide_fast(sm, mode, flags, theta, eps, E, D, true, act_o, must_o, keep_o, I_o, load_o, scalars);
  else caee_prune_decide(sm, mode, flags, theta, eps, E, D, w_eff, part, true, act_o, must_o, keep_o, I_o, load_o, scalars);
}

// Large steps: S2 and the per-token rules by one warp per token over many CTAs, into the global
// integer accumulators that k_decide also uses (decide_scratch: zero between steps) ...
__global__ void __launch_bounds__(256) k_prune_accum(int mode, int flags, double theta, int T, int k,
                                                     const int32_t* __restrict__ idx, const float* __restrict__ gate,
                                                     unsigned long long* acc_I, unsigned char* acc_act, unsigned char* acc_must) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t < T) caee_prune_token(mode, flags, theta, k, idx + (size_t)t * k, gate + (size_t)t * k, lane, acc_I, acc_act, acc_must);
}

// ... then one CTA takes the batch-global decision from them and zeroes them again.  Integer
// sums and flag bytes: the same masks as the one-CTA k_prune, whatever the order of the atomics.
__global__ void __launch_bounds__(PRUNE_THREADS) k_prune_from_acc(int mode, int flags, double theta, double eps, int E, int D,
                                                                  unsigned long long* acc_I, unsigned char* acc_act,
                                                                  unsigned char* acc_must, const int64_t* __restrict__ w_eff,
                                                                  const int32_t* __restrict__ part, const PartLists pl,
                                                                  uint8_t* __restrict__ act_o,
                                                                  uint8_t* __restrict__ must_o, uint8_t* __restrict__ keep_o,
                                                                  int64_t* __restrict__ I_o, int64_t* __restrict__ load_o,
                                                                  int64_t* __restrict__ scalars) {
  __shared__ caee_prune_smem sm;
  for (int e = threadIdx.x; e < E; e += PRUNE_THREADS) {
    sm.I[e] = __ldcg(acc_I + e); sm.act[e] = __ldcg(acc_act + e); sm.must[e] = __ldcg(acc_must + e);
    acc_I[e] = 0; acc_act[e] = 0; acc_must[e] = 0;
  }
  if (pl.fast) caee_prune_preload(sm, E, D, w_eff, part, pl.experts, pl.start);
  __syncthreads();
  if (pl.fast) caee_prune_decide_fast(sm, mode, flags, theta, eps, E, D, true, act_o, must_o, keep_o, I_o, load_o, scalars);
  else caee_prune_decide(sm, mode, flags, theta, eps, E, D, w_eff, part, true, act_o, must_o, keep_o, I_o, load_o, scalars);
}

template <int NV>
__global__ void __launch_bounds__(128) k_compensate(const float* __restrict__ scores, const float* __restrict__ corr_bias,
                                                    const uint8_t* __restrict__ keep, int flags, int T, int E, int k,
                                                    int norm_topk, int32_t* __restrict__ idx, float* __restrict__ gate) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t >= T) return;
  int32_t* ir = idx + (size_t)t * k;
  bool bad = false;
  if (lane < k) { int e = ir[lane]; bad = e >= 0 && !keep[e]; }
  bool affected = __any_sync(0xffffffffu, bad) || (flags & CAEE_COMP_ALL_TOKENS);
  if (!affected) return;
  float cb[NV];
  caee_load_vec<NV>(corr_bias, E, lane, cb);
  caee_compensate_token<NV>(scores + (size_t)t * E, corr_bias != nullptr, cb, keep, E, k, norm_topk, lane, ir,
                            gate + (size_t)t * k, (flags & CAEE_COMP_RANDOM) != 0, t);
}

}  // namespace

void caee_launch_prune(caee_ctx* c, int mode, int flags, double theta, double eps, int T, const int32_t* idx,
                       const float* gate, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  const PartLists pl = {c->pl_experts, c->pl_start, c->part_max <= 32};
  c->n_launches += T > 512 ? 2 : 1;
  if (T > 512) {
    // the token pass of a prefill-size step takes ~100 us on one CTA: spread it over the GPU
    const size_t E = d.E;
    unsigned long long* acc_I = reinterpret_cast<unsigned long long*>(c->decide_scratch);   // layout: decide.cu
    unsigned char* acc_act = c->decide_scratch + E * 8;
    unsigned char* acc_must = c->decide_scratch + E * 9;
    k_prune_accum<<<caee_ceil_div(T, 8), 256, 0, st>>>(mode, flags, theta, T, d.k, idx, gate, acc_I, acc_act, acc_must);
    k_prune_from_acc<<<1, PRUNE_THREADS, 0, st>>>(mode, flags, theta, eps, d.E, d.D, acc_I, acc_act, acc_must, c->w_eff, c->part, pl, c->act,
                                                  c->must, c->keep, c->I_fix, c->load, c->scalars);
    return;
  }
  k_prune<<<1, PRUNE_THREADS, 0, st>>>(mode, flags, theta, eps, T, d.E, d.k, d.D, idx, gate, c->w_eff, c->part, pl, c->act,
                                       c->must, c->keep, c->I_fix, c->load, c->scalars);
}

void caee_launch_compensate(caee_ctx* c, int flags, const float* scores, int T, int32_t* idx, float* gate,
                            cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  ++c->n_launches;
  int nv = caee_ceil_div(d.E, 32);
  dim3 grid(caee_ceil_div(T, 4));
#define CAEE_COMP(NV) \
  k_compensate<NV><<<grid, 128, 0, st>>>(scores, c->corr_bias, c->keep, flags, T, d.E, d.k, d.norm_topk, idx, gate)
  if (nv <= 1) CAEE_COMP(1);
  else if (nv <= 2) CAEE_COMP(2);
  else if (nv <= 4) CAEE_COMP(4);
  else if (nv <= 8) CAEE_COMP(8);
  else CAEE_COMP(16);
#undef CAEE_COMP
}
