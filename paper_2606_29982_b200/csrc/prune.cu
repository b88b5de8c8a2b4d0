// prune.cu — S2 activation set + importance, S3 cost lookup / F_cost, S4 cost-aware pruning
// and S5 compensation.
//
// The pruning decision is batch-global (x_e is per expert) and tiny
// (E <= 512), so one CTA takes it; integers everywhere (importance in units of 2^-40, costs
// in ns ticks) make the result independent of summation order.  Compensation is one warp per
// token again (warp_select.cuh).
#include "caee_internal.cuh"
#include "warp_select.cuh"

namespace {

constexpr int PRUNE_THREADS = 512;

__global__ void __launch_bounds__(PRUNE_THREADS) k_prune(int mode, int flags, double theta, int T, int E, int k, int D,
                                                         const int32_t* __restrict__ idx, const float* __restrict__ gate,
                                                         const int64_t* __restrict__ w_eff, const int32_t* __restrict__ part,
                                                         uint8_t* __restrict__ act_o, uint8_t* __restrict__ must_o,
                                                         uint8_t* __restrict__ keep_o, int64_t* __restrict__ I_o,
                                                         int64_t* __restrict__ load_o, int64_t* __restrict__ scalars) {
  __shared__ unsigned long long I[CAEE_MAX_E];
  __shared__ long long w[CAEE_MAX_E];
  __shared__ int prt[CAEE_MAX_E];
  __shared__ int sorted[CAEE_MAX_E];
  __shared__ unsigned char act[CAEE_MAX_E], must[CAEE_MAX_E], keep[CAEE_MAX_E];
  __shared__ unsigned long long load[CAEE_MAX_D], load_must[CAEE_MAX_D];
  __shared__ long long F_base_s;
  __shared__ int n_cand_s, cnt[4];
  const int tid = threadIdx.x;
  for (int e = tid; e < E; e += PRUNE_THREADS) {
    I[e] = 0; act[e] = 0; must[e] = 0; keep[e] = 0;
    w[e] = w_eff[e]; prt[e] = part[e];
  }
  for (int d = tid; d < D; d += PRUNE_THREADS) { load[d] = 0; load_must[d] = 0; }
  if (tid < 4) cnt[tid] = 0;
  if (tid == 0) n_cand_s = 0;
  __syncthreads();

  // S2: A_act and I_fix(e) = sum_t floor(G * 2^40)  (exact in fp32: power-of-two scale)
  for (int i = tid; i < T * k; i += PRUNE_THREADS) {
    int e = idx[i];
    if (e >= 0) {
      act[e] = 1;
      atomicAdd(&I[e], (unsigned long long)__float2ll_rz(__fmul_rn(gate[i], CAEE_FIX_ONE_F)));
    }
  }
  // per-token rules of step 1
  if (mode == CAEE_PRUNE_CIR) {
    const float th = (float)theta;
    for (int t = tid; t < T; t += PRUNE_THREADS) {
      const int32_t* ir = idx + (size_t)t * k;
      const float* gr = gate + (size_t)t * k;
      float pk = 0.f;
      for (int j = 0; j < k; ++j)
        if (ir[j] >= 0) pk = __fadd_rn(pk, gr[j]);
      const float rhs = __fmul_rn(th, pk);
      float pm = 0.f;
      for (int j = 0; j < k; ++j) {
        if (ir[j] < 0) break;
        must[ir[j]] = 1;
        pm = __fadd_rn(pm, gr[j]);
        if (pm >= rhs) break;
      }
    }
  } else if (mode == CAEE_PRUNE_RANK) {
    const int b = (int)theta;
    for (int i = tid; i < T * k; i += PRUNE_THREADS) {
      int e = idx[i];
      if (e >= 0 && (i % k) < k - b) must[e] = 1;
    }
  }
  if ((flags & CAEE_KEEP_TOP1) && mode != CAEE_PRUNE_NONE)
    for (int t = tid; t < T; t += PRUNE_THREADS)
      if (idx[(size_t)t * k] >= 0) must[idx[(size_t)t * k]] = 1;
  __syncthreads();

  // per-expert rules of step 1
  for (int e = tid; e < E; e += PRUNE_THREADS) {
    if (!act[e]) continue;
    atomicAdd(&cnt[0], 1);  // |A_act|
    if (mode == CAEE_PRUNE_NONE) must[e] = 1;
    else if (mode == CAEE_PRUNE_THRESH) {
      long long thr = (long long)floor(theta * 1099511627776.0);
      if ((long long)I[e] >= thr) must[e] = 1;
    }
  }
  __syncthreads();
  if (mode == CAEE_PRUNE_FRAC) {
    const long long n_cand = (long long)floor(theta * (double)cnt[0]);
    for (int e = tid; e < E; e += PRUNE_THREADS) {
      if (!act[e]) continue;
      int rank = 0;  // position in ascending (I, id) order among A_act
      for (int f = 0; f < E; ++f)
        if (act[f] && (I[f] < I[e] || (I[f] == I[e] && f < e))) ++rank;
      if (rank >= n_cand) must[e] = 1;
    }
    __syncthreads();
  }

  // step 2: F_base = max_d sum_{e in A_must ∩ E_d} w_e
  for (int e = tid; e < E; e += PRUNE_THREADS) {
    if (must[e]) {
      keep[e] = 1;
      atomicAdd(&cnt[1], 1);
      atomicAdd(&load_must[prt[e]], (unsigned long long)w[e]);
    }
  }
  __syncthreads();
  if (tid == 0) {
    long long m = 0;
    for (int d = 0; d < D; ++d) m = max(m, (long long)load_must[d]);
    F_base_s = m;
  }
  // candidates A_cand = A_act \ A_must ordered by (I desc, id asc)  (R3, R7)
  for (int e = tid; e < E; e += PRUNE_THREADS) {
    if (act[e] && !must[e]) {
      int rank = 0;
      for (int f = 0; f < E; ++f)
        if (act[f] && !must[f] && (I[f] > I[e] || (I[f] == I[e] && f < e))) ++rank;
      sorted[rank] = e;
      atomicAdd(&n_cand_s, 1);
    }
  }
  for (int d = tid; d < D; d += PRUNE_THREADS) load[d] = load_must[d];
  __syncthreads();
  // step 3: cost-invariant expansion; partitions are independent given F_base (R5, R6)
  if (tid < D) {
    const long long Fb = F_base_s;
    long long l = (long long)load[tid];
    const int nc = n_cand_s;
    for (int r = 0; r < nc; ++r) {
      int e = sorted[r];
      if (prt[e] != tid) continue;
      if (l + w[e] <= Fb) { keep[e] = 1; l += w[e]; }
    }
    load[tid] = (unsigned long long)l;
  }
  __syncthreads();

  // step 4 + reporting
  __shared__ unsigned long long dense[CAEE_MAX_D];
  __shared__ unsigned long long F_imp_s;
  for (int d = tid; d < D; d += PRUNE_THREADS) dense[d] = 0;
  if (tid == 0) F_imp_s = 0;
  __syncthreads();
  for (int e = tid; e < E; e += PRUNE_THREADS) {
    if (act[e]) atomicAdd(&dense[prt[e]], (unsigned long long)w[e]);
    if (keep[e]) atomicAdd(&cnt[2], 1);
    if (act[e] && !keep[e]) atomicAdd(&F_imp_s, I[e]);
    act_o[e] = act[e]; must_o[e] = must[e]; keep_o[e] = keep[e]; I_o[e] = (long long)I[e];
  }
  __syncthreads();
  for (int d = tid; d < D; d += PRUNE_THREADS) load_o[d] = (long long)load[d];
  if (tid == 0) {
    long long Fd = 0, Fc = 0;
    for (int d = 0; d < D; ++d) { Fd = max(Fd, (long long)dense[d]); Fc = max(Fc, (long long)load[d]); }
    scalars[0] = F_base_s; scalars[1] = Fd; scalars[2] = Fc; scalars[3] = (long long)F_imp_s;
    scalars[4] = cnt[0]; scalars[5] = cnt[1]; scalars[6] = cnt[2];
  }
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
  float s[NV], sp[NV];
  uint32_t ok = 0;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int e = lane + 32 * i;
    s[i] = e < E ? scores[(size_t)t * E + e] : 0.f;
    sp[i] = (corr_bias && e < E) ? __fadd_rn(s[i], corr_bias[e]) : s[i];
    if (e < E && keep[e]) ok |= 1u << i;
  }
  __syncwarp();
  caee_warp_select<NV>(s, sp, ok, k, norm_topk, lane, ir, gate + (size_t)t * k);
}

}  // namespace

void caee_launch_prune(caee_ctx* c, int mode, int flags, double theta, int T, const int32_t* idx, const float* gate,
                       cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  k_prune<<<1, PRUNE_THREADS, 0, st>>>(mode, flags, theta, T, d.E, d.k, d.D, idx, gate, c->w_eff, c->part, c->act,
                                       c->must, c->keep, c->I_fix, c->load, c->scalars);
}

void caee_launch_compensate(caee_ctx* c, int flags, const float* scores, int T, int32_t* idx, float* gate,
                            cudaStream_t st) {
  const caee_layer_desc& d = c->d;
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
