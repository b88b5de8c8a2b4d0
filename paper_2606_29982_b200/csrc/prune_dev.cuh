// prune_dev.cuh — the block-level body of S2-S4, shared by k_prune
// (prune.cu) and the fused decode-size decision kernel k_decide (decide.cu).
//
// The decision is batch-global (x_e is per expert) and tiny (E <= 512), so
// one CTA takes it.  Integers everywhere (importance in units of 2^-40, costs in ns ticks)
// make the result independent of summation order.
#pragma once
#include "caee_internal.cuh"

struct caee_prune_smem {
  unsigned long long I[CAEE_MAX_E];      // I_fix(e)
  unsigned int I_lo[CAEE_MAX_E], I_hi[CAEE_MAX_E];  // 20-bit split accumulators (T <= 2048)
  long long w[CAEE_MAX_E];               // effective cost R(e,d) C~(e,d), ns
  int prt[CAEE_MAX_E];
  int sorted[CAEE_MAX_E];                // A_cand in (I desc, id asc) order
  unsigned char act[CAEE_MAX_E], must[CAEE_MAX_E], keep[CAEE_MAX_E];
  unsigned long long load[CAEE_MAX_D], load_must[CAEE_MAX_D], dense[CAEE_MAX_D];
  unsigned long long F_imp;
  long long F_base, thr;
  int n_cand, cnt[4];
};

// All threads of the block call this; idx/gate may point to shared or global memory.
// On return (after the final __syncthreads) sm.keep / sm.act are valid for the whole block.
__device__ __forceinline__ void caee_prune_block(caee_prune_smem& sm, int mode, int flags, double theta, int T, int E, int k,
                                                 int D, const int32_t* idx, const float* gate,
                                                 const int64_t* __restrict__ w_eff, const int32_t* __restrict__ part,
                                                 uint8_t* __restrict__ act_o, uint8_t* __restrict__ must_o,
                                                 uint8_t* __restrict__ keep_o, int64_t* __restrict__ I_o,
                                                 int64_t* __restrict__ load_o, int64_t* __restrict__ scalars) {
  const int tid = threadIdx.x, nth = blockDim.x;
  const bool split = T <= 2048;   // sum of <= 2048 values below 2^20 (+1) fits 32 bits: native shared atomics
  for (int e = tid; e < E; e += nth) {
    sm.I[e] = 0; sm.I_lo[e] = 0; sm.I_hi[e] = 0;
    sm.act[e] = 0; sm.must[e] = 0; sm.keep[e] = 0;
    sm.w[e] = w_eff[e]; sm.prt[e] = part[e];
  }
  for (int d = tid; d < D; d += nth) { sm.load[d] = 0; sm.load_must[d] = 0; sm.dense[d] = 0; }
  if (tid < 4) sm.cnt[tid] = 0;
  if (tid == 0) {
    sm.n_cand = 0;
    sm.F_imp = 0;
    sm.thr = mode == CAEE_PRUNE_THRESH ? (long long)floor(theta * 1099511627776.0) : 0;
  }
  __syncthreads();

  // S2: A_act and I_fix(e) = sum_t floor(G * 2^40)  (exact in fp32: power-of-two scale)
  for (int i = tid; i < T * k; i += nth) {
    const int e = idx[i];
    if (e >= 0) {
      sm.act[e] = 1;
      const unsigned long long v = (unsigned long long)__float2ll_rz(__fmul_rn(gate[i], CAEE_FIX_ONE_F));
      if (split) {
        atomicAdd(&sm.I_lo[e], (unsigned int)(v & 0xFFFFFu));
        atomicAdd(&sm.I_hi[e], (unsigned int)(v >> 20));
      } else {
        atomicAdd(&sm.I[e], v);
      }
    }
  }
  // per-token rules of step 1
  if (mode == CAEE_PRUNE_CIR) {
    const float th = (float)theta;
    for (int t = tid; t < T; t += nth) {
      const int32_t* ir = idx + (size_t)t * k;
      const float* gr = gate + (size_t)t * k;
      float pk = 0.f;
      for (int j = 0; j < k; ++j)
        if (ir[j] >= 0) pk = __fadd_rn(pk, gr[j]);
      const float rhs = __fmul_rn(th, pk);
      float pm = 0.f;
      for (int j = 0; j < k; ++j) {
        if (ir[j] < 0) break;
        sm.must[ir[j]] = 1;
        pm = __fadd_rn(pm, gr[j]);
        if (pm >= rhs) break;
      }
    }
  } else if (mode == CAEE_PRUNE_RANK) {
    const int b = (int)theta;
    for (int i = tid; i < T * k; i += nth) {
      const int e = idx[i];
      if (e >= 0 && (i % k) < k - b) sm.must[e] = 1;
    }
  }
  if ((flags & CAEE_KEEP_TOP1) && mode != CAEE_PRUNE_NONE)
    for (int t = tid; t < T; t += nth)
      if (idx[(size_t)t * k] >= 0) sm.must[idx[(size_t)t * k]] = 1;
  __syncthreads();

  // per-expert rules of step 1
  for (int e = tid; e < E; e += nth) {
    if (split) sm.I[e] = ((unsigned long long)sm.I_hi[e] << 20) + sm.I_lo[e];
    if (!sm.act[e]) continue;
    atomicAdd(&sm.cnt[0], 1);  // |A_act|
    if (mode == CAEE_PRUNE_NONE) sm.must[e] = 1;
    else if (mode == CAEE_PRUNE_THRESH && (long long)sm.I[e] >= sm.thr) sm.must[e] = 1;
  }
  __syncthreads();
  if (mode == CAEE_PRUNE_FRAC) {
    const long long n_cand = (long long)floor(theta * (double)sm.cnt[0]);
    for (int e = tid; e < E; e += nth) {
      if (!sm.act[e]) continue;
      const unsigned long long Ie = sm.I[e];
      int rank = 0;  // position in ascending (I, id) order among A_act
      for (int f = 0; f < E; ++f)
        if (sm.act[f] && (sm.I[f] < Ie || (sm.I[f] == Ie && f < e))) ++rank;
      if (rank >= n_cand) sm.must[e] = 1;
    }
    __syncthreads();
  }

  // step 2: F_base = max_d sum_{e in A_must ∩ E_d} w_e
  for (int e = tid; e < E; e += nth) {
    if (sm.must[e]) {
      sm.keep[e] = 1;
      atomicAdd(&sm.cnt[1], 1);
      atomicAdd(&sm.load_must[sm.prt[e]], (unsigned long long)sm.w[e]);
    }
  }
  __syncthreads();
  if (tid == 0) {
    long long m = 0;
    for (int d = 0; d < D; ++d) m = max(m, (long long)sm.load_must[d]);
    sm.F_base = m;
  }
  // candidates A_cand = A_act \ A_must ordered by (I desc, id asc)  (R3, R7)
  for (int e = tid; e < E; e += nth) {
    if (sm.act[e] && !sm.must[e]) {
      const unsigned long long Ie = sm.I[e];
      int rank = 0;
      for (int f = 0; f < E; ++f)
        if (sm.act[f] && !sm.must[f] && (sm.I[f] > Ie || (sm.I[f] == Ie && f < e))) ++rank;
      sm.sorted[rank] = e;
      atomicAdd(&sm.n_cand, 1);
    }
  }
  for (int d = tid; d < D; d += nth) sm.load[d] = sm.load_must[d];
  __syncthreads();
  // step 3: cost-invariant expansion; partitions are independent given F_base (R5, R6)
  if (tid < D) {
    const long long Fb = sm.F_base;
    long long l = (long long)sm.load[tid];
    const int nc = sm.n_cand;
    for (int r = 0; r < nc; ++r) {
      const int e = sm.sorted[r];
      if (sm.prt[e] != tid) continue;
      if (l + sm.w[e] <= Fb) { sm.keep[e] = 1; l += sm.w[e]; }
    }
    sm.load[tid] = (unsigned long long)l;
  }
  __syncthreads();

  // step 4 + reporting
  for (int e = tid; e < E; e += nth) {
    if (sm.act[e]) atomicAdd(&sm.dense[sm.prt[e]], (unsigned long long)sm.w[e]);
    if (sm.keep[e]) atomicAdd(&sm.cnt[2], 1);
    if (sm.act[e] && !sm.keep[e]) atomicAdd(&sm.F_imp, sm.I[e]);
    act_o[e] = sm.act[e]; must_o[e] = sm.must[e]; keep_o[e] = sm.keep[e]; I_o[e] = (long long)sm.I[e];
  }
  __syncthreads();
  for (int d = tid; d < D; d += nth) load_o[d] = (long long)sm.load[d];
  if (tid == 0) {
    long long Fd = 0, Fc = 0;
    for (int d = 0; d < D; ++d) { Fd = max(Fd, (long long)sm.dense[d]); Fc = max(Fc, (long long)sm.load[d]); }
    scalars[0] = sm.F_base; scalars[1] = Fd; scalars[2] = Fc; scalars[3] = (long long)sm.F_imp;
    scalars[4] = sm.cnt[0]; scalars[5] = sm.cnt[1]; scalars[6] = sm.cnt[2];
  }
}
