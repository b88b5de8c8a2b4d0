// prune_dev.cuh — device bodies of S2-S4, shared by the stand-alone
// k_prune (prune.cu) and the fused decode-size decision kernel (decide.cu).
//
//   caee_prune_token   one warp, one token: A_act bits, importance I_fix(e) += floor(G 2^40),
//                      and the per-token rules of step 1 (CIR, RANK, KEEP_TOP1) -> must bits
//   caee_prune_decide  one CTA, batch-global (x_e is per expert): per-expert
//                      rules of step 1, F_base, cost-invariant expansion, reporting
//
// Integers everywhere (importance in units of 2^-40, costs in ns ticks) make the result
// independent of summation order, so the masks are bit-exact against the CPU oracle.
#pragma once
#include "caee_internal.cuh"

#ifdef CAEE_DECIDE_TIMING
__device__ long long g_prune_clk[16];
#define PSTAMP(i) do { if (threadIdx.x == 0 && blockIdx.x == 0) g_prune_clk[i] = clock64(); } while (0)
#else
#define PSTAMP(i)
#endif

struct caee_prune_smem {
  unsigned long long I[CAEE_MAX_E];      // I_fix(e)
  unsigned long long key[CAEE_MAX_E];    // ordering key of the current ranking pass
  long long w[CAEE_MAX_E];               // effective cost R(e,d) C~(e,d), ns
  int prt[CAEE_MAX_E];
  int plist[CAEE_MAX_E];                 // A_cand grouped by partition, (I desc, id asc) inside a partition
  unsigned char act[CAEE_MAX_E], must[CAEE_MAX_E], keep[CAEE_MAX_E];
  long long load[CAEE_MAX_D], load_must[CAEE_MAX_D], dense[CAEE_MAX_D];
  int pcnt[CAEE_MAX_D], pbase[CAEE_MAX_D];
  unsigned long long F_imp;
  long long F_base, F_dense, F_cost, thr;
  int cnt[4];                            // |A_act|, |A_must|, |A_trans|
};

// S2 + per-token rules of step 1 for one token (all 32 lanes call it).  ir/gr: the token's
// K_t and gates; I/act/must: accumulators in shared or global memory.
// The per-token rules (CIR, RANK, KEEP_TOP1) see K_t "sorted by their gating scores"
// (PAPER.md:244): by (gate descending, expert id ascending), R36 — the route's list order is by
// the biased selection score and differs from it when corr_bias != 0.
__device__ __forceinline__ void caee_prune_token(int mode, int flags, double theta, int k, const int32_t* ir, const float* gr,
                                                 int lane, unsigned long long* I, unsigned char* act, unsigned char* must) {
  int e = -1;
  float g = 0.f;
  if (lane < k) { e = ir[lane]; g = gr[lane]; }
  if (e >= 0) {
    act[e] = 1;
    // exact in fp32: power-of-two scale, then truncation
    atomicAdd(&I[e], (unsigned long long)__float2ll_rz(__fmul_rn(g, CAEE_FIX_ONE_F)));
  }
  const bool top1 = (flags & CAEE_KEEP_TOP1) && mode != CAEE_PRUNE_NONE;
  if (mode != CAEE_PRUNE_CIR && mode != CAEE_PRUNE_RANK && !top1) return;
  // lane m <- the m-th entry of K_t by (gate desc, id asc); empty slots go last
  const float kg = e >= 0 ? g : -INFINITY;
  const int kid = e >= 0 ? e : (1 << 30) + lane;
  int rank = 0;
  for (int j = 0; j < k; ++j) {
    const float gj = __shfl_sync(0xffffffffu, kg, j);
    const int ij = __shfl_sync(0xffffffffu, kid, j);
    rank += (gj > kg) | ((gj == kg) & (ij < kid));
  }
  int se = -1;
  float sg = 0.f;
  for (int m = 0; m < k; ++m) {
    const int src = __ffs(__ballot_sync(0xffffffffu, lane < k && rank == m)) - 1;
    const float gv = __shfl_sync(0xffffffffu, g, src);
    const int ev = __shfl_sync(0xffffffffu, e, src);
    if (lane == m) { sg = gv; se = ev; }
  }
  if (mode == CAEE_PRUNE_CIR) {
    // minimal m* with p_m >= theta_imp * p_k, sums in sorted order (R9); k <= 32 values live in the lanes
    float pk = 0.f;
    for (int j = 0; j < k; ++j) {
      const float gj = __shfl_sync(0xffffffffu, sg, j);
      const int ej = __shfl_sync(0xffffffffu, se, j);
      if (ej >= 0) pk = __fadd_rn(pk, gj);
    }
    const float rhs = __fmul_rn((float)theta, pk);
    float pm = 0.f;
    bool open = true;    // slot j is within the first m*
    for (int j = 0; j < k; ++j) {
      const float gj = __shfl_sync(0xffffffffu, sg, j);
      const int ej = __shfl_sync(0xffffffffu, se, j);
      if (ej < 0) open = false;
      if (open && lane == j) must[se] = 1;
      pm = __fadd_rn(pm, gj);
      if (pm >= rhs) open = false;
    }
  } else if (mode == CAEE_PRUNE_RANK) {
    if (se >= 0 && lane < k - (int)theta) must[se] = 1;
  }
  if (top1 && lane == 0 && se >= 0) must[se] = 1;
}

__device__ __forceinline__ long long caee_warp_sum_ll(long long v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Warp-cooperative rank (all 32 lanes call it): the number of f in [0,E) whose (key, f) comes
// before (ke, e) — larger key first (kDesc) or smaller key first, ties -> lower index (R22) —
// and, with prt != nullptr, that lie in partition d.  Branch-free; keys live in shared memory.
template <bool kDesc>
__device__ __forceinline__ int caee_warp_rank(const unsigned long long* key, const int* prt, int d, int E,
                                              unsigned long long ke, int e, int lane) {
  int rank = 0;
  for (int f = lane; f < E; f += 32) {
    const unsigned long long kf = key[f];
    const int first = kDesc ? (kf > ke) : (kf < ke);
    const int same = prt ? (prt[f] == d) : 1;
    rank += (first | ((kf == ke) & (f < e))) & same;
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) rank += __shfl_xor_sync(0xffffffffu, rank, o);
  return rank;
}

// Steps 1 (per-expert rules) - 4 of the heuristic for the whole batch; all threads of the CTA
// call it.  On entry sm.I / sm.act / sm.must hold S2's result and the per-token rules, and
// the CTA is synchronised.  With `out` set the CTA also writes the result arrays (else only
// shared memory is filled: several CTAs may take the same decision redundantly).
// On return (synchronised) sm.keep, sm.load, sm.F_*, sm.cnt are valid.
__device__ __forceinline__ void caee_prune_decide(caee_prune_smem& sm, int mode, int flags, double theta, double eps, int E, int D,
                                                  const int64_t* __restrict__ w_eff, const int32_t* __restrict__ part, bool out,
                                                  uint8_t* __restrict__ act_o, uint8_t* __restrict__ must_o,
                                                  uint8_t* __restrict__ keep_o, int64_t* __restrict__ I_o,
                                                  int64_t* __restrict__ load_o, int64_t* __restrict__ scalars) {
  const int tid = threadIdx.x, nth = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nth >> 5;
  const int Er = (E + 31) & ~31;   // warp-uniform trip counts
  PSTAMP(0);
  if (tid < 4) sm.cnt[tid] = 0;
  if (tid == 0) {
    sm.F_imp = 0;
    sm.thr = mode == CAEE_PRUNE_THRESH ? (long long)floor(theta * 1099511627776.0) : 0;
  }
  for (int e = tid; e < E; e += nth) { sm.w[e] = w_eff[e]; sm.prt[e] = part[e]; sm.keep[e] = 0; }
  __syncthreads();
  PSTAMP(1);

  // step 1, per-expert rules: THRESH / NONE; |A_act|
  for (int e = tid; e < Er; e += nth) {
    const bool a = e < E && sm.act[e];
    if (a) {
      if (mode == CAEE_PRUNE_NONE) sm.must[e] = 1;
      else if (mode == CAEE_PRUNE_THRESH && (long long)sm.I[e] >= sm.thr) sm.must[e] = 1;
    }
    const unsigned b = __ballot_sync(0xffffffffu, a);
    if (lane == 0 && b) atomicAdd(&sm.cnt[0], __popc(b));
    if (e < E) sm.key[e] = a ? sm.I[e] : ~0ull;     // FRAC: ascending (I, id) among A_act
  }
  __syncthreads();
  if (mode == CAEE_PRUNE_FRAC) {
    const long long n_cand = (long long)floor(theta * (double)sm.cnt[0]);
    for (int e = warp; e < E; e += nwarps)   // warp-uniform: one expert per warp at a time
      if (sm.act[e] && caee_warp_rank<false>(sm.key, nullptr, 0, E, sm.key[e], e, lane) >= n_cand && lane == 0) sm.must[e] = 1;
    __syncthreads();
  }

  PSTAMP(2);
  // step 2: loads of A_must (and of A_act, for F_cost_dense) per partition; candidates per partition
  for (int e = tid; e < Er; e += nth) {
    const bool m = e < E && sm.must[e];
    if (m) sm.keep[e] = 1;
    const unsigned b = __ballot_sync(0xffffffffu, m);
    if (lane == 0 && b) atomicAdd(&sm.cnt[1], __popc(b));
    // A_cand = A_act \ A_must, ordered by (I desc, id asc)  (R3, R7); I + 1 > 0 marks membership
    if (e < E) sm.key[e] = (sm.act[e] && !m) ? sm.I[e] + 1 : 0ull;
  }
  __syncthreads();
  PSTAMP(3);
  for (int d = warp; d < D; d += nwarps) {
    long long lm = 0, la = 0;
    int nc = 0;
    for (int e = lane; e < E; e += 32) {
      if (sm.prt[e] != d) continue;
      if (sm.must[e]) lm += sm.w[e];
      if (sm.act[e]) la += sm.w[e];
      nc += sm.key[e] != 0;
    }
    lm = caee_warp_sum_ll(lm);
    la = caee_warp_sum_ll(la);
#pragma unroll
    for (int o = 16; o; o >>= 1) nc += __shfl_xor_sync(0xffffffffu, nc, o);
    if (lane == 0) { sm.load_must[d] = lm; sm.dense[d] = la; sm.pcnt[d] = nc; }
  }
  __syncthreads();
  if (tid == 0) {
    long long fb = 0, fd = 0;
    int base = 0;
    for (int d = 0; d < D; ++d) {
      fb = max(fb, sm.load_must[d]);   // F_base = max_d sum_{A_must ∩ E_d} R C~
      fd = max(fd, sm.dense[d]);
      sm.pbase[d] = base;
      base += sm.pcnt[d];
    }
    sm.F_base = fb;
    sm.F_dense = fd;
  }
  __syncthreads();
  PSTAMP(4);
  // each candidate's place among the candidates of its own partition
  for (int e = warp; e < E; e += nwarps) {
    const unsigned long long ke = sm.key[e];
    if (ke == 0) continue;
    const int d = sm.prt[e];
    const int rank = caee_warp_rank<true>(sm.key, sm.prt, d, E, ke, e, lane);
    if (lane == 0) sm.plist[sm.pbase[d] + rank] = e;
  }
  __syncthreads();
  PSTAMP(5);
  // step 3: cost-invariant expansion; only part(e)'s load changes, so the
  // partitions are independent given F_base (R5); "= F_base" is "<= F_base" on integer ticks (R6)
  if (tid < D) {
    const long long Fb = sm.F_base;
    long long l = sm.load_must[tid];
    const int* lst = sm.plist + sm.pbase[tid];
    const int nc = sm.pcnt[tid];
    for (int r = 0; r < nc; ++r) {
      const int e = lst[r];
      const long long we = sm.w[e];
      if (l + we <= Fb) { sm.keep[e] = 1; l += we; }
    }
    sm.load[tid] = l;
  }
  __syncthreads();
  if (flags & CAEE_IMP_BOUND) {
    // importance bound F_imp(X) <= eps (R37): the pruned experts return in
    // descending (I, id asc) order while the pruned importance exceeds eps, i.e. expert e returns
    // iff the importance of the pruned experts from e onwards in that order exceeds eps
    const long long eps_fix = (long long)floor(eps * 1099511627776.0);
    for (int e = tid; e < E; e += nth) sm.key[e] = (sm.act[e] && !sm.keep[e]) ? sm.I[e] + 1 : 0ull;
    __syncthreads();
    for (int e = warp; e < E; e += nwarps) {
      const unsigned long long ke = sm.key[e];
      if (ke == 0) continue;
      long long tail = 0;
      for (int f = lane; f < E; f += 32) {
        const unsigned long long kf = sm.key[f];
        const bool from_e = kf != 0 && (kf < ke || (kf == ke && f >= e));
        tail += from_e ? (long long)(kf - 1) : 0;
      }
      tail = caee_warp_sum_ll(tail);
      if (lane == 0 && tail > eps_fix) sm.keep[e] = 1;
    }
    __syncthreads();
    for (int d = warp; d < D; d += nwarps) {
      long long l = 0;
      for (int e = lane; e < E; e += 32)
        if (sm.prt[e] == d && sm.keep[e]) l += sm.w[e];
      l = caee_warp_sum_ll(l);
      if (lane == 0) sm.load[d] = l;
    }
    __syncthreads();
  }

  PSTAMP(6);
  // step 4 + reporting
  for (int e = tid; e < Er; e += nth) {
    const bool kp = e < E && sm.keep[e];
    const unsigned b = __ballot_sync(0xffffffffu, kp);
    if (lane == 0 && b) atomicAdd(&sm.cnt[2], __popc(b));
    long long lost = (e < E && sm.act[e] && !kp) ? (long long)sm.I[e] : 0;
    lost = caee_warp_sum_ll(lost);
    if (lane == 0 && lost) atomicAdd(&sm.F_imp, (unsigned long long)lost);
    if (out && e < E) { act_o[e] = sm.act[e]; must_o[e] = sm.must[e]; keep_o[e] = sm.keep[e]; I_o[e] = (long long)sm.I[e]; }
  }
  __syncthreads();
  if (tid == 0) {
    long long fc = 0;
    for (int d = 0; d < D; ++d) fc = max(fc, sm.load[d]);
    sm.F_cost = fc;
  }
  __syncthreads();
  if (out) {
    for (int d = tid; d < D; d += nth) load_o[d] = sm.load[d];
    if (tid == 0) {
      scalars[0] = sm.F_base; scalars[1] = sm.F_dense; scalars[2] = sm.F_cost; scalars[3] = (long long)sm.F_imp;
      scalars[4] = sm.cnt[0]; scalars[5] = sm.cnt[1]; scalars[6] = sm.cnt[2];
    }
  }
  PSTAMP(7);
}
