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
  unsigned long long key[CAEE_MAX_E];    // ordering key of the current ranking pass / costs of a partition's candidates in visiting order
  long long w[CAEE_MAX_E];               // effective cost R(e,d) C~(e,d), ns
  int prt[CAEE_MAX_E];
  int plist[CAEE_MAX_E];                 // A_cand grouped by partition, (I desc, id asc) inside a partition;
                                         // the partition-per-warp path keeps the static lists E_d here (ascending id)
  unsigned char act[CAEE_MAX_E], must[CAEE_MAX_E], keep[CAEE_MAX_E];
  long long load[CAEE_MAX_D], load_must[CAEE_MAX_D], dense[CAEE_MAX_D];
  unsigned long long lost[CAEE_MAX_D];   // importance pruned in a partition
  int pcnt[CAEE_MAX_D], pbase[CAEE_MAX_D + 1];
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


// ---------------------------------------------------------------------------------------------
// The same decision (steps 1-4) with one WARP per partition, for partition
// tables whose largest E_d has at most 32 experts (c->part_max; every BASELINE.json config):
// a partition's experts sit one per lane, so its loads are two redux.sync adds, the order of its
// candidates is 32 shuffles, and the cost-invariant expansion of step 3 — independent between
// partitions once F_base is known (R5) — is a division when the partition's candidates cost the
// same and otherwise a short serial pass by one lane.  Four block barriers instead of fourteen;
// bit-identical to caee_prune_decide (integer arithmetic, same visiting order R7/R22).
//
// caee_prune_preload copies the per-layer tables into shared memory; kernels call it first so
// that the (cold) loads overlap the token pass.  pl_experts: the experts grouped by partition,
// ascending id inside a partition; pl_start[d]: where E_d starts (D + 1 entries).
__device__ __forceinline__ void caee_prune_preload(caee_prune_smem& sm, int E, int D, const int64_t* __restrict__ w_eff,
                                                   const int32_t* __restrict__ part, const int32_t* __restrict__ pl_experts,
                                                   const int32_t* __restrict__ pl_start) {
  for (int e = threadIdx.x; e < E; e += blockDim.x) { sm.w[e] = w_eff[e]; sm.prt[e] = part[e]; sm.plist[e] = pl_experts[e]; }
  for (int d = threadIdx.x; d <= D; d += blockDim.x) sm.pbase[d] = pl_start[d];
}

// sum over the warp of non-negative values < 2^41 (costs are <= 2^40 ns): two 32-bit redux.sync adds
__device__ __forceinline__ long long caee_warp_sum_cost(long long v) {
  const unsigned lo = __reduce_add_sync(0xffffffffu, (unsigned)(v & 0x3fffff));
  const unsigned hi = __reduce_add_sync(0xffffffffu, (unsigned)(v >> 22));
  return ((long long)hi << 22) + (long long)lo;
}

__device__ __forceinline__ void caee_prune_decide_fast(caee_prune_smem& sm, int mode, int flags, double theta, double eps, int E,
                                                       int D, bool out, uint8_t* __restrict__ act_o, uint8_t* __restrict__ must_o,
                                                       uint8_t* __restrict__ keep_o, int64_t* __restrict__ I_o,
                                                       int64_t* __restrict__ load_o, int64_t* __restrict__ scalars) {
  const int tid = threadIdx.x, nth = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nth >> 5;
  PSTAMP(0);
  // step 1, per-expert rules (thread e owns expert e; blockDim.x >= E)
  const bool a = tid < E && sm.act[tid];
  const int n_act = __syncthreads_count(a);
  bool m = false;
  if (mode == CAEE_PRUNE_FRAC) {
    if (tid < E) sm.key[tid] = a ? sm.I[tid] : ~0ull;      // ascending (I, id) among A_act
    __syncthreads();
    const long long n_cand = (long long)floor(theta * (double)n_act);
    for (int e = warp; e < E; e += nwarps)
      if (sm.act[e] && caee_warp_rank<false>(sm.key, nullptr, 0, E, sm.key[e], e, lane) >= n_cand && lane == 0) sm.must[e] = 1;
    __syncthreads();
    m = a && sm.must[tid];
  } else if (a) {
    m = sm.must[tid] || mode == CAEE_PRUNE_NONE ||
        (mode == CAEE_PRUNE_THRESH && (long long)sm.I[tid] >= (long long)floor(theta * 1099511627776.0));
    sm.must[tid] = m;
  }
  const int n_must = __syncthreads_count(m);            // also publishes sm.must
  PSTAMP(1);
  // step 2: per-partition loads of A_must and of A_act
  for (int d = warp; d < D; d += nwarps) {
    const int p0 = sm.pbase[d], nd = sm.pbase[d + 1] - p0;
    const int e = lane < nd ? sm.plist[p0 + lane] : -1;
    const long long we = e >= 0 ? sm.w[e] : 0;
    const long long lm = caee_warp_sum_cost((e >= 0 && sm.must[e]) ? we : 0);
    const long long la = caee_warp_sum_cost((e >= 0 && sm.act[e]) ? we : 0);
    if (lane == 0) { sm.load_must[d] = lm; sm.dense[d] = la; }
  }
  __syncthreads();
  PSTAMP(2);
  long long Fb = 0, Fd = 0;       // F_base = max_d sum_{A_must ∩ E_d} R C~; every thread takes the max itself
  for (int d = 0; d < D; ++d) { Fb = max(Fb, sm.load_must[d]); Fd = max(Fd, sm.dense[d]); }
  // step 3: cost-invariant expansion, one warp per partition
  for (int d = warp; d < D; d += nwarps) {
    const int p0 = sm.pbase[d], nd = sm.pbase[d + 1] - p0;
    const int e = lane < nd ? sm.plist[p0 + lane] : -1;
    const bool ea = e >= 0 && sm.act[e], em = e >= 0 && sm.must[e];
    const bool cand = ea && !em;
    const long long we = e >= 0 ? sm.w[e] : 0;
    const unsigned long long Ie = e >= 0 ? sm.I[e] : 0ull;
    const unsigned cmask = __ballot_sync(0xffffffffu, cand);
    const int nc = __popc(cmask);
    const long long lm = sm.load_must[d];
    long long l = lm;
    bool kept = false;
    if (nc > 0) {
      // place among the partition's candidates: descending I, ties -> lower id = lower lane (R7, R22)
      int rank = 0;
      for (int q = 0; q < nd; ++q) {
        const unsigned long long Iq = __shfl_sync(0xffffffffu, Ie, q);
        rank += ((cmask >> q) & 1u) & ((Iq > Ie) | ((Iq == Ie) & (q < lane)));
      }
      const long long w0 = __shfl_sync(0xffffffffu, we, __ffs(cmask) - 1);
      const bool uniform = __all_sync(0xffffffffu, !cand || we == w0);
      if (uniform) {
        // equal costs: the first floor((F_base - load) / w) candidates fit, the rest do not
        const long long room = Fb - lm;
        const int fit = w0 == 0 ? nc : (int)min((long long)nc, room / w0);
        kept = cand && rank < fit;
        l = lm + (long long)fit * w0;
      } else {
        if (cand) sm.key[p0 + rank] = (unsigned long long)we;
        __syncwarp();
        unsigned bits = 0;
        if (lane == 0) {
          for (int r = 0; r < nc; ++r) {
            const long long wr = (long long)sm.key[p0 + r];
            if (l + wr <= Fb) { l += wr; bits |= 1u << r; }
          }
        }
        bits = __shfl_sync(0xffffffffu, bits, 0);
        l = __shfl_sync(0xffffffffu, l, 0);
        kept = cand && ((bits >> rank) & 1u);
      }
    }
    const bool kp = em || kept;
    if (e >= 0) sm.keep[e] = kp;
    const unsigned kmask = __ballot_sync(0xffffffffu, kp);
    const long long lost = caee_warp_sum_ll((ea && !kp) ? (long long)Ie : 0);
    if (lane == 0) { sm.load[d] = l; sm.pcnt[d] = __popc(kmask); sm.lost[d] = (unsigned long long)lost; }
  }
  if (tid >= E && tid < CAEE_MAX_E) sm.keep[tid] = 0;
  __syncthreads();
  PSTAMP(3);
  if (flags & CAEE_IMP_BOUND) {
    // importance bound F_imp(X) <= eps (R37): as in caee_prune_decide
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
      const int p0 = sm.pbase[d], nd = sm.pbase[d + 1] - p0;
      const int e = lane < nd ? sm.plist[p0 + lane] : -1;
      const bool kp = e >= 0 && sm.keep[e];
      const long long l = caee_warp_sum_cost(kp ? sm.w[e] : 0);
      const long long lost = caee_warp_sum_ll((e >= 0 && sm.act[e] && !kp) ? (long long)sm.I[e] : 0);
      const unsigned kmask = __ballot_sync(0xffffffffu, kp);
      if (lane == 0) { sm.load[d] = l; sm.pcnt[d] = __popc(kmask); sm.lost[d] = (unsigned long long)lost; }
    }
    __syncthreads();
  }
  // step 4 + reporting
  if (tid == 0) {
    long long fc = 0;
    unsigned long long fi = 0;
    int nk = 0;
    for (int d = 0; d < D; ++d) { fc = max(fc, sm.load[d]); fi += sm.lost[d]; nk += sm.pcnt[d]; }
    sm.F_base = Fb; sm.F_dense = Fd; sm.F_cost = fc; sm.F_imp = fi;
    sm.cnt[0] = n_act; sm.cnt[1] = n_must; sm.cnt[2] = nk;
    if (out) {
      scalars[0] = Fb; scalars[1] = Fd; scalars[2] = fc; scalars[3] = (long long)fi;
      scalars[4] = n_act; scalars[5] = n_must; scalars[6] = nk;
    }
  }
  if (out) {
    if (tid < E) { act_o[tid] = sm.act[tid]; must_o[tid] = sm.must[tid]; keep_o[tid] = sm.keep[tid]; I_o[tid] = (long long)sm.I[tid]; }
    if (tid < D) load_o[tid] = sm.load[tid];
  }
  __syncthreads();
  PSTAMP(4);
}
