// decide.cu — the decode-size decision step as ONE kernel: S1 top-k + gates, S2 activation set
// and importance, S3 cost lookup / F_cost, S4 cost-aware pruning, S5 compensation, S6
// compaction into the expert kernel's work list, and the step's caee_fwd_stats
// (BASELINE.json north_star subsystem (1)).
//
// Why one CTA.  The pruning decision is batch-global: x_e is one bit per expert for the whole
// batch, so every token's top-k must be known before any expert can be
// pruned, and every expert's fate before any token can be compensated.  At decode sizes
// (T*k <= 2048 entries, E <= 512) the whole state fits one CTA's shared memory, so the grid-wide
// dependencies become __syncthreads and the five launches (plus two memsets) of the
// stand-alone path collapse into this one; each stage runs exactly the device code of the
// stand-alone kernels (warp_select.cuh, prune_dev.cuh, worklist_dev.cuh), so both paths give
// bit-identical decisions.  Larger steps (prefill) use the stand-alone kernels.
#include "caee_internal.cuh"
#include "prune_dev.cuh"
#include "warp_select.cuh"
#include "worklist_dev.cuh"

namespace {

constexpr int kDecideThreads = 1024;
constexpr int kMaxEnt = CAEE_DECIDE_MAX_ENTRIES;

struct DecideParams {
  const float* logits;     // [T,E] x W_r^T (k_router_logits), or NULL with scores_in
  const float* b_logit;
  const float* scores_in;  // [T,E] caller's post-activation scores, or NULL
  const float* corr_bias;
  float* scores;           // [T,E] scratch: the scores this step used (read back by compensation)
  int32_t* idx;            // [T,k] out: K_final
  float* gate;             // [T,k] out
  int T, E, k, S, D, n_group, topk_group, score_fn, norm_topk;
  int has_prune, mode, flags;
  double theta;
  const int64_t* w_eff;
  const int32_t* part;
  const uint8_t* resident;
  uint8_t *act, *must, *keep;
  int64_t *I_fix, *load, *scalars;
  caee_worklist wl;
  int n_sched;             // ints of wl.sched to zero (tile tickets + per-run counters)
  caee_fwd_stats* stats;   // or NULL
  long long bytes_per_expert;
};

template <int NV>
__global__ void __launch_bounds__(kDecideThreads, 1) k_decide(const DecideParams p) {
  __shared__ caee_prune_smem sm;
  __shared__ int32_t s_idx[kMaxEnt];
  __shared__ float s_gate[kMaxEnt];
  __shared__ int32_t s_cnt[CAEE_MAX_E], s_est[CAEE_MAX_E];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = kDecideThreads / 32;
  const int T = p.T, E = p.E, k = p.k;

  for (int i = tid; i < p.n_sched; i += kDecideThreads) p.wl.sched[i] = 0;
  for (int e = tid; e < E; e += kDecideThreads) s_cnt[e] = 0;

  // S0 tail + S1: one warp per token
  for (int t = warp; t < T; t += nwarps) {
    float s[NV];
    caee_token_scores<NV>(p.scores_in ? p.scores_in + (size_t)t * E : nullptr, p.logits ? p.logits + (size_t)t * E : nullptr,
                          p.b_logit, E, p.score_fn, lane, s);
    if (!p.scores_in) {
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        const int e = lane + 32 * i;
        if (e < E) p.scores[(size_t)t * E + e] = s[i];
      }
    }
    caee_route_token<NV>(s, p.corr_bias, E, k, p.n_group, p.topk_group, p.norm_topk, lane, s_idx + t * k, s_gate + t * k);
  }
  __syncthreads();

  // S2-S4
  const bool prunes = p.has_prune && p.mode != CAEE_PRUNE_NONE;
  if (p.has_prune) {
    caee_prune_block(sm, p.mode, p.flags, p.theta, T, E, k, p.D, s_idx, s_gate, p.w_eff, p.part, p.act, p.must, p.keep,
                     p.I_fix, p.load, p.scalars);
    __syncthreads();
  }
  // S5: tokens that lost an expert re-select inside A_trans
  if (prunes) {
    const float* sc = p.scores_in ? p.scores_in : p.scores;
    for (int t = warp; t < T; t += nwarps) {
      int32_t* ir = s_idx + t * k;
      bool bad = false;
      if (lane < k) { const int e = ir[lane]; bad = e >= 0 && !sm.keep[e]; }
      const bool affected = __any_sync(0xffffffffu, bad) || (p.flags & CAEE_COMP_ALL_TOKENS);
      if (affected) caee_compensate_token<NV>(sc + (size_t)t * E, p.corr_bias, sm.keep, E, k, p.norm_topk, lane, ir, s_gate + t * k);
    }
    __syncthreads();
  }

  // S6: counts -> scan -> fill; K_final to global
  for (int i = tid; i < T * k; i += kDecideThreads) {
    const int e = s_idx[i];
    p.idx[i] = e;
    p.gate[i] = s_gate[i];
    if (e >= 0) atomicAdd(&s_cnt[e], 1);
  }
  __syncthreads();
  if (warp == 0) caee_wl_scan_warp(p.wl, s_cnt, s_est, p.resident, T, E, p.S, k, lane);
  __syncthreads();
  for (int e = warp; e < E + p.S; e += nwarps) caee_wl_fill_expert(p.wl, s_cnt, s_est, s_idx, s_gate, T, E, p.S, k, e, lane);
  if (p.stats && tid < 64)
    caee_stats_fill(p.stats, p.scalars, p.load, p.wl.meta, p.D, p.S, p.has_prune, p.bytes_per_expert, 0, tid, 64);
}

}  // namespace

bool caee_decide_fits(const caee_ctx* c, int T) { return T > 0 && (long long)T * c->d.k <= kMaxEnt; }

void caee_launch_decide(caee_ctx* c, const float* scores_in, int T, const caee_prune_params* pp, caee_fwd_stats* stats,
                        cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  DecideParams p;
  p.logits = scores_in ? nullptr : c->logits;
  p.b_logit = c->b_logit; p.scores_in = scores_in; p.corr_bias = c->corr_bias;
  p.scores = c->scores; p.idx = c->idx; p.gate = c->gate;
  p.T = T; p.E = d.E; p.k = d.k; p.S = d.S; p.D = d.D; p.n_group = d.n_group; p.topk_group = d.topk_group;
  p.score_fn = d.score_fn; p.norm_topk = d.norm_topk;
  p.has_prune = pp != nullptr; p.mode = pp ? pp->mode : CAEE_PRUNE_NONE; p.flags = pp ? pp->flags : 0;
  p.theta = pp ? pp->theta : 0.0;
  p.w_eff = c->w_eff; p.part = c->part; p.resident = c->resident;
  p.act = c->act; p.must = c->must; p.keep = c->keep; p.I_fix = c->I_fix; p.load = c->load; p.scalars = c->scalars;
  p.wl = c->wl; p.n_sched = c->wl.n_tickets + c->wl.max_runs;
  p.stats = stats; p.bytes_per_expert = caee_expert_bytes(c);
  const int nv = caee_ceil_div(d.E, 32);
  if (nv <= 1) k_decide<1><<<1, kDecideThreads, 0, st>>>(p);
  else if (nv <= 2) k_decide<2><<<1, kDecideThreads, 0, st>>>(p);
  else if (nv <= 4) k_decide<4><<<1, kDecideThreads, 0, st>>>(p);
  else if (nv <= 8) k_decide<8><<<1, kDecideThreads, 0, st>>>(p);
  else k_decide<16><<<1, kDecideThreads, 0, st>>>(p);
}
