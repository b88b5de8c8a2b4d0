// decide.cu — the decode-size decision step as ONE cooperative kernel: S1 top-k + gates, S2
// activation set and importance, S3 cost lookup / F_cost, S4 cost-aware pruning, S5
// compensation, S6 compaction into the expert kernel's work list, and the step's
// caee_fwd_stats (BASELINE.json north_star subsystem (1)).
//
// Shape.  One warp per token (a token's E scores live in the warp's registers; selection is
// warp shuffles, warp_select.cuh), 16 tokens per CTA, ceil(T/16) <= 16 CTAs, launched
// cooperatively.  The pruning decision is batch-global — x_e is one bit per expert for the
// whole batch — so there are two grid-wide dependencies:
//   A  route own token; add its gates to the global importance accumulators, set A_act /
//      per-token must bits                                         ── grid barrier 1 ──
//   B  EVERY CTA takes the (deterministic, integer) pruning decision redundantly from the
//      accumulators in its own shared memory (prune_dev.cuh): cheaper than a second barrier
//   C  compensate own token if it lost an expert; publish K_final as bits of the E x T
//      membership matrix M                                         ── grid barrier 2 ──
//   D  every CTA scans the per-expert counts (popcounts of M) itself; each warp places its
//      token's entries (position = popcount prefix in M); CTA 0 writes runs, meta, stats.
// The last CTA to leave clears the accumulators, M and the barrier counters for the next
// step.  Each stage runs the device code of the stand-alone kernels (router.cu, prune.cu,
// worklist.cu), so both paths give bit-identical decisions; steps with more than 256 tokens
// (prefill) use the stand-alone kernels.
#include <cooperative_groups.h>

#include "act_split_dev.cuh"
#include "caee_internal.cuh"
#include "prune_dev.cuh"
#include "warp_select.cuh"
#include "worklist_dev.cuh"

#ifdef CAEE_DECIDE_TIMING
__device__ long long g_decide_clk[16];
#define STAMP(i) do { if (threadIdx.x == 0 && blockIdx.x == 0) g_decide_clk[i] = clock64(); } while (0)
extern "C" void caee_debug_decide_clocks(long long* out) { cudaMemcpyFromSymbol(out, g_decide_clk, sizeof(long long) * 16); }
extern "C" void caee_debug_route_clocks(long long* out) { cudaMemcpyFromSymbol(out, g_route_clk, sizeof(long long) * 16); }
extern "C" void caee_debug_prune_clocks(long long* out) { cudaMemcpyFromSymbol(out, g_prune_clk, sizeof(long long) * 16); }
#else
#define STAMP(i)
#endif

namespace {

constexpr int kThreads = CAEE_MAX_E;          // 512: thread e owns expert e in the batch-global stages
constexpr int kWarps = kThreads / 32;         // tokens per CTA
constexpr int kWords = CAEE_DECIDE_MAX_TOKENS / 32;

struct DecideParams {
  const float* logits;     // [n_part][T,E] split-K partials of x W_r^T (k_router_logits), or NULL with scores_in
  int n_part;
  const float* b_logit;
  const float* scores_in;  // [T,E] caller's post-activation scores, or NULL
  const float* corr_bias;
  float* scores;           // [T,E] scratch: the scores this step used (read back by compensation)
  int32_t* idx;            // [T,k] out: K_final
  float* gate;             // [T,k] out
  int T, E, k, S, D, n_group, topk_group, score_fn, norm_topk;
  int has_prune, mode, flags;
  double theta, eps;
  const int64_t* w_eff;
  const int32_t* part;
  const int32_t *pl_experts, *pl_start;   // E_d as lists (prune_dev.cuh)
  int fast;                               // one warp per partition (largest E_d <= 32)
  const uint8_t* resident;
  uint8_t *act, *must, *keep;
  int64_t *I_fix, *load, *scalars;
  caee_worklist wl;
  int n_sched;             // ints of wl.sched to zero (tile tickets + per-run counters)
  caee_fwd_stats* stats;   // or NULL
  long long bytes_per_expert;
  // self-cleaning global scratch (zero between steps)
  unsigned long long* acc_I;  // [E]
  unsigned char* acc_act;     // [E]
  unsigned char* acc_must;    // [E]
  uint32_t* M;                // [E, kWords]
  int* bar;                   // [4]: barrier 1, barrier 2, exit ticket
  // e4m3 decode steps of <= 16 tokens: the one-CTA kernel also splits x into its two e4m3 terms (expert_fp8.cu),
  // before it waits for the router GEMM — the split depends on x alone, so its launch and its time disappear
  const __nv_bfloat16* split_x;   // NULL: not this step
  uint8_t *split_hi, *split_lo;
  float* split_scale;
  int split_blocks;               // T * H / 128
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// All CTAs of the (co-resident, cooperative) grid arrive; nobody leaves before everyone has.
__device__ __forceinline__ void grid_barrier(int* ctr, int G) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(ctr, 1);
    while (ld_acquire_gpu(ctr) < G) {}
    __threadfence();
  }
  __syncthreads();
}

// kSingle: the whole step fits ONE CTA (T <= 16).  The accumulators and the membership matrix then
// live in shared memory, the two grid barriers are block barriers, nothing has to be cleaned up
// for the next step, and the kernel needs no cooperative launch.
template <int NV, bool kSingle>
__global__ void __launch_bounds__(kThreads, 1) k_decide(const DecideParams p) {
  __shared__ caee_prune_smem sm;
  __shared__ int32_t s_idx[kWarps][32];
  __shared__ float s_gate[kWarps][32];
  __shared__ int32_t s_est[CAEE_MAX_E];
  __shared__ int s_scan[33 * 6];
  __shared__ int s_last;
  __shared__ uint32_t s_M[kSingle ? CAEE_MAX_E : 1];     // one 32-bit word per expert covers the <= 16 tokens
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, G = gridDim.x;
  const int T = p.T, E = p.E, k = p.k;
  const int t = blockIdx.x * kWarps + warp;   // this warp's token
  const bool live = t < T;
  const bool prunes = p.has_prune && p.mode != CAEE_PRUNE_NONE;
  int32_t* ir = s_idx[warp];
  float* gr = s_gate[warp];
  unsigned long long* acc_I = kSingle ? sm.I : p.acc_I;
  unsigned char* acc_act = kSingle ? sm.act : p.acc_act;
  unsigned char* acc_must = kSingle ? sm.must : p.acc_must;
  uint32_t* M = kSingle ? s_M : p.M;
  const int mwords = kSingle ? 1 : kWords;

  STAMP(0);
  // everything up to the first read of the router's partial logits touches only per-layer tables:
  // with a programmatic dependent launch it overlaps the router GEMM's tail
  float bl[NV], cb[NV];
  caee_load_vec<NV>(p.scores_in ? nullptr : p.b_logit, E, lane, bl);
  caee_load_vec<NV>(p.corr_bias, E, lane, cb);
  if (p.has_prune && p.fast) caee_prune_preload(sm, E, p.D, p.w_eff, p.part, p.pl_experts, p.pl_start);
  if (kSingle) {
    for (int e = tid; e < E; e += kThreads) { sm.I[e] = 0; sm.act[e] = 0; sm.must[e] = 0; s_M[e] = 0; }
    if (p.split_x)
      for (int b = warp; b < p.split_blocks; b += kWarps) caee_act_split_block(p.split_x, p.split_hi, p.split_lo, p.split_scale, (size_t)b, lane);
    __syncthreads();
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the expert kernel's CTAs may be scheduled (they wait for this grid)
  if (blockIdx.x == 0)
    for (int i = tid; i < p.n_sched; i += kThreads) p.wl.sched[i] = 0;

  // ---- A: S0 tail + S1 for this warp's token; S2 + per-token rules into the accumulators
  if (live) {
    float s[NV];
    caee_token_scores<NV>(p.scores_in ? p.scores_in + (size_t)t * E : nullptr, p.logits ? p.logits + (size_t)t * E : nullptr,
                          p.n_part, (size_t)T * E, p.b_logit != nullptr, bl, E, p.score_fn, lane, s);
    if (!p.scores_in && prunes) {
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        const int e = lane + 32 * i;
        if (e < E) p.scores[(size_t)t * E + e] = s[i];
      }
    }
    caee_route_token<NV>(s, p.corr_bias != nullptr, cb, E, k, p.n_group, p.topk_group, p.norm_topk, lane, ir, gr);
    __syncwarp();
    if (p.has_prune) caee_prune_token(p.mode, p.flags, p.theta, k, ir, gr, lane, acc_I, acc_act, acc_must);
  }
  STAMP(1);
  if (p.has_prune) {
    if (kSingle) __syncthreads();
    else grid_barrier(p.bar + 0, G);
    STAMP(2);
    // ---- B: S2-S4 for the batch, redundantly per CTA; CTA 0 writes the result arrays
    if (!kSingle) {
      for (int e = tid; e < E; e += kThreads) {
        sm.I[e] = __ldcg(p.acc_I + e);
        sm.act[e] = __ldcg(p.acc_act + e);
        sm.must[e] = __ldcg(p.acc_must + e);
      }
      __syncthreads();
    }
    if (p.fast)
      caee_prune_decide_fast(sm, p.mode, p.flags, p.theta, p.eps, E, p.D, blockIdx.x == 0, p.act, p.must, p.keep, p.I_fix, p.load,
                             p.scalars);
    else
      caee_prune_decide(sm, p.mode, p.flags, p.theta, p.eps, E, p.D, p.w_eff, p.part, blockIdx.x == 0, p.act, p.must, p.keep,
                        p.I_fix, p.load, p.scalars);
    STAMP(3);
    // ---- C: S5 — a token that lost an expert re-selects inside A_trans
    if (live && prunes) {
      bool bad = false;
      if (lane < k) { const int e = ir[lane]; bad = e >= 0 && !sm.keep[e]; }
      const bool affected = __any_sync(0xffffffffu, bad) || (p.flags & CAEE_COMP_ALL_TOKENS);
      if (affected) {
        const float* sc = p.scores_in ? p.scores_in : p.scores;
        caee_compensate_token<NV>(sc + (size_t)t * E, p.corr_bias != nullptr, cb, sm.keep, E, k, p.norm_topk, lane, ir, gr,
                                  (p.flags & CAEE_COMP_RANDOM) != 0, t);
        __syncwarp();
      }
    }
  }
  // publish K_final: global idx/gate rows and the membership bits
  if (live && lane < k) {
    const int e = ir[lane];
    p.idx[(size_t)t * k + lane] = e;
    p.gate[(size_t)t * k + lane] = gr[lane];
    if (e >= 0) atomicOr(M + (size_t)e * mwords + (t >> 5), 1u << (t & 31));
  }
  STAMP(4);
  if (kSingle) __syncthreads();
  else grid_barrier(p.bar + 1, G);
  STAMP(5);

  // ---- D: S6 — counts and scans per CTA, entries per token, runs/meta/stats by CTA 0
  int cnt = 0;
  if (tid < E) {
    if (kSingle) {
      cnt = __popc(s_M[tid]);
    } else {
      const uint4* row = reinterpret_cast<const uint4*>(p.M + (size_t)tid * kWords);
#pragma unroll
      for (int q = 0; q < kWords / 4; ++q) {
        const uint4 v = __ldcg(row + q);
        cnt += __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w);
      }
    }
  }
  caee_wl_scan_block(p.wl, cnt, s_est, p.resident, T, E, p.S, k, blockIdx.x == 0, s_scan);
  __syncthreads();
  STAMP(6);
  if (live) caee_wl_fill_token<kSingle>(p.wl, M, mwords, s_est, ir, gr, t, T, E, p.S, k, lane);
  if (blockIdx.x == 0 && p.stats && tid < 64)
    caee_stats_fill(p.stats, p.scalars, p.load, p.wl.meta, p.D, p.S, p.has_prune, p.bytes_per_expert, 0, tid, 64);
  if (kSingle) return;

  // ---- exit: the last CTA out clears the scratch for the next step
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_last = atomicAdd(p.bar + 2, 1) == G - 1;
  }
  __syncthreads();
  if (s_last) {
    for (int e = tid; e < E; e += kThreads) { p.acc_I[e] = 0; p.acc_act[e] = 0; p.acc_must[e] = 0; }
    for (int i = tid; i < E * kWords; i += kThreads) p.M[i] = 0;
    if (tid < 4) p.bar[tid] = 0;
  }
  STAMP(7);
}

}  // namespace

bool caee_decide_fits(const caee_ctx* c, int T) { (void)c; return T > 0 && T <= CAEE_DECIDE_MAX_TOKENS; }

size_t caee_decide_scratch_bytes(const caee_ctx* c) {
  const size_t E = c->d.E;
  return E * 8 + E + E + 16 /* align */ + E * kWords * 4 + 64;
}

bool caee_decide_splits_x(const caee_ctx* c, int T) {
  return T <= kWarps && c->kernel == CAEE_KERNEL_UMMA && c->d.w_dtype == CAEE_E4M3 && c->xq != nullptr && c->d.H % 128 == 0;
}

cudaError_t caee_launch_decide(caee_ctx* c, const float* scores_in, int T, const caee_prune_params* pp, caee_fwd_stats* stats,
                               cudaStream_t st, const void* x_split) {
  const caee_layer_desc& d = c->d;
  DecideParams p;
  p.logits = scores_in ? nullptr : c->partial;
  { int tt; caee_router_shape(c, T, &tt, &p.n_part, nullptr); }
  p.b_logit = c->b_logit; p.scores_in = scores_in; p.corr_bias = c->corr_bias;
  p.scores = c->scores; p.idx = c->idx; p.gate = c->gate;
  p.T = T; p.E = d.E; p.k = d.k; p.S = d.S; p.D = d.D; p.n_group = d.n_group; p.topk_group = d.topk_group;
  p.score_fn = d.score_fn; p.norm_topk = d.norm_topk;
  p.has_prune = pp != nullptr; p.mode = pp ? pp->mode : CAEE_PRUNE_NONE; p.flags = pp ? pp->flags : 0;
  p.theta = pp ? pp->theta : 0.0; p.eps = pp ? pp->eps : 0.0;
  p.w_eff = c->w_eff; p.part = c->part; p.resident = c->resident;
  p.act = c->act; p.must = c->must; p.keep = c->keep; p.I_fix = c->I_fix; p.load = c->load; p.scalars = c->scalars;
  p.wl = c->wl; p.n_sched = c->wl.n_tickets + c->wl.max_runs;
  p.stats = stats; p.bytes_per_expert = caee_expert_bytes(c);
  const size_t E = d.E;
  uint8_t* z = c->decide_scratch;
  p.acc_I = reinterpret_cast<unsigned long long*>(z);
  p.acc_act = z + E * 8;
  p.acc_must = z + E * 9;
  const size_t m_off = (E * 10 + 15) & ~(size_t)15;
  p.M = reinterpret_cast<uint32_t*>(z + m_off);
  p.bar = reinterpret_cast<int*>(z + m_off + E * kWords * 4);
  p.pl_experts = c->pl_experts; p.pl_start = c->pl_start; p.fast = c->part_max <= 32;
  p.split_x = nullptr; p.split_hi = p.split_lo = nullptr; p.split_scale = nullptr; p.split_blocks = 0;
  if (x_split && caee_decide_splits_x(c, T)) {
    p.split_x = (const __nv_bfloat16*)x_split;
    p.split_hi = c->xq; p.split_lo = c->xq + (size_t)d.max_tokens * d.H; p.split_scale = c->xs;
    p.split_blocks = T * (d.H / 128);
  }
  const int nv = caee_ceil_div(d.E, 32);
  void* args[] = {&p};
  ++c->n_launches;
  if (T <= kWarps) {
    // one CTA: an ordinary launch, programmatically dependent on the router GEMM (its set-up overlaps that kernel's tail)
    const void* fn = nv <= 1   ? (const void*)k_decide<1, true>
                     : nv <= 2 ? (const void*)k_decide<2, true>
                     : nv <= 4 ? (const void*)k_decide<4, true>
                     : nv <= 8 ? (const void*)k_decide<8, true>
                               : (const void*)k_decide<16, true>;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(1);
    cfg.blockDim = dim3(kThreads);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = c->pdl ? 1 : 0;
    return cudaLaunchKernelExC(&cfg, fn, args);
  }
  const void* fn = nv <= 1   ? (const void*)k_decide<1, false>
                   : nv <= 2 ? (const void*)k_decide<2, false>
                   : nv <= 4 ? (const void*)k_decide<4, false>
                   : nv <= 8 ? (const void*)k_decide<8, false>
                             : (const void*)k_decide<16, false>;
  return cudaLaunchCooperativeKernel(fn, dim3(caee_ceil_div(T, kWarps)), dim3(kThreads), args, 0, st);
}
