// worklist.cu — S6 compaction: expert-major token lists for the experts that receive at
// least one token after compensation (BASELINE.json north_star (1)), plus the "runs" the
// expert kernels consume (<= CAEE_RUN_TOKENS tokens of one expert each; shared experts are
// appended as runs over all tokens).  Integer work only; the result is unique: experts
// ascending, tokens ascending inside an expert.
#include "caee_internal.cuh"
#include "worklist_dev.cuh"

namespace {

__global__ void k_wl_count(const int32_t* __restrict__ idx, int n, int32_t* __restrict__ counts) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    int e = idx[i];
    if (e >= 0) atomicAdd(&counts[e], 1);
  }
}

__global__ void __launch_bounds__(CAEE_MAX_E) k_wl_scan(caee_worklist wl, const uint8_t* __restrict__ resident, int T, int E,
                                                        int S, int k) {
  __shared__ int scratch[33 * 6];
  caee_wl_scan_block(wl, threadIdx.x < E ? wl.counts[threadIdx.x] : 0, wl.estart, resident, T, E, S, k, true, scratch);
}

__global__ void k_wl_fill(caee_worklist wl, const int32_t* __restrict__ idx, const float* __restrict__ gate, int T, int E,
                          int S, int k) {
  caee_wl_fill_expert(wl, wl.counts, wl.estart, idx, gate, T, E, S, k, blockIdx.x, threadIdx.x);
}

// Large steps (T k > kFillSeg entries): block b owns entries [kFillSeg b, kFillSeg b + kFillSeg).
// k_wl_hist counts them per expert (hist[b][e], and the totals counts[e]); after the scan,
// k_wl_fill_seg places every entry at estart[e] + (entries of e in lower blocks) + (its rank among
// the block's entries of e) — ascending entry order inside an expert, as the warp-per-expert fill.
constexpr int kFillSeg = 256;

__global__ void __launch_bounds__(kFillSeg) k_wl_hist(const int32_t* __restrict__ idx, int n, int E, int32_t* __restrict__ counts,
                                                      int32_t* __restrict__ hist) {
  extern __shared__ int h[];
  for (int e = threadIdx.x; e < E; e += kFillSeg) h[e] = 0;
  __syncthreads();
  const int i = blockIdx.x * kFillSeg + threadIdx.x;
  if (i < n) {
    const int e = idx[i];
    if (e >= 0) atomicAdd(&h[e], 1);
  }
  __syncthreads();
  for (int e = threadIdx.x; e < E; e += kFillSeg) {
    const int v = h[e];
    hist[(size_t)blockIdx.x * E + e] = v;
    if (v) atomicAdd(&counts[e], v);
  }
}

__global__ void __launch_bounds__(kFillSeg) k_wl_fill_seg(caee_worklist wl, const int32_t* __restrict__ idx,
                                                          const float* __restrict__ gate, int T, int E, int S, int k,
                                                          const int32_t* __restrict__ hist) {
  extern __shared__ int sm[];
  int* base = sm;        // [E] first list position of this block's entries of expert e
  int* wc = sm + E;      // [kFillSeg / 32][E] entries of e per warp of this block
  const int b = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int KS = k + S, TK = T * k;
  for (int e = threadIdx.x; e < E; e += kFillSeg) {
    int s = wl.estart[e];
    for (int bb = 0; bb < b; ++bb) s += hist[(size_t)bb * E + e];
    base[e] = s;
  }
  for (int i = threadIdx.x; i < (kFillSeg / 32) * E; i += kFillSeg) wc[i] = 0;
  __syncthreads();
  const int i = b * kFillSeg + threadIdx.x;
  const int e = i < TK ? idx[i] : -1;
  const unsigned m = __match_any_sync(0xffffffffu, e);
  const int rank = __popc(m & ((1u << lane) - 1u));
  if (e >= 0 && rank == 0) wc[warp * E + e] = __popc(m);
  __syncthreads();
  if (e >= 0) {
    int pos = base[e] + rank;
    for (int w = 0; w < warp; ++w) pos += wc[w * E + e];
    const int t = i / k, j = i - t * k;
    wl.ent_tok[pos] = t;
    wl.ent_slot[pos] = j;
    wl.ent_wt[pos] = gate[i];
    wl.ent_dst[pos] = t * KS + j;
  }
  // shared experts: every token, in token order
  for (int q = blockIdx.x * kFillSeg + threadIdx.x; q < S * T; q += gridDim.x * kFillSeg) {
    const int s = q / T, t = q - s * T;
    wl.ent_tok[TK + q] = t;
    wl.ent_dst[TK + q] = t * KS + k + s;
  }
}

__global__ void k_wl_export(caee_worklist wl, caee_prune_out out, int E, int64_t* scalars) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  const int n_nz = wl.meta[0], n_ent = wl.meta[2];
  if (tid == 0) {
    if (out.n_run) *out.n_run = n_nz;
    if (scalars) scalars[7] = n_nz;
  }
  for (int i = tid; i <= n_nz; i += nth) {
    if (out.offs) out.offs[i] = wl.offs[i];
    if (out.expert_ids && i < n_nz) out.expert_ids[i] = wl.expert_ids[i];
  }
  for (int i = tid; i < n_ent; i += nth) {
    if (out.tok) out.tok[i] = wl.ent_tok[i];
    if (out.slot) out.slot[i] = wl.ent_slot[i];
    if (out.wt) out.wt[i] = wl.ent_wt[i];
  }
}

}  // namespace

void caee_launch_worklist(caee_ctx* c, int T, const int32_t* idx, const float* gate, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  cudaMemsetAsync(c->wl.counts, 0, sizeof(int32_t) * d.E, st);
  cudaMemsetAsync(c->wl.sched, 0, sizeof(int32_t) * (c->wl.n_tickets + c->wl.max_runs), st);
  int n = T * d.k;
  c->n_launches += n > 0 ? 3 : 2;   // the two memsets are copy-engine work, not kernels of ours
  if (n > 4096 && c->wl_hist) {
    const int nb = caee_ceil_div(n, kFillSeg);
    k_wl_hist<<<nb, kFillSeg, sizeof(int) * d.E, st>>>(idx, n, d.E, c->wl.counts, c->wl_hist);
    k_wl_scan<<<1, CAEE_MAX_E, 0, st>>>(c->wl, c->resident, T, d.E, d.S, d.k);
    k_wl_fill_seg<<<nb, kFillSeg, sizeof(int) * d.E * (1 + kFillSeg / 32), st>>>(c->wl, idx, gate, T, d.E, d.S, d.k, c->wl_hist);
    return;
  }
  if (n > 0) k_wl_count<<<caee_ceil_div(n, 256), 256, 0, st>>>(idx, n, c->wl.counts);
  k_wl_scan<<<1, CAEE_MAX_E, 0, st>>>(c->wl, c->resident, T, d.E, d.S, d.k);
  k_wl_fill<<<d.E + d.S, 32, 0, st>>>(c->wl, idx, gate, T, d.E, d.S, d.k);
}

size_t caee_wl_hist_ints(const caee_ctx* c) {
  const size_t n = (size_t)c->d.max_tokens * c->d.k;
  return n > 4096 ? (size_t)caee_ceil_div((int)n, kFillSeg) * c->d.E : 0;
}

void caee_launch_export_worklist(caee_ctx* c, int T, const caee_prune_out* out, cudaStream_t st) {
  caee_prune_out o = {};
  if (out) o = *out;
  int n = T * c->d.k;
  int blocks = n > 0 ? caee_ceil_div(n, 256) : 1;
  ++c->n_launches;
  k_wl_export<<<blocks > 64 ? 64 : blocks, 256, 0, st>>>(c->wl, o, c->d.E, c->scalars);
}
