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
  if (n > 0) k_wl_count<<<caee_ceil_div(n, 256), 256, 0, st>>>(idx, n, c->wl.counts);
  k_wl_scan<<<1, CAEE_MAX_E, 0, st>>>(c->wl, c->resident, T, d.E, d.S, d.k);
  k_wl_fill<<<d.E + d.S, 32, 0, st>>>(c->wl, idx, gate, T, d.E, d.S, d.k);
}

void caee_launch_export_worklist(caee_ctx* c, int T, const caee_prune_out* out, cudaStream_t st) {
  caee_prune_out o = {};
  if (out) o = *out;
  int n = T * c->d.k;
  int blocks = n > 0 ? caee_ceil_div(n, 256) : 1;
  k_wl_export<<<blocks > 64 ? 64 : blocks, 256, 0, st>>>(c->wl, o, c->d.E, c->scalars);
}
