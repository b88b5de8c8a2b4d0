// ep.cu — expert parallelism, device side ("token dispatch ->
// expert activation -> computation -> result aggregation ... across devices", :97, :127).
//
// The data path needs no kernel of its own: a device's slice of the step is the runs of the experts it
// owns (worklist_dev.cuh builds runs for those alone), and the "result aggregation" all-to-all is fused
// into the expert kernels' epilogues, which store every o row straight into the o buffer of the token's
// home device over peer memory (caee_o_base, caee_internal.cuh).  What lives here is the explicit
// dispatch plan of a step, for inspection and for transports that want send lists: the valid
// (token, slot) entries in ascending (device, expert, token) order (reading R38) with per-device
// counts and offsets — derived from the step's expert-major work list and the owner table.
#include "caee_internal.cuh"

namespace {

__global__ void __launch_bounds__(CAEE_MAX_E) k_ep_plan(caee_worklist wl, const int32_t* __restrict__ owner, int world,
                                                        int32_t* __restrict__ counts, int32_t* __restrict__ offs,
                                                        int32_t* __restrict__ tok, int32_t* __restrict__ slot,
                                                        int32_t* __restrict__ expert) {
  __shared__ int s_cnt[CAEE_MAX_E], s_dev[CAEE_MAX_E], s_dst[CAEE_MAX_E], s_tot[CAEE_EP_MAX + 1];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  const int n_nz = wl.meta[0];      // experts with at least one entry, ascending id
  if (tid <= CAEE_EP_MAX) s_tot[tid] = 0;
  __syncthreads();
  int cnt = 0, dev = -1;
  if (tid < n_nz) {
    cnt = wl.offs[tid + 1] - wl.offs[tid];
    dev = owner[wl.expert_ids[tid]];
    atomicAdd(&s_tot[dev], cnt);
  }
  s_cnt[tid] = cnt; s_dev[tid] = dev;
  __syncthreads();
  if (tid == 0) {
    int run = 0;
    for (int d = 0; d < world; ++d) { const int c = s_tot[d]; counts[d] = c; offs[d] = run; s_tot[d] = run; run += c; }
    offs[world] = run;
  }
  __syncthreads();
  if (tid < n_nz) {
    int before = 0;       // entries of lower experts on the same device
    for (int i = 0; i < tid; ++i) before += s_dev[i] == dev ? s_cnt[i] : 0;
    s_dst[tid] = s_tot[dev] + before;
  }
  __syncthreads();
  for (int i = warp; i < n_nz; i += nwarps) {
    const int src = wl.offs[i], dst = s_dst[i], e = wl.expert_ids[i];
    for (int q = lane; q < s_cnt[i]; q += 32) {
      tok[dst + q] = wl.ent_tok[src + q];
      slot[dst + q] = wl.ent_slot[src + q];
      expert[dst + q] = e;
    }
  }
}

}  // namespace

void caee_launch_ep_plan(caee_ctx* c, const int32_t* owner_dev, int world, int32_t* counts, int32_t* offs, int32_t* tok,
                         int32_t* slot, int32_t* expert, cudaStream_t st) {
  ++c->n_launches;
  k_ep_plan<<<1, CAEE_MAX_E, 0, st>>>(c->wl, owner_dev, world, counts, offs, tok, slot, expert);
}
