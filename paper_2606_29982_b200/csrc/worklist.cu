// worklist.cu — S6 compaction: expert-major token lists for the experts that receive at
// least one token after compensation (BASELINE.json north_star (1)), plus the "runs" the
// expert kernels consume (<= CAEE_RUN_TOKENS tokens of one expert each; shared experts are
// appended as runs over all tokens).  Integer work only; the result is unique: experts
// ascending, tokens ascending inside an expert.
#include "caee_internal.cuh"

namespace {

__global__ void k_wl_count(const int32_t* __restrict__ idx, int n, int32_t* __restrict__ counts) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    int e = idx[i];
    if (e >= 0) atomicAdd(&counts[e], 1);
  }
}

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  return v;
}

// One warp: scans over experts -> compact ids/offsets, per-expert entry starts, runs.
// Run order: resident routed experts (ascending id), then the shared experts, then the
// non-resident routed experts (ascending id) — so that an offloading step can launch the
// resident part while the misses are still being fetched (meta[4] = runs in the first two groups).
__global__ void k_wl_scan(caee_worklist wl, const uint8_t* __restrict__ resident, int T, int E, int S, int k) {
  const int lane = threadIdx.x;
  int n_nz = 0, n_ent = 0;
  for (int e0 = 0; e0 < E; e0 += 32) {
    int e = e0 + lane;
    int c = e < E ? wl.counts[e] : 0;
    int nz = c > 0;
    int s_nz = warp_incl_scan(nz, lane), s_c = warp_incl_scan(c, lane);
    if (e < E) {
      int start = n_ent + s_c - c;
      wl.estart[e] = start;
      if (nz) {
        int pos = n_nz + s_nz - 1;
        wl.expert_ids[pos] = e;
        wl.offs[pos] = start;
      }
    }
    n_nz += __shfl_sync(0xffffffffu, s_nz, 31);
    n_ent += __shfl_sync(0xffffffffu, s_c, 31);
  }
  int n_runs = 0, n_rows = 0;
  for (int pass = 0; pass < 2; ++pass) {
    for (int e0 = 0; e0 < E; e0 += 32) {
      int e = e0 + lane;
      int c = (e < E && (resident[e] != 0) == (pass == 0)) ? wl.counts[e] : 0;
      int nch = (c + CAEE_RUN_TOKENS - 1) / CAEE_RUN_TOKENS, rows = (c + 15) & ~15;
      int s_ch = warp_incl_scan(nch, lane), s_rows = warp_incl_scan(rows, lane);
      if (c > 0) {
        int start = wl.estart[e];
        int r0 = n_runs + s_ch - nch, h0 = n_rows + s_rows - rows;
        for (int j = 0; j < nch; ++j) {
          wl.run_expert[r0 + j] = e;
          wl.run_start[r0 + j] = start + j * CAEE_RUN_TOKENS;
          wl.run_n[r0 + j] = min(CAEE_RUN_TOKENS, c - j * CAEE_RUN_TOKENS);
          wl.run_hrow[r0 + j] = h0 + j * CAEE_RUN_TOKENS;
        }
      }
      n_runs += __shfl_sync(0xffffffffu, s_ch, 31);
      n_rows += __shfl_sync(0xffffffffu, s_rows, 31);
    }
    if (pass == 0) {
      if (lane == 0 && T > 0) {
        const int TK = T * k;
        for (int s = 0; s < S; ++s)
          for (int t0 = 0; t0 < T; t0 += CAEE_RUN_TOKENS) {
            int n = min(CAEE_RUN_TOKENS, T - t0);
            wl.run_expert[n_runs] = E + s;
            wl.run_start[n_runs] = TK + s * T + t0;
            wl.run_n[n_runs] = n;
            wl.run_hrow[n_runs] = n_rows;
            n_rows += (n + 15) & ~15;
            ++n_runs;
          }
      }
      n_runs = __shfl_sync(0xffffffffu, n_runs, 0);
      n_rows = __shfl_sync(0xffffffffu, n_rows, 0);
      if (lane == 0) wl.meta[4] = n_runs;
    }
  }
  if (lane == 0) {
    wl.offs[n_nz] = n_ent;
    wl.meta[0] = n_nz;
    wl.meta[2] = n_ent;
    wl.meta[1] = n_runs;
    wl.meta[3] = n_rows;
  }
}

// Block e < E: one warp lists expert e's (token, slot) pairs in ascending entry order.
// Blocks E..E+S-1: shared expert entries (every token).
__global__ void k_wl_fill(caee_worklist wl, const int32_t* __restrict__ idx, const float* __restrict__ gate, int T, int E,
                          int S, int k) {
  const int lane = threadIdx.x, e = blockIdx.x, KS = k + S, TK = T * k;
  if (e >= E) {
    int s = e - E;
    for (int t = lane; t < T; t += 32) {
      wl.ent_tok[TK + s * T + t] = t;
      wl.ent_dst[TK + s * T + t] = t * KS + k + s;
    }
    return;
  }
  if (wl.counts[e] == 0) return;
  int pos = wl.estart[e];
  for (int i0 = 0; i0 < TK; i0 += 32) {
    int i = i0 + lane;
    bool hit = i < TK && idx[i] == e;
    unsigned b = __ballot_sync(0xffffffffu, hit);
    if (hit) {
      int p = pos + __popc(b & ((1u << lane) - 1));
      int t = i / k, j = i - t * k;
      wl.ent_tok[p] = t;
      wl.ent_slot[p] = j;
      wl.ent_wt[p] = gate[i];
      wl.ent_dst[p] = t * KS + j;
    }
    pos += __popc(b);
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
  if (n > 0) k_wl_count<<<caee_ceil_div(n, 256), 256, 0, st>>>(idx, n, c->wl.counts);
  k_wl_scan<<<1, 32, 0, st>>>(c->wl, c->resident, T, d.E, d.S, d.k);
  k_wl_fill<<<d.E + d.S, 32, 0, st>>>(c->wl, idx, gate, T, d.E, d.S, d.k);
}

void caee_launch_export_worklist(caee_ctx* c, int T, const caee_prune_out* out, cudaStream_t st) {
  caee_prune_out o = {};
  if (out) o = *out;
  int n = T * c->d.k;
  int blocks = n > 0 ? caee_ceil_div(n, 256) : 1;
  k_wl_export<<<blocks > 64 ? 64 : blocks, 256, 0, st>>>(c->wl, o, c->d.E, c->scalars);
}
