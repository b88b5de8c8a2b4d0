// worklist_dev.cuh — warp-level bodies of S6 (compaction into expert-major lists and runs),
// shared by the stand-alone kernels of worklist.cu and the fused decision kernel (decide.cu).
#pragma once
#include "caee_internal.cuh"

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  return v;
}

// One warp (all 32 lanes call it): scans over experts -> compact ids/offsets, per-expert entry starts, runs.
// Run order: resident routed experts (ascending id), then the shared experts, then the
// non-resident routed experts (ascending id) — so that an offloading step can launch the
// resident part while the misses are still being fetched (meta[4] = runs in the first two groups).
__device__ __forceinline__ void caee_wl_scan_warp(const caee_worklist& wl, const int32_t* counts, int32_t* estart,
                                                  const uint8_t* __restrict__ resident, int T, int E, int S, int k, int lane) {
  int n_nz = 0, n_ent = 0;
  for (int e0 = 0; e0 < E; e0 += 32) {
    int e = e0 + lane;
    int c = e < E ? counts[e] : 0;
    int nz = c > 0;
    int s_nz = warp_incl_scan(nz, lane), s_c = warp_incl_scan(c, lane);
    if (e < E) {
      int start = n_ent + s_c - c;
      estart[e] = start;
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
      int c = (e < E && (resident[e] != 0) == (pass == 0)) ? counts[e] : 0;
      int nch = (c + CAEE_RUN_TOKENS - 1) / CAEE_RUN_TOKENS, rows = (c + 15) & ~15;
      int s_ch = warp_incl_scan(nch, lane), s_rows = warp_incl_scan(rows, lane);
      if (c > 0) {
        int start = estart[e];
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

// One warp lists expert e's (token, slot) pairs in ascending entry order (e < E), or the
// entries of shared expert e - E (every token).
__device__ __forceinline__ void caee_wl_fill_expert(const caee_worklist& wl, const int32_t* counts, const int32_t* estart,
                                                    const int32_t* idx, const float* gate, int T, int E, int S, int k, int e,
                                                    int lane) {
  const int KS = k + S, TK = T * k;
  if (e >= E) {
    int s = e - E;
    for (int t = lane; t < T; t += 32) {
      wl.ent_tok[TK + s * T + t] = t;
      wl.ent_dst[TK + s * T + t] = t * KS + k + s;
    }
    return;
  }
  if (counts[e] == 0) return;
  int pos = estart[e];
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


// caee_fwd_stats of one step (all threads of the calling group take part; nth >= 1).
__device__ __forceinline__ void caee_stats_fill(caee_fwd_stats* st, const int64_t* scalars, const int64_t* load,
                                                const int32_t* meta, int D, int S, int pruned, long long bytes_per_expert,
                                                int n_fetch, int tid, int nth) {
  if (tid == 0) {
    st->F_base = pruned ? scalars[0] : 0;
    st->F_cost_dense = pruned ? scalars[1] : 0;
    st->F_cost = pruned ? scalars[2] : 0;
    st->F_imp = pruned ? scalars[3] : 0;
    st->n_act = pruned ? (int32_t)scalars[4] : meta[0];
    st->n_keep = pruned ? (int32_t)scalars[6] : meta[0];
    st->n_run = meta[0];
    int n_sh = meta[1] > 0 ? S : 0;
    st->weight_bytes = (long long)(meta[0] + n_sh) * bytes_per_expert;
    st->n_fetch = n_fetch;
    st->h2d_bytes = (long long)n_fetch * bytes_per_expert;
  }
  for (int d = tid; d < 64; d += nth) st->load[d] = (pruned && d < D) ? load[d] : 0;
}
