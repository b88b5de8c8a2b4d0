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


// Block-wide exclusive scan of N ints per thread (blockDim.x <= 1024, a multiple of 32).
// scratch: 33 * N ints of shared memory.  ex = sum over lower threads, tot = sum over the block.
template <int N>
__device__ __forceinline__ void caee_block_excl_scan(const int (&v)[N], int (&ex)[N], int (&tot)[N], int* scratch) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  int inc[N];
#pragma unroll
  for (int i = 0; i < N; ++i) inc[i] = warp_incl_scan(v[i], lane);
  if (lane == 31) {
#pragma unroll
    for (int i = 0; i < N; ++i) scratch[warp * N + i] = inc[i];
  }
  __syncthreads();
  if (warp == 0) {
#pragma unroll
    for (int i = 0; i < N; ++i) {
      const int w = lane < nwarps ? scratch[lane * N + i] : 0;
      const int s = warp_incl_scan(w, lane);
      if (lane < nwarps) scratch[lane * N + i] = s - w;
      if (lane == 31) scratch[32 * N + i] = s;
    }
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < N; ++i) {
    ex[i] = scratch[warp * N + i] + inc[i] - v[i];
    tot[i] = scratch[32 * N + i];
  }
  __syncthreads();
}

// S6 scans for a whole CTA (blockDim.x >= E): thread e owns expert e.  Fills estart[e] (shared
// or global) and, with `write`, the compact ids/offsets, the runs and meta of wl.
// Run order: resident routed experts (ascending id), then the shared experts, then the
// non-resident routed experts (ascending id) — so that an offloading step can launch the
// resident part while the misses are still being fetched (meta[4] = runs in the first two groups).
__device__ __forceinline__ void caee_wl_scan_block(const caee_worklist& wl, int count_e, int32_t* estart,
                                                   const uint8_t* __restrict__ resident, int T, int E, int S, int k, bool write,
                                                   int* scratch /* 33 * 6 ints */) {
  const int e = threadIdx.x, cap = wl.run_cap;   // tokens per run (a multiple of 16)
  const int c = e < E ? count_e : 0;
  const bool res = e < E && resident[e] != 0;
  // expert parallelism: the lists hold every entry, runs exist only for the experts this device owns
  const int cr = (e < E && wl.ep_owned && !wl.ep_owned[e]) ? 0 : c;
  const int t_lo = wl.ep_owned ? min(wl.ep_tlo, T) : 0, Th = (wl.ep_owned ? min(wl.ep_thi, T) : T) - t_lo;   // home tokens
  const int nch = (cr + cap - 1) / cap, rows = (cr + 15) & ~15;
  const int v[6] = {c > 0, c, res ? nch : 0, res ? rows : 0, res ? 0 : nch, res ? 0 : rows};
  int ex[6], tot[6];
  caee_block_excl_scan<6>(v, ex, tot, scratch);
  if (e < E) estart[e] = ex[1];
  if (!write) return;
  const int sh_chunks = Th > 0 ? (Th + cap - 1) / cap : 0;
  const int sh_runs = S * sh_chunks;
  int sh_rows_each = 0;   // h rows of one shared expert: every chunk padded to 16
  for (int t0 = 0; t0 < Th; t0 += cap) sh_rows_each += (min(cap, Th - t0) + 15) & ~15;
  if (c > 0) {
    wl.expert_ids[ex[0]] = e;
    wl.offs[ex[0]] = ex[1];
    const int r0 = res ? ex[2] : tot[2] + sh_runs + ex[4];
    const int h0 = res ? ex[3] : tot[3] + S * sh_rows_each + ex[5];
    CAEE_DEV_ASSERT(r0 + nch <= wl.max_runs && h0 + rows <= wl.hrow_cap && ex[1] + c <= wl.ent_cap);
    for (int j = 0; j < nch; ++j) {
      wl.run_expert[r0 + j] = e;
      wl.run_start[r0 + j] = ex[1] + j * cap;
      wl.run_n[r0 + j] = min(cap, cr - j * cap);
      wl.run_hrow[r0 + j] = h0 + j * cap;
    }
  }
  for (int i = e; i < sh_runs; i += blockDim.x) {   // shared-expert runs over all (home) tokens
    const int s = i / sh_chunks, j = i - s * sh_chunks, t0 = j * cap;
    const int r = tot[2] + i;
    CAEE_DEV_ASSERT(r < wl.max_runs && tot[3] + s * sh_rows_each + j * cap + ((min(cap, Th - t0) + 15) & ~15) <= wl.hrow_cap);
    wl.run_expert[r] = E + s;
    wl.run_start[r] = T * k + s * T + t_lo + t0;
    wl.run_n[r] = min(cap, Th - t0);
    wl.run_hrow[r] = tot[3] + s * sh_rows_each + j * cap;
  }
  if (e == 0) {
    wl.offs[tot[0]] = tot[1];
    wl.meta[0] = tot[0];
    wl.meta[1] = tot[2] + sh_runs + tot[4];
    wl.meta[2] = tot[1];
    wl.meta[3] = tot[3] + S * sh_rows_each + tot[5];
    wl.meta[4] = tot[2] + sh_runs;
  }
}

// Decode-size fill (T <= 256): M is the E x W bit matrix "expert e is in K_final of token t"
// (W = 8 words per expert), so an entry's place in its expert's list is a popcount.
// One warp, one token: lanes j < k place the token's routed entries, lanes s < S the shared ones.
// kShared: M lives in shared memory (the one-CTA step), else in global memory behind a grid barrier.
template <bool kShared>
__device__ __forceinline__ void caee_wl_fill_token(const caee_worklist& wl, const uint32_t* M, int W, const int32_t* estart,
                                                   const int32_t* ir, const float* gr, int t, int T, int E, int S, int k,
                                                   int lane) {
  const int KS = k + S, TK = T * k;
  if (lane < k) {
    const int e = ir[lane];
    if (e >= 0) {
      const uint32_t* row = M + (size_t)e * W;
      int pos = estart[e];
      for (int w = 0; w < (t >> 5); ++w) pos += __popc(kShared ? row[w] : __ldcg(row + w));
      pos += __popc((kShared ? row[t >> 5] : __ldcg(row + (t >> 5))) & ((1u << (t & 31)) - 1u));
      CAEE_DEV_ASSERT(pos >= 0 && pos < TK && e < E);
      wl.ent_tok[pos] = t;
      wl.ent_slot[pos] = lane;
      wl.ent_wt[pos] = gr[lane];
      wl.ent_dst[pos] = t * KS + lane;
    }
  }
  if (lane < S) {
    wl.ent_tok[TK + lane * T + t] = t;
    wl.ent_dst[TK + lane * T + t] = t * KS + k + lane;
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
