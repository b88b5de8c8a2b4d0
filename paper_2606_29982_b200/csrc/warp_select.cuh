// warp_select.cuh — warp-shuffle top-k used by the router (S1) and by compensation (S5).
// A warp holds one token's E scores, expert e = lane + 32*i in register slot i.  Every
// comparison is "(value desc, expert id asc)" so that ties go to the lower index (R22),
// and gates are summed in list order with round-to-nearest fp32 adds and an IEEE divide
// so that the result is a deterministic function of the scores.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define CAEE_NONE_ID 0x7fffffff
#ifdef CAEE_DECIDE_TIMING
__device__ long long g_route_clk[16];
#define RSTAMP(i) do { if (threadIdx.x == 0 && blockIdx.x == 0) g_route_clk[i] = clock64(); } while (0)
#else
#define RSTAMP(i)
#endif

__device__ __forceinline__ bool caee_before(float va, int ia, float vb, int ib) {
  return va > vb || (va == vb && ia < ib);
}

// Order-preserving map float -> uint32 (a > b  <=>  key(a) > key(b), a == b <=> key(a) == key(b) for
// non-NaN values; -0 is folded into +0 first).  Keys of real scores are >= 1, so 0 can mean "none".
// It lets a warp take a maximum with ONE redux.sync instead of a five-step shuffle butterfly.
__device__ __forceinline__ uint32_t caee_okey(float v) {
  const uint32_t u = __float_as_uint(__fadd_rn(v, 0.0f));
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float caee_okey_inv(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// Group-limited routing: group score = sum of the two largest s' in the group; the
// topk_group best groups (ties -> lower group id) stay allowed.  Returns the per-lane slot
// mask of allowed experts.  Requires n_group <= 32.
template <int NV>
__device__ __forceinline__ uint32_t caee_group_mask(const float (&sp)[NV], uint32_t ok, int E, int n_group,
                                                    int topk_group, int lane) {
  const int gs = E / n_group;
  int grp[NV];  // group of this lane's expert in slot i (-1: not allowed)
#pragma unroll
  for (int i = 0; i < NV; ++i) grp[i] = ((ok >> i) & 1u) ? (lane + 32 * i) / gs : -1;
  float my_gscore = -INFINITY;  // lane g holds the score of group g
  if (gs == 32 && n_group <= NV) {
    // Register slot i is exactly group i.  The two largest s' of a group by two warp maxima over
    // order-preserving keys (redux.sync), written branch-free so that the NV groups' reductions
    // issue back to back; the sum of two floats does not depend on their order.  The results are
    // warp-uniform, so every lane ranks "its" group (lane g < n_group) against all of them without a
    // shuffle, and with slot == group the allowed-slot mask is the ballot of the kept groups itself.
    uint32_t key[NV], m1[NV], m2[NV];
    bool dup[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) key[i] = grp[i] >= 0 ? caee_okey(sp[i]) : 0u;
#pragma unroll
    for (int i = 0; i < NV; ++i) m1[i] = __reduce_max_sync(0xffffffffu, key[i]);
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      const unsigned eq = __ballot_sync(0xffffffffu, key[i] == m1[i]);
      dup[i] = (eq & (eq - 1u)) != 0u;                 // the maximum occurs at least twice
    }
#pragma unroll
    for (int i = 0; i < NV; ++i) m2[i] = __reduce_max_sync(0xffffffffu, key[i] == m1[i] ? 0u : key[i]);
    float gsc[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      const uint32_t second = dup[i] ? m1[i] : m2[i];
      const float a = caee_okey_inv(m1[i]), bsum = __fadd_rn(a, caee_okey_inv(second));
      gsc[i] = m1[i] == 0u ? -INFINITY : (second == 0u ? a : bsum);
    }
    float mine = -INFINITY;
#pragma unroll
    for (int i = 0; i < NV; ++i) mine = lane == i ? gsc[i] : mine;
    int before = 0;
#pragma unroll
    for (int i = 0; i < NV; ++i) before += (i < n_group) & ((gsc[i] > mine) | ((gsc[i] == mine) & (i < lane)));
    const uint32_t gsel = __ballot_sync(0xffffffffu, lane < n_group && before < topk_group);
    return gsel & ok;
  }
  // top-2 merge of two (m1 >= m2) pairs
#define CAEE_TOP2_MERGE(m1, m2, o1, o2)                   \
  do {                                                    \
    const float hi_ = fmaxf(m1, o1), lo_ = fminf(m1, o1); \
    m2 = fmaxf(lo_, fmaxf(m2, o2));                       \
    m1 = hi_;                                             \
  } while (0)
  if ((gs & 31) == 0) {
    // a register slot lies inside one group: NV independent butterflies, then merge a group's slots
    const int sg = gs >> 5;
    float a1[NV], a2[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) { a1[i] = grp[i] >= 0 ? sp[i] : -INFINITY; a2[i] = -INFINITY; }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        const float o1 = __shfl_xor_sync(0xffffffffu, a1[i], o), o2 = __shfl_xor_sync(0xffffffffu, a2[i], o);
        CAEE_TOP2_MERGE(a1[i], a2[i], o1, o2);
      }
    }
    float m1 = -INFINITY, m2 = -INFINITY;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      if (i * 32 < E) {
        if (i % sg == 0) { m1 = -INFINITY; m2 = -INFINITY; }
        CAEE_TOP2_MERGE(m1, m2, a1[i], a2[i]);
        if (i % sg == sg - 1 && lane == i / sg) my_gscore = __fadd_rn(m1, m2);
      }
    }
  } else if (gs < 32 && (gs & (gs - 1)) == 0) {
    // a group is an aligned segment of gs lanes of one slot: segmented butterflies
    const int per = 32 / gs;   // groups per slot
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      float m1 = grp[i] >= 0 ? sp[i] : -INFINITY, m2 = -INFINITY;
      for (int o = gs >> 1; o; o >>= 1) {
        const float o1 = __shfl_xor_sync(0xffffffffu, m1, o), o2 = __shfl_xor_sync(0xffffffffu, m2, o);
        CAEE_TOP2_MERGE(m1, m2, o1, o2);
      }
      const float sc = gs >= 2 ? __fadd_rn(m1, m2) : m1;
      const float v = __shfl_sync(0xffffffffu, sc, (lane % per) * gs);
      if (lane / per == i) my_gscore = v;
    }
  } else {
    for (int g = 0; g < n_group; ++g) {
      float m1 = -INFINITY, m2 = -INFINITY;
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        if (grp[i] == g) {
          float v = sp[i];
          if (v > m1) { m2 = m1; m1 = v; }
          else if (v > m2) m2 = v;
        }
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        const float o1 = __shfl_xor_sync(0xffffffffu, m1, o), o2 = __shfl_xor_sync(0xffffffffu, m2, o);
        CAEE_TOP2_MERGE(m1, m2, o1, o2);
      }
      const float sc = gs >= 2 ? __fadd_rn(m1, m2) : m1;
      if (lane == g) my_gscore = sc;
    }
  }
#undef CAEE_TOP2_MERGE
  // the topk_group best groups by (score desc, id asc): lane g counts the groups before it
  int before = 0;
  for (int g = 0; g < n_group; ++g) {
    const float og = __shfl_sync(0xffffffffu, my_gscore, g);
    before += caee_before(og, g, my_gscore, lane) ? 1 : 0;
  }
  const uint32_t gsel = __ballot_sync(0xffffffffu, lane < n_group && before < topk_group);
  uint32_t m = 0;
#pragma unroll
  for (int i = 0; i < NV; ++i)
    if (grp[i] >= 0 && ((gsel >> grp[i]) & 1u)) m |= 1u << i;
  return m;
}

// Top-k of sp over the allowed slots, listed in descending order; gates from s.
// Writes idx_out[0..k) (-1 for empty slots) and gate_out[0..k).  k <= 32.
// Each of the k rounds is: per-lane maximum over its slots (strict '>' keeps the lower slot = lower
// id on ties), one redux.sync max over the warp, one redux.sync min over the ids that hold it
// (ties -> lower id, R22), one shuffle for the winner's unbiased score.
template <int NV>
__device__ __forceinline__ void caee_warp_select(const float (&s)[NV], const float (&sp)[NV], uint32_t ok, int k,
                                                 int norm_topk, int lane, int32_t* idx_out, float* gate_out) {
  uint32_t key[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) key[i] = ((ok >> i) & 1u) ? caee_okey(sp[i]) : 0u;
  int sel_e = -1;
  float sel_s = 0.f;
  for (int j = 0; j < k; ++j) {
    // per-lane maximum as a tree; on equal keys the lower slot (= lower id) stays
    uint32_t tk[NV];
    int ti[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) { tk[i] = key[i]; ti[i] = i; }
#pragma unroll
    for (int w = 1; w < NV; w *= 2) {
#pragma unroll
      for (int i = 0; i + w < NV; i += 2 * w) {
        const bool up = tk[i + w] > tk[i];
        tk[i] = up ? tk[i + w] : tk[i];
        ti[i] = up ? ti[i + w] : ti[i];
      }
    }
    const uint32_t m = __reduce_max_sync(0xffffffffu, tk[0]);
    // m == 0: nothing left (fewer than k allowed experts) — win = 0xffffffff then matches no lane and no slot
    const uint32_t win = __reduce_min_sync(0xffffffffu, (tk[0] == m && m != 0u) ? (uint32_t)(lane + 32 * ti[0]) : 0xffffffffu);
    float mine = 0.f;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      const bool hit = win == (uint32_t)(lane + 32 * i);
      mine = hit ? s[i] : mine;
      key[i] = hit ? 0u : key[i];
    }
    const float ws = __shfl_sync(0xffffffffu, mine, win & 31);
    if (lane == j) { sel_e = (int)win; sel_s = ws; }      // 0xffffffff == -1: an empty slot
  }
  float sum = 0.f;
  for (int j = 0; j < k; ++j) {
    int ej = __shfl_sync(0xffffffffu, sel_e, j);
    float sj = __shfl_sync(0xffffffffu, sel_s, j);
    if (ej >= 0) sum = __fadd_rn(sum, sj);
  }
  if (lane < k) {
    idx_out[lane] = sel_e;
    gate_out[lane] = sel_e < 0 ? 0.f : (norm_topk ? __fdiv_rn(sel_s, sum) : sel_s);
  }
}

// One token's post-activation scores s (S0 tail): either loaded (scores_row) or computed from
// the token's logits row + b_logit: sigmoid, or softmax over the E experts (R1).
// Per-expert vector (b_logit, corr_bias) into the warp's register layout; zeros without one.
// Kernels load these first so that their (cold) latency overlaps the first score loads.
template <int NV>
__device__ __forceinline__ void caee_load_vec(const float* __restrict__ p, int E, int lane, float (&v)[NV]) {
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int e = lane + 32 * i;
    v[i] = (p && e < E) ? p[e] : 0.f;
  }
}

// logits_row: the token's row of the first split-K partial of the router GEMM; n_part partials lie
// part_stride floats apart and are added here in ascending order (a fixed order: the scores are a
// deterministic function of x and W_r whatever the schedule of the GEMM's CTAs was).
template <int NV>
__device__ __forceinline__ void caee_token_scores(const float* __restrict__ scores_row, const float* __restrict__ logits_row,
                                                  int n_part, size_t part_stride, bool has_bl, const float (&bl)[NV], int E,
                                                  int score_fn, int lane, float (&s)[NV]) {
  RSTAMP(0);
  if (scores_row) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int e = lane + 32 * i;
      s[i] = e < E ? scores_row[e] : 0.f;
    }
    return;
  }
  float l[NV];
  float mx = -INFINITY;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int e = lane + 32 * i;
    l[i] = e < E ? __ldcg(logits_row + e) : 0.f;
  }
  // four partials' loads in flight at a time, added in ascending order
  int q = 1;
  for (; q + 4 <= n_part; q += 4) {
    float v[4][NV];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const float* pr = logits_row + (size_t)(q + u) * part_stride;
#pragma unroll
      for (int i = 0; i < NV; ++i) {
        int e = lane + 32 * i;
        v[u][i] = e < E ? __ldcg(pr + e) : 0.f;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < NV; ++i) l[i] = __fadd_rn(l[i], v[u][i]);
  }
  for (; q < n_part; ++q) {
    const float* pr = logits_row + (size_t)q * part_stride;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int e = lane + 32 * i;
      if (e < E) l[i] = __fadd_rn(l[i], __ldcg(pr + e));
    }
  }
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int e = lane + 32 * i;
    if (e < E) {
      if (has_bl) l[i] += bl[i];
      mx = fmaxf(mx, l[i]);
    }
  }
  if (score_fn == 1 /* CAEE_SCORE_SIGMOID */) {
#pragma unroll
    for (int i = 0; i < NV; ++i) s[i] = 1.0f / (1.0f + expf(-l[i]));
  } else {
#pragma unroll
    for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    float den = 0.f;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      int e = lane + 32 * i;
      s[i] = e < E ? expf(l[i] - mx) : 0.f;
      den += s[i];
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) den += __shfl_xor_sync(0xffffffffu, den, o);
#pragma unroll
    for (int i = 0; i < NV; ++i) s[i] = s[i] / den;
  }
}

// S1 for one token: selection score s' = s + corr_bias, group limit, top-k, gates.
template <int NV>
__device__ __forceinline__ void caee_route_token(const float (&s)[NV], bool has_cb, const float (&cb)[NV], int E, int k,
                                                 int n_group, int topk_group, int norm_topk, int lane, int32_t* idx_out,
                                                 float* gate_out) {
  float sp[NV];
  uint32_t ok = 0;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int e = lane + 32 * i;
    sp[i] = (has_cb && e < E) ? __fadd_rn(s[i], cb[i]) : s[i];
    if (e < E) ok |= 1u << i;
  }
  RSTAMP(1);
  if (n_group > 1 && topk_group < n_group) ok &= caee_group_mask<NV>(sp, ok, E, n_group, topk_group, lane);
  RSTAMP(2);
  caee_warp_select<NV>(s, sp, ok, k, norm_topk, lane, idx_out, gate_out);
  RSTAMP(3);
}

// Counter-based uniform draw in [0,1) for (token, expert): murmur3's 32-bit finalizer over t, e and
// a fixed constant (CAEE_COMP_RANDOM, R35).
__device__ __forceinline__ float caee_unit_draw(int t, int e) {
  uint32_t h = (uint32_t)t * 0x9e3779b1u + (uint32_t)e * 0x85ebca77u + 0x26062998u;
  h ^= h >> 16; h *= 0x85ebca6bu; h ^= h >> 13; h *= 0xc2b2ae35u; h ^= h >> 16;
  return __fmul_rn((float)(h >> 8), 1.0f / 16777216.0f);
}

// S5 for one token: top-k of s' over the experts of A_trans only, no group limit (R13).
// random (CAEE_COMP_RANDOM, the ablation baseline of PAPER.md:250-256): the selection key is
// 2 + u(t,e) for a pick of idx_out that survived and u(t,e) otherwise, so the survivors stay and the
// vacated slots are filled uniformly from the rest of A_trans; gates as always from s.
template <int NV>
__device__ __forceinline__ void caee_compensate_token(const float* __restrict__ scores_row, bool has_cb, const float (&cb)[NV],
                                                      const uint8_t* keep, int E, int k, int norm_topk, int lane,
                                                      int32_t* idx_out, float* gate_out, bool random = false, int t = 0) {
  float s[NV], sp[NV];
  uint32_t ok = 0;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int e = lane + 32 * i;
    s[i] = e < E ? scores_row[e] : 0.f;
    sp[i] = (has_cb && e < E) ? __fadd_rn(s[i], cb[i]) : s[i];
    if (e < E && keep[e]) ok |= 1u << i;
  }
  if (random) {
    const int mine = lane < k ? idx_out[lane] : -1;      // the token's current picks
#pragma unroll
    for (int i = 0; i < NV; ++i) sp[i] = caee_unit_draw(t, lane + 32 * i);
    for (int j = 0; j < k; ++j) {
      const int ej = __shfl_sync(0xffffffffu, mine, j);
      if (ej >= 0 && (ej & 31) == lane) {
#pragma unroll
        for (int i = 0; i < NV; ++i)
          if (i == (ej >> 5) && ((ok >> i) & 1u)) sp[i] = __fadd_rn(2.0f, sp[i]);
      }
    }
  }
  __syncwarp();
  caee_warp_select<NV>(s, sp, ok, k, norm_topk, lane, idx_out, gate_out);
}
