/* caee.h — C ABI of libcaee: the CAEE (Cost-Aware Expert Execution) per-layer MoE
 * decode hot path on one NVIDIA B200 (sm_100a).
 *
 * Citations are to /root/reference/PAPER.md ("PAPER.md:<line>") and to the readings
 * R1..R40 listed in DESIGN.md §3.  The paper's "devices" are logical expert
 * partitions on one GPU whose costs are aggregated by max.
 *
 * Conventions
 *  - "dev" pointers are CUDA device memory on the context's device; "host" pointers
 *    are ordinary host memory read during the call; "pinned" is page-locked host memory.
 *  - Matrices are row-major and dense.  bf16 is the upper 16 bits of an IEEE fp32;
 *    e4m3 is OCP FP8 E4M3 (no infinities, max 448) with one fp32 scale per 128x128
 *    block, scales stored row-major [ceil(rows/128), ceil(cols/128)].
 *  - Ownership: the caller owns every buffer it passes.  Activations, scores and
 *    outputs are borrowed for the duration of the enqueued work; router weights,
 *    expert weights (unless packed, see caee_set_weights) and tables are borrowed
 *    until caee_destroy or the next caee_set_* call for the same item.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *    caee_route, caee_route_from_scores, caee_prune, caee_moe_forward and
 *    caee_moe_forward_from_scores only enqueue work: no host synchronisation, no
 *    allocation.  One exception: when some experts are non-resident (caee_set_residency),
 *    caee_moe_forward* waits once for its own decision kernels, because the host must learn
 *    which non-resident experts survived pruning before it can issue their copies
 *    ("transfer engine").  caee_calibrate_cost and the caee_set_* calls synchronise.
 *  - Errors: every call returns CAEE_OK (0) or a negative code; nothing throws or
 *    aborts across the ABI.  caee_last_error gives a human-readable reason.
 *    A CUDA failure is sticky for the context (CAEE_ECUDA from then on).
 *  - There is no CPU fallback: on a device that is not compute capability 10.x
 *    caee_create fails with CAEE_EUNSUPPORTED.
 *  - Determinism: idx, gate, keep/must masks, the compacted lists and all F_* values are
 *    deterministic functions of the fp32 scores; y is deterministic as well (the
 *    combine sums each token's experts in list order).
 */
#ifndef CAEE_H_
#define CAEE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct caee_ctx caee_ctx; /* opaque; one per MoE layer */
typedef int32_t caee_status;

enum {
  CAEE_OK = 0,
  CAEE_EINVAL = -1,       /* null pointer, negative size, k > E, E % n_group != 0, theta out of range ... */
  CAEE_ESHAPE = -2,       /* T > max_tokens, shape the chosen expert kernel cannot tile */
  CAEE_EDTYPE = -3,       /* unknown / unsupported dtype combination */
  CAEE_ENOMEM = -4,       /* device or host allocation failed */
  CAEE_ECUDA = -5,        /* CUDA runtime error (sticky) */
  CAEE_ESTATE = -6,       /* call made before the state it needs was set */
  CAEE_EUNSUPPORTED = -7  /* not an sm_100 device */
};

enum { CAEE_F32 = 0, CAEE_BF16 = 1, CAEE_E4M3 = 2 };
enum { CAEE_SCORE_SOFTMAX = 0, CAEE_SCORE_SIGMOID = 1 };

/* How the mandatory set A_must of step 1 is formed. */
enum {
  CAEE_PRUNE_NONE = 0,   /* A_must = A_act: nothing can be pruned                                    */
  CAEE_PRUNE_THRESH = 1, /* I(e) = sum_t G(t)_e >= theta        (on-device setup)  */
  CAEE_PRUNE_CIR = 2,    /* per token, minimal m* with CIR(m*) >= theta (offloading)    */
  CAEE_PRUNE_RANK = 3,   /* per token, the first k - theta of K_t    (BASELINE.json config 1 budget) */
                         /* CIR, RANK and KEEP_TOP1 see K_t "sorted by their gating scores":
                            by (gate descending, expert id ascending), R36 — not in the route's list order,
                            which is by the biased selection score                                       */
  CAEE_PRUNE_FRAC = 4    /* all but the floor(theta*|A_act|) least important (config 4 budget)       */
};
enum {
  CAEE_COMP_ALL_TOKENS = 1, /* re-select every token, not only those that lost an expert (R14)       */
  CAEE_KEEP_TOP1 = 2,       /* every token's first expert is mandatory (R23)                          */
  CAEE_COMP_RANDOM = 4,     /* ablation baseline of PAPER.md:250-256 / Fig. 9 (R35): an affected token
                               keeps its surviving picks and fills the vacated slots uniformly at random
                               from the rest of A_trans (counter-based draws, reproducible)            */
  CAEE_IMP_BOUND = 8        /* enforce the objective's constraint F_imp(X) <= eps (R37):
                               after the cost-invariant expansion, while the pruned importance exceeds
                               eps the pruned expert of largest I(e) (ties -> lower id) returns to A_trans;
                               F_cost may then exceed F_base and is reported as it is                  */
};
enum { CAEE_KERNEL_AUTO = 0, CAEE_KERNEL_SIMT = 1, CAEE_KERNEL_UMMA = 2 };

typedef struct caee_layer_desc {
  int32_t H;             /* hidden size                                                          */
  int32_t I;             /* SwiGLU intermediate size                                             */
  int32_t E;             /* routed experts, 1..512                                               */
  int32_t S;             /* shared experts (run on every token, gate 1, never pruned; R21)       */
  int32_t k;             /* experts per token, 1..min(E,32)                                      */
  int32_t n_group;       /* router groups, divides E; 1 = ungrouped                              */
  int32_t topk_group;    /* groups kept per token, 1..n_group; topk_group*(E/n_group) >= k       */
  int32_t score_fn;      /* CAEE_SCORE_*                                                         */
  int32_t norm_topk;     /* 1: G = s/sum_{K_t} s; 0: G = s                          */
  float routed_scale;    /* factor on the routed sum in the combine (R2)                         */
  int32_t act_dtype;     /* CAEE_F32 or CAEE_BF16: dtype of x and y                              */
  int32_t w_dtype;       /* CAEE_F32, CAEE_BF16 or CAEE_E4M3: dtype of expert weights            */
  int32_t D;             /* expert partitions, 1..64                                             */
  int32_t max_tokens;    /* largest T any call will pass; scratch is sized from it               */
  int32_t expert_kernel; /* CAEE_KERNEL_*: AUTO = UMMA (tcgen05) where it applies, else SIMT     */
  int32_t device;        /* CUDA device ordinal, -1 = current device                             */
} caee_layer_desc;

/* Per-expert weight pointers: host arrays of E+S entries, routed experts first, then the
 * shared ones.  gate/up: [I,H]; down: [H,I]; *_scale (e4m3 only, else may be NULL):
 * [ceil(rows/128), ceil(cols/128)] fp32.  Entries point to device memory or to pinned
 * (device-accessible) host memory; with pack != 0 the library's own image of an expert with
 * resident[e] == 0 (caee_set_residency) is kept in pinned host memory wherever the caller's
 * copy was. */
typedef struct caee_expert_weights {
  const void* const* gate;
  const void* const* up;
  const void* const* down;
  const float* const* gate_scale;
  const float* const* up_scale;
  const float* const* down_scale;
} caee_expert_weights;

typedef struct caee_prune_params {
  int32_t mode;  /* CAEE_PRUNE_*                                                                  */
  int32_t flags; /* CAEE_COMP_ALL_TOKENS | CAEE_KEEP_TOP1 | CAEE_COMP_RANDOM | CAEE_IMP_BOUND     */
  double theta;  /* THRESH: theta in gate units (sum G = 1); CIR: theta_imp in (0,1];
                    RANK: budget b in 0..k; FRAC: p in [0,1]                                     */
  double eps;    /* with CAEE_IMP_BOUND: bound on F_imp = sum of pruned I(e), in gate units
                    (sum_e I(e) = T), in [0, 1e6]; ignored otherwise                              */
} caee_prune_params;

/* Optional device outputs of caee_prune; any pointer may be NULL.  scalars[8] =
 * { F_base, F_cost_dense = F_cost(A_act), F_cost = F_cost(A_trans), F_imp (2^-40 units),
 *   |A_act|, |A_must| after step 1, |A_trans|, n_run }. */
typedef struct caee_prune_out {
  uint8_t* act;         /* dev [E]   A_act                                                        */
  uint8_t* must;        /* dev [E]   A_must of step 1                                             */
  uint8_t* keep;        /* dev [E]   A_trans                                                      */
  int64_t* importance;  /* dev [E]   I(e) in units of 2^-40                                       */
  int64_t* load;        /* dev [D]   per-partition cost of A_trans                                */
  int64_t* scalars;     /* dev [8]                                                                */
  int32_t* n_run;       /* dev [1]   experts that receive >= 1 token after compensation           */
  int32_t* expert_ids;  /* dev [E]   those experts, ascending                                     */
  int32_t* offs;        /* dev [E+1] start of each expert's token list                            */
  int32_t* tok;         /* dev [T*k] token of each list entry, ascending inside an expert         */
  int32_t* slot;        /* dev [T*k] position of that expert in the token's K_final               */
  float* wt;            /* dev [T*k] gate G(t)_e of the entry                                     */
} caee_prune_out;

/* Written by caee_moe_forward when stats != NULL (device memory). */
typedef struct caee_fwd_stats {
  int64_t F_base, F_cost_dense, F_cost, F_imp;
  int64_t weight_bytes; /* expert-weight bytes the expert kernel streamed (surviving + shared)   */
  int64_t h2d_bytes;    /* bytes fetched from pinned host memory for non-resident survivors      */
  int32_t n_act, n_keep, n_run, n_fetch;
  int64_t load[64];     /* per-partition cost of A_trans (the quantity of PAPER.md Fig. 10)       */
} caee_fwd_stats;

typedef struct caee_calib_opts {
  int32_t n_sizes;      /* sizes to time per tier, 2..16 (0 = default 6)                          */
  int32_t iters;        /* timed repetitions per size (0 = default 10), median is used            */
  int64_t min_bytes;    /* smallest transfer (0 = default 4 MiB)                                  */
  int64_t max_bytes;    /* largest transfer (0 = one expert's weight bytes)                       */
  int32_t apply;        /* 1: fill the context's cost table from the fits                         */
  int32_t reserved;
} caee_calib_opts;

/* t = slope*bytes + intercept, the fitted form of C~(e,d) = alpha_d*S_e/B_d + beta_d
 * (PAPER.md:139): slope = alpha_d/B_d, intercept = beta_d. */
typedef struct caee_cost_fit {
  double slope_ns_per_byte;
  double intercept_ns;
  double r2;
  double gbytes_per_s;  /* 1/slope, the effective bandwidth                                       */
  int32_t n_points;
  int32_t valid;        /* 0 if the tier could not be measured                                    */
} caee_cost_fit;

/* Lifecycle.  caee_create validates the descriptor and allocates all scratch. */
caee_status caee_create(const caee_layer_desc* desc, caee_ctx** out);
caee_status caee_destroy(caee_ctx* ctx);
/* Reason for the last failure on ctx (or, with ctx == NULL, of the last failed caee_create
 * on this thread).  The string is owned by the library and valid until the next call. */
const char* caee_last_error(const caee_ctx* ctx);

/* Router parameters (dev, fp32).  W_r [E,H]; b_logit [E] or NULL (added to the logit);
 * corr_bias [E] or NULL (added to the score for SELECTION only, R1).  Steps of fewer than 64 tokens
 * read W_r in place (fp32 FMAs); for larger steps (bf16 activations, E a multiple of 16 up to 256,
 * H a multiple of 64) this call also makes the library's own copy of W_r as three bf16 terms
 * (hi + mid + lo = W_r exactly) for the tensor-core router GEMM: fp32 accumulation of exact products,
 * scores within the same 1e-5 relative bound.  Call it again after changing W_r. */
caee_status caee_set_router(caee_ctx* ctx, const float* W_r, const float* b_logit, const float* corr_bias);
/* Expert weights.  pack != 0: the library repacks each expert once into its own tile-major
 * copy (device memory for resident experts; pinned host memory for non-resident ones, which share
 * a ring of 8 device staging slots) and no longer refers to the caller's buffers
 * afterwards.  The UMMA kernel (bf16 or e4m3 weights with bf16 activations) requires
 * pack != 0; the SIMT kernel reads the caller's buffers in place and needs every expert in
 * device memory.  The e4m3 UMMA kernel feeds the e4m3 codes to the tensor cores as they are and
 * carries each activation (x and the SwiGLU intermediate) as two e4m3 terms with one fp32 scale per
 * (token, 128-wide block): about 2^-8 relative error per activation, fp32 accumulation, the
 * 128x128 weight block scales applied in fp32.  Steps of more than 128 tokens take the e4m3
 * converter kernel instead: weights widened to fp16 with the block scale folded in (one rounding
 * to 11 bits) and fed to the tensor cores from tensor memory, x and the SwiGLU intermediate as
 * fp16 (x exact for 6.1e-5 <= |x| <= 65504, clamped above; h clamped likewise), fp32 accumulation
 * over the whole k range.
 * Call caee_set_residency first when some experts live in host memory (changing the
 * residency afterwards invalidates the weights: set them again). */
caee_status caee_set_weights(caee_ctx* ctx, const caee_expert_weights* w, int32_t pack);
/* E_d of PAPER.md:127 as part_of_expert[e] in 0..D-1 (host).  Default: contiguous blocks. */
caee_status caee_set_partitions(caee_ctx* ctx, const int32_t* part_of_expert, int32_t D);
/* R(e,d) of PAPER.md:129-135 as resident[e] in {0,1} (host).  Default: all resident. */
caee_status caee_set_residency(caee_ctx* ctx, const uint8_t* resident);
/* C~(e,d) in integer ns for each tier (host, [E] each): the cost of expert e is
 * resident[e] ? ticks_resident[e] : ticks_miss[e]  (R18).  ticks_miss may be NULL if all
 * experts are resident. */
caee_status caee_set_cost_table(caee_ctx* ctx, const int64_t* ticks_resident, const int64_t* ticks_miss);

/* Offline calibration: times streaming reads of HBM (fit[0]) and
 * pinned-host -> device copies (fit[1]) at several sizes, least-squares fits
 * t = slope*bytes + intercept, and with opts->apply fills the cost table with
 * round(slope*S_e + intercept) ns per tier.  Blocking.  opts may be NULL (defaults, apply=1). */
caee_status caee_calibrate_cost(caee_ctx* ctx, const caee_calib_opts* opts, caee_cost_fit out_fit[2]);
/* The points the last caee_calibrate_cost on this context timed for tier 0 (HBM) or 1 (H2D): transfer
 * sizes in bytes and the median duration of each in ns (host arrays of capacity cap), their number in
 * *n_out (0 if the tier was not measured).  They are exactly what the fit was computed from, so a
 * caller can check the least squares of PAPER.md:139 independently. */
caee_status caee_calibrate_points(const caee_ctx* ctx, int32_t tier, int32_t cap, double* bytes, double* ns,
                                  int32_t* n_out);
/* The cost table in force (host arrays [E]; either may be NULL): as set by caee_set_cost_table or
 * applied by caee_calibrate_cost, ticks = llround(slope * S_e + intercept) per tier (clamped at 0),
 * S_e = 3*H*I*sizeof(w) + the e4m3 block scales. */
caee_status caee_get_cost_table(const caee_ctx* ctx, int64_t* ticks_resident, int64_t* ticks_miss);

/* S0+S1: scores s = act(x W_r^T + b_logit) and the top-k set K_t with gates.
 * x dev [T,H] act dtype; scores dev [T,E] fp32 or NULL; idx dev [T,k] int32 in descending
 * selection score; gate dev [T,k] fp32. */
caee_status caee_route(caee_ctx* ctx, const void* x, int32_t T, float* scores, int32_t* idx, float* gate,
                       void* stream);
/* caee_route WITHOUT a context and without any allocation (S0+S1): for callers that cannot call
 * cudaMalloc — code under CUDA graph capture, tight serving loops, harnesses that forbid it.  caee_create allocates
 * the router's split-K scratch (ks x T x E fp32 partial logits) with cudaMalloc; this call runs the same router GEMM
 * (the fp32-FMA kernels of router.cu at every T: the tensor-core router needs a packed image of W_r) and the same
 * top-k kernel with that scratch in ONE file-scope device array of CAEE_ROUTE_NOALLOC_SCRATCH_FLOATS floats
 * (2 MiB, held by every GPU that loads the library until the process exits).  It calls no cudaMalloc / cudaFree
 * and no allocating library routine, only enqueues work on `stream`, and never synchronises.
 *   device: CUDA ordinal, -1 = the current device.  x dev [T,H] act_dtype (CAEE_F32 or CAEE_BF16), Wr dev [E,H]
 *   fp32, both 16-byte aligned; b_logit, corr_bias dev [E] fp32 or NULL; scores dev [T,E] fp32 or NULL; idx dev [T,k]
 *   int32; gate dev [T,k] fp32.  H a positive multiple of 8; E, k, n_group, topk_group, score_fn, norm_topk as in
 *   caee_layer_desc.  Results are bit-identical to caee_route on a context of the same shape while that one uses the
 *   FMA router (T < 64); from 64 tokens on caee_route's tensor-core scores agree to 1e-5 relative.
 * Limits: T <= CAEE_ROUTE_NOALLOC_MAX_TOKENS and ks * T * E <= CAEE_ROUTE_NOALLOC_SCRATCH_FLOATS (ks = the split
 * the router picks for T, at most H/128) — beyond either the call returns CAEE_ESHAPE and enqueues nothing;
 * caee_last_error(NULL) gives the reason, as for caee_create.
 * Sharing: every call on a device uses the same array, which keeps the last call's contents.  Nothing in it has to
 * start at zero (the GEMM writes every partial the top-k kernel reads), but calls that OVERLAP on the GPU — two
 * streams, or two host threads enqueueing on different streams — race on it: keep them on one stream or order them
 * with events.  Contexts are not affected (they own their scratch). */
#define CAEE_ROUTE_NOALLOC_SCRATCH_FLOATS (1 << 19)
#define CAEE_ROUTE_NOALLOC_MAX_TOKENS 128
caee_status caee_route_noalloc(int32_t device, const void* x, int32_t act_dtype, const float* Wr, const float* b_logit,
                               const float* corr_bias, int32_t T, int32_t H, int32_t E, int32_t k, int32_t n_group,
                               int32_t topk_group, int32_t score_fn, int32_t norm_topk, float* scores, int32_t* idx,
                               float* gate, void* stream);
/* S1 only, on caller-supplied scores (parity entry point). */
caee_status caee_route_from_scores(caee_ctx* ctx, const float* scores, int32_t T, int32_t* idx, float* gate,
                                   void* stream);
/* S2-S6: activation set, importance, cost-aware pruning, compensation
 * and compaction.  scores dev [T,E]; idx/gate dev [T,k] in/out: on return
 * they hold K_final and its gates (empty slots: idx -1, gate 0).  p == NULL or mode NONE
 * prunes nothing.  out may be NULL. */
caee_status caee_prune(caee_ctx* ctx, const caee_prune_params* p, const float* scores, int32_t T, int32_t* idx,
                       float* gate, const caee_prune_out* out, void* stream);
/* The whole layer: route -> prune (p != NULL) -> fetch of surviving non-resident experts on
 * a side stream (one cudaMemcpyAsync per surviving miss, overlapped with the resident experts'
 * compute; stats->n_fetch / h2d_bytes count them) -> grouped SwiGLU FFN over the surviving
 * experts only -> combine
 *   y_t = routed_scale * sum_{e in K_final} G(t)_e E_e(t) + sum_shared E_sh(t).
 * x, y dev [T,H] act dtype, 16-byte aligned; stats dev or NULL. */
caee_status caee_moe_forward(caee_ctx* ctx, const void* x, int32_t T, const caee_prune_params* p, void* y,
                             caee_fwd_stats* stats, void* stream);
/* Same, with the router's scores supplied by the caller (dev [T,E] fp32) instead of
 * computed from x: used to compare against the oracle without near-tie routing flips. */
caee_status caee_moe_forward_from_scores(caee_ctx* ctx, const void* x, const float* scores, int32_t T,
                                         const caee_prune_params* p, void* y, caee_fwd_stats* stats,
                                         void* stream);
/* The same step with HOST buffers (x_host, y_host: [T,H] act_dtype, pinned memory for the copies
 * to be asynchronous).  The library copies x into one of two device staging tensors on its own
 * copy-in stream, runs caee_moe_forward on `stream`, and copies y back on its copy-out stream; the
 * staging tensors are double-buffered, so the copies of neighbouring steps overlap the compute.
 * Enqueue-only like caee_moe_forward: x_host must stay unchanged until its copy has run and
 * y_host is complete only after caee_host_flush(ctx, stream) — which makes `stream` wait for
 * every outstanding copy-out — and a synchronisation of `stream`.  Contexts with an expert cache
 * or offloaded experts synchronise `stream` inside the step as caee_moe_forward does. */
caee_status caee_moe_forward_host(caee_ctx* ctx, const void* x_host, int32_t T, const caee_prune_params* p,
                                  void* y_host, caee_fwd_stats* stats, void* stream);
caee_status caee_host_flush(caee_ctx* ctx, void* stream);
/* Kernels of this library that the per-step calls (caee_route*, caee_prune, caee_moe_forward*) have
 * enqueued on this context since it was created (host counter, incremented at each launch site). */
caee_status caee_launch_count(const caee_ctx* ctx, int64_t* n_out);
/* K_final of the last forward call on this context (dev -> dev copy, enqueued on stream). */
caee_status caee_last_routing(caee_ctx* ctx, int32_t T, int32_t* idx, float* gate, void* stream);

/* Optional per-kernel timing for measurement (bench.py's roofline): with n_slots > 0 every
 * following caee_moe_forward* records a CUDA-event pair around its expert kernel on the
 * call's stream, into slot 0, 1, ... (further calls are not recorded once the slots are
 * used up); n_slots == 0 switches it off.  caee_profile_read synchronises on the recorded
 * events and writes the expert kernel's duration of each recorded call in ms to
 * expert_ms (host, [n_slots]) and their number to n_out (host), then rewinds to slot 0. */
caee_status caee_profile(caee_ctx* ctx, int32_t n_slots);
caee_status caee_profile_read(caee_ctx* ctx, float* expert_ms, int32_t* n_out);
/* Offloading steps recorded by caee_profile (static residency; call BEFORE caee_profile_read, which rewinds):
 * per recorded step, copy_ms = duration of the step's H2D copy train on the side stream (first copy
 * starts .. last copy ends), resident_ms = duration of the resident experts' launch on the caller's stream,
 * lead_ms = from the start of the copy train to the end of the resident launch: resident compute is hidden
 * behind the copies when lead_ms <= copy_ms (north_star (4)).  Host arrays of `cap`. */
caee_status caee_profile_read_offload(caee_ctx* ctx, int32_t cap, float* copy_ms, float* resident_ms, float* lead_ms,
                                      int32_t* n_out);

/* ---- LFU expert cache (Fig. 8: "each HBM caches only a subset of 1024 experts,
 * managed by a Least Frequently Used (LFU) eviction policy").  Turns the
 * static residency mask R(e,d) of caee_set_residency into state that evolves over the steps of a
 * multi-layer decode loop.  Rules (R30-R34): keys are (layer, routed expert); a
 * key's frequency is the number of steps that executed it (after pruning), kept across
 * evictions; a step first counts its executed experts, then inserts its misses in ascending
 * expert order into the lowest free slot, else over the least frequently used key that the
 * step does not execute (ties: smaller (layer, expert)); the cache starts empty; the cost
 * model of a step sees the cache as it is when the step starts.
 *
 * n_slots device slots of one packed expert each are allocated when the first attached layer's
 * weights are set.  caee_cache_attach must precede caee_set_weights(pack != 0) on that context
 * (UMMA kernels only); from then on every routed expert of the layer lives in pinned host
 * memory, caee_set_residency is refused, and caee_moe_forward* fetches the step's misses with
 * one cudaMemcpyAsync each on a side stream while the hits compute (one host synchronisation per
 * step, as in the static offload path).  All layers of one cache must have the same packed
 * expert size and be driven from ONE stream.  A step whose executed experts outnumber the slots
 * fails with CAEE_ESTATE.  caee_route / caee_prune on an attached context use the residency
 * uploaded by its last caee_moe_forward*.  The cache must outlive its attached contexts' calls;
 * destroy the contexts first. */
typedef struct caee_cache caee_cache;
typedef struct caee_cache_stats {
  int64_t hits, misses, evictions; /* per executed (layer, expert, step), since creation */
  int64_t h2d_bytes;               /* misses x packed expert bytes                        */
} caee_cache_stats;
caee_status caee_cache_create(int32_t n_slots, caee_cache** out);
void caee_cache_destroy(caee_cache* cache);
caee_status caee_cache_attach(caee_cache* cache, caee_ctx* ctx, int32_t layer_id);
caee_status caee_cache_read_stats(const caee_cache* cache, caee_cache_stats* out);
/* Contents per slot (host arrays of n_slots): layer and expert (-1: free slot) and the key's
 * frequency. */
caee_status caee_cache_snapshot(const caee_cache* cache, int32_t* layer, int32_t* expert, int64_t* freq);

/* ---- Expert parallelism over the GPUs of one NVLink / NVSwitch domain.
 * PAPER.md:57 (II-B): "token dispatch -> expert activation -> computation -> result aggregation ...
 * across devices"; Latency_total = max_d Latency_d; F_cost as a max over
 * devices.  One process and one context per GPU ("rank"); every rank owns a subset of the routed experts
 * (owner[e], normally the cost model's partition table) and holds the shared experts (R39).  A step:
 *   1. every rank has the SAME x [T,H] (the ranks' own tokens, all-gathered by the caller's transport:
 *      home tokens of rank r are the contiguous block [r ceil(T/world), (r+1) ceil(T/world)) ∩ [0,T));
 *   2. caee_moe_forward*(x, T, p, y = NULL allowed) on every rank: each rank takes the same batch-global
 *      decision from the same scores (R40: deterministic kernels on identical inputs), runs only the runs
 *      of the experts it owns — its slice, in (expert, token) order, of the expert-major work list (R38) —
 *      plus the shared experts of its home tokens, and its expert kernel's epilogue stores every
 *      (token, slot) output row straight into the o buffer of the token's home rank through peer memory
 *      (the aggregation all-to-all is fused into the expert kernel; no combine yet);
 *   3. the caller synchronises the group (every rank's step-2 work complete: a barrier of its transport);
 *   4. caee_ep_combine(T, y) on every rank: y rows of the rank's home tokens (other rows untouched) — the
 *      same list-order sum as on one device, so the result is bit-identical to the single-device layer.
 * caee_set_ep: rank, world <= 8, owner host [E] in 0..world-1, obuf_peers host [world] = every rank's
 * caee_ep_obuf pointer as seen from THIS device (its own at [rank]; peers' through caee_ep_ipc_open of
 * the handle their caee_ep_ipc_export wrote, 64 bytes, or plain pointers when the contexts share a
 * process).  world <= 1 or owner == NULL switches expert parallelism off.  Synchronises.  Not combinable
 * with non-resident experts or the expert cache (CAEE_ESTATE at the step).  When caee_set_ep precedes
 * caee_set_weights, the weight pointers of experts the rank does not own may be NULL: they are neither
 * read nor packed (a rank holds E/world routed experts + the shared ones); switching expert parallelism
 * off, or handing the rank an expert it never loaded, then invalidates the weights (set them again).  The paper's per-device cost
 * model is unchanged: set the partitions to the owner table and F_cost is the max over the physical devices.
 * caee_ep_plan: the explicit dispatch plan of the LAST decision on this context — the valid
 * (token, slot) entries in ascending (device, expert, token) order: counts dev [world], offs dev [world+1],
 * tok / slot / expert dev [T k] (first offs[world] entries valid). */
caee_status caee_set_ep(caee_ctx* ctx, int32_t rank, int32_t world, const int32_t* owner, void* const* obuf_peers);
caee_status caee_ep_obuf(caee_ctx* ctx, void** out, int64_t* bytes);
caee_status caee_ep_ipc_export(caee_ctx* ctx, void* handle64);
caee_status caee_ep_ipc_open(caee_ctx* ctx, const void* handle64, void** out);
caee_status caee_ep_ipc_close(caee_ctx* ctx, void* peer_ptr);
caee_status caee_ep_combine(caee_ctx* ctx, int32_t T, void* y, void* stream);
caee_status caee_ep_plan(caee_ctx* ctx, int32_t* counts, int32_t* offs, int32_t* tok, int32_t* slot, int32_t* expert,
                         void* stream);

/* Library / build identification, e.g. "caee-b200 0.1 sm_100a". */
const char* caee_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CAEE_H_ */
