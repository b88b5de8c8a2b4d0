// caee_internal.cuh — context layout and launch declarations shared by the .cu files of
// libcaee.  Not part of the public ABI (include/caee.h).
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/caee.h"

// Bounds checks of our own (compute-sanitizer is closed on this pool): a build with -DCAEE_ASSERTS
// (CAEE_NVCC_EXTRA) traps the kernel when an index computed on the device leaves its array; the small parity
// tests are run under such a build (profiles/r02_asserts.md).  Compiled out of the product build.
#ifdef CAEE_ASSERTS
#include <cassert>
#define CAEE_DEV_ASSERT(cond) assert(cond)
#else
#define CAEE_DEV_ASSERT(cond) ((void)0)
#endif

#define CAEE_FIX_ONE_F 1099511627776.0f /* 2^40: fixed-point unit of I(e) */
#define CAEE_MAX_E 512
#define CAEE_MAX_D 64
#define CAEE_RUN_TOKENS 128 /* most tokens per run: one UMMA N tile */
#define CAEE_RUN_TOKENS_MIN 64
#define CAEE_RUN_TOKENS_TS 192 /* e4m3 prefill kernel with the weights in tensor memory (expert_fp8_ts.cu), its wider shape */
#define CAEE_RUN_TOKENS_WIDE 256 /* e4m3 prefill kernel (expert_fp8_wide.cu): one N = 256 UMMA tile */
#define CAEE_FP8_WIDE_MIN_TOKENS 129 /* e4m3 steps of at least this many tokens take the converter kernels (expert_fp8_ts.cu / _wide.cu):
                                        measured on C4 against the decode kernel, T=192 -6%, T=256 -7%, T=128 +4% (the x gather) */
#define CAEE_STAGE_RING 8  /* staging slots of the static offload path */
#define CAEE_FETCH_GROUP 4 /* fetched experts per expert-kernel launch */
#define CAEE_EP_MAX 8 /* most devices of an expert-parallel group (one NVSwitch domain) */
#define CAEE_DECIDE_MAX_TOKENS 256 /* largest step the one-kernel decision path takes (decide.cu) */

// One unit of expert work: <= CAEE_RUN_TOKENS tokens of one expert.
struct caee_worklist {
  // experts with >= 1 token (ABI view, S6)
  int32_t* counts;      // [E]   tokens per routed expert
  int32_t* estart;      // [E]   first entry of expert e (exclusive scan of counts)
  int32_t* offs;        // [E+1] exclusive scan over experts with >= 1 token (compacted)
  int32_t* expert_ids;  // [E]
  int32_t* ent_tok;     // [Tmax*(k+S)] token of each entry; routed entries first, shared after Tmax*k... see worklist.cu
  int32_t* ent_slot;    // [Tmax*k]
  float* ent_wt;        // [Tmax*k]
  int32_t* ent_dst;     // [Tmax*(k+S)] destination row in o
  // runs (kernel view)
  int32_t* run_expert;  // [max_runs] expert id in 0..E+S-1
  int32_t* run_start;   // [max_runs] first entry
  int32_t* run_n;       // [max_runs] tokens in the run, 1..CAEE_RUN_TOKENS
  int32_t* run_hrow;    // [max_runs] first row of the run in the h scratch (rows padded to 16 per run)
  int32_t* meta;        // [16]: 0 n_run(ABI) 1 n_runs 2 n_entries(routed) 3 h rows total
                        //       4 runs of resident + shared experts (they come first) 5.. reserved
  int32_t* sched;       // [n_tickets + max_runs]: tile-ticket counters (one per expert-kernel launch of a step),
  int32_t* ready;       //   then (= sched + n_tickets) per-run "h complete" counters; zeroed every step
  int32_t max_runs, n_tickets;
  int32_t ent_cap, hrow_cap;   // entries of ent_tok / ent_dst, rows of the h scratch (bounds, CAEE_ASSERTS builds)
  int32_t run_cap;      // tokens per run this step: CAEE_RUN_TOKENS, 64 (UMMA decode steps, T <= 128) or
                        // CAEE_RUN_TOKENS_WIDE (e4m3 prefill steps)
  // Expert parallelism (caee_set_ep): this device runs only the experts it
  // owns (runs are built for them alone; the lists still hold every entry) and the shared experts of its home
  // tokens [ep_tlo, ep_thi); an o row goes to the o buffer of the token's home device, ep_obuf[t / ep_per]
  const uint8_t* ep_owned;   // [E] 1: this device owns the expert; NULL: no expert parallelism
  int32_t ep_world, ep_per;  // devices; home tokens per device this step = ceil(T / world)
  int32_t ep_tlo, ep_thi;
  float* ep_obuf[CAEE_EP_MAX];
};

// the o buffer a (token, slot) output row goes to
__device__ __forceinline__ float* caee_o_base(const caee_worklist& wl, float* local, int tok) {
  return wl.ep_owned ? wl.ep_obuf[tok / wl.ep_per] : local;
}

struct caee_packed {
  // per expert (E+S) device pointer to the packed tile image, or NULL if not packed / not resident
  uint8_t** dev_ptrs;            // device array [E+S]
  std::vector<uint8_t*> base;    // host copy of the pointers (device memory or pinned host)
  std::vector<uint8_t> on_host;  // 1: base[e] is pinned host memory
  size_t bytes_per_expert = 0;
  size_t p1_tile_bytes = 0, p2_tile_bytes = 0;  // bytes of one phase-1 / phase-2 tile (all k-blocks)
};

struct caee_ctx;

// LFU expert cache shared by the layers (contexts) attached to it (cache.cu; include/caee.h).
struct caee_cache {
  int n_slots = 0, device = 0;
  size_t slot_bytes = 0;                       // packed expert bytes; 0 until the first layer's weights are set
  std::vector<uint8_t*> slot_ptr;              // [n_slots] device slots
  std::vector<int32_t> slot_layer, slot_expert;  // [n_slots] key of each slot, -1 = free
  std::vector<caee_ctx*> layers;               // by layer id (NULL: not attached)
  std::vector<std::vector<int64_t>> freq;      // [layer][E] executions so far (kept across evictions)
  std::vector<std::vector<int32_t>> slot_of;   // [layer][E] slot of a cached key, else -1
  caee_cache_stats st = {0, 0, 0, 0};
};

struct caee_ctx {
  caee_layer_desc d;
  int device = 0, num_sms = 0;
  int kernel = CAEE_KERNEL_SIMT;  // resolved expert kernel
  std::string err;
  bool cuda_failed = false;

  // router (borrowed)
  const float* Wr = nullptr;
  const float* b_logit = nullptr;
  const float* corr_bias = nullptr;
  bool have_router = false, have_weights = false, have_cost = false;

  // tables
  std::vector<int32_t> part_h;
  std::vector<uint8_t> resident_h;
  std::vector<int64_t> ticks_res_h, ticks_miss_h;
  int32_t* part = nullptr;      // dev [E]
  int32_t* pl_experts = nullptr;  // dev [E]   the experts grouped by partition (ascending id inside E_d)
  int32_t* pl_start = nullptr;    // dev [D+1] where each E_d starts in pl_experts
  int part_max = 0;               // largest |E_d|: <= 32 lets the decision run one warp per partition (prune_dev.cuh)
  uint8_t* resident = nullptr;  // dev [E]
  int64_t* w_eff = nullptr;     // dev [E] = resident ? ticks_resident : ticks_miss

  // raw weights (borrowed): device arrays of E+S pointers
  const void** wg = nullptr;
  const void** wu = nullptr;
  const void** wd = nullptr;
  const float** sg = nullptr;
  const float** su = nullptr;
  const float** sd = nullptr;
  std::vector<const void*> wg_h, wu_h, wd_h;
  std::vector<const float*> sg_h, su_h, sd_h;
  caee_packed packed;

  int router_small_waves = 1;       // CTAs per SM of the GEMV-shaped router (steps of <= 4 tokens); env CAEE_ROUTER_SMALL_WAVES
  uint8_t* wr_img = nullptr;        // three bf16 terms of W_r as MMA stage images (router_mma.cu); NULL: shape not supported
  int router_mma_min_tokens = 64;   // steps of at least this many tokens take the tensor-core router (env CAEE_ROUTER_MMA_MIN_TOKENS;
                                    // measured on C3: T=32 +-0, T=64 -4 us, T=128 -17 us, T=256 -42 us, T=4096 -440 us per step)

  // scratch
  float* partial = nullptr;  // [ksplit, T, E] split-K partial logits of x W_r^T (sized for the worst T)
  uint8_t* decide_scratch = nullptr;  // k_decide's self-cleaning accumulators, membership matrix, barriers
  float* scores = nullptr;   // [Tmax, E]
  int32_t* idx = nullptr;    // [Tmax, k]
  float* gate = nullptr;     // [Tmax, k]
  uint8_t* act = nullptr;    // [E]
  uint8_t* must = nullptr;
  uint8_t* keep = nullptr;
  int64_t* I_fix = nullptr;  // [E]
  int64_t* load = nullptr;   // [D]
  int64_t* scalars = nullptr;  // [8]
  caee_worklist wl;
  int32_t* wl_hist = nullptr;        // [ceil(Tmax k / 256), E] per-block entry counts of the large-step fill (worklist.cu)
  float* hbuf_f32 = nullptr;         // SIMT: h rows [rows, I] fp32
  __nv_bfloat16* hbuf_b16 = nullptr; // UMMA: h rows [rows, I] bf16 (bf16 weights) / fp16 (e4m3 weights)
  uint8_t* xq = nullptr;             // UMMA e4m3: hi | lo e4m3 terms of x, [Tmax, H] each
  float* xs = nullptr;               //   and its (token, 128-block) scales [Tmax, H/128]
  uint8_t* hq = nullptr;             // UMMA e4m3: hi | lo terms of h, [rows, I] each
  float* hs = nullptr;               //   and its scales [rows, I/128]
  alignas(64) unsigned char tm_x[128] = {0}, tm_h[128] = {0};  // CUtensorMap of xq / hq (row gathers), see expert_fp8.cu
  uint8_t* xg = nullptr;             // e4m3 converter kernels (expert_fp8_ts.cu, expert_fp8_wide.cu): per-run stage images of the gathered x rows
  bool tm_ready = false;
  int wide_max_pairs = -1;           // co-resident CTA pairs of the e4m3 prefill kernel on this device (-1: not asked yet)
  unsigned attr_done = 0;            // bit i: this context's device has kernel i's MaxDynamicSharedMemorySize (a per-device attribute)
  int fp8_wide_min_tokens = CAEE_FP8_WIDE_MIN_TOKENS;
  bool pdl = true;                   // programmatic dependent launches on the decode path (env CAEE_NO_PDL=1 switches them off)
  int step_prefill = 0;              // this step's e4m3 expert kernel: 0 decode (expert_fp8.cu), 1 expert_fp8_wide.cu, 2 expert_fp8_ts.cu
  int ts_run_tokens = CAEE_RUN_TOKENS_TS;   // run cap of expert_fp8_ts.cu steps: CAEE_RUN_TOKENS_TS (192) or 128 (env CAEE_TS_RUN_TOKENS=128)
  bool fp8_ts = true;                // prefill-size e4m3 steps take the A-from-TMEM kernel (expert_fp8_ts.cu); env CAEE_FP8_TS=0: expert_fp8_wide.cu
  bool fp8_wide_pairs = false;       // e4m3 prefill kernel on CTA pairs (cta_group::2); env CAEE_FP8_WIDE_PAIRS=1 at caee_create
  float* ks_part = nullptr;          // UMMA decode kernels: partial sums of split phase-1 tiles (KSplit, umma_common.cuh)
  int32_t* ks_cnt = nullptr;         //   and their per-tile counters (zero between steps)
  int ks_tile_cap = 0;               //   steps with at most this many phase-1 tiles split them (0: never; env CAEE_NO_KSPLIT=1)
  float* obuf = nullptr;             // [Tmax*(k+S), H] fp32 expert outputs, token-major slots
  size_t h_rows_cap = 0;

  // expert parallelism (caee_set_ep)
  int ep_rank = 0, ep_world = 1;
  uint8_t* ep_owned = nullptr;       // dev [E]
  std::vector<int32_t> ep_owner_h;   // [E] owner device of every routed expert
  float* ep_obuf_h[CAEE_EP_MAX] = {nullptr};
  bool weights_partial = false;      // caee_set_weights skipped experts this rank does not own
  int32_t* ep_owner = nullptr;       // dev [E]

  long long n_launches = 0;          // kernels of this library enqueued by the per-step calls (caee_launch_count)
  // the timed points of the last caee_calibrate_cost (caee_calibrate_points): [tier] -> sizes in bytes, medians in ns
  std::vector<double> calib_bytes[2], calib_ns[2];

  // optional expert-kernel timing (caee_profile)
  std::vector<cudaEvent_t> prof_ev;  // 2 per slot
  int prof_used = 0;

  // offload (S9): packed images of non-resident experts live in pinned host memory
  // (packed.base[e], on_host) and are copied into their staging slot (stage_slot[e], device)
  // on the side stream, only when they survive pruning
  cudaStream_t side_stream = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  // Static offload stages the fetched images in a small RING of device slots (not one slot per non-resident
  // expert: 192 x 88 MB would pin 16.9 GB of HBM): miss i of a step goes to slot (ring_next + i) % n, after the
  // expert-kernel launch that last read that slot (ring_free_ev).  Fetched experts run in groups of
  // CAEE_FETCH_GROUP per expert-kernel launch, each launch behind the last copy of its group.
  std::vector<uint8_t*> stage_ring;      // device slots of one packed expert each
  std::vector<cudaEvent_t> ring_free_ev; // per slot: the last launch that read it has been enqueued up to here
  uint8_t** ring_ptr_pin = nullptr;      // pinned copy of stage_ring (source of the per-miss image-pointer updates)
  unsigned ring_next = 0;
  std::vector<cudaEvent_t> fetch_ev;     // one per non-resident expert
  // copy-train timing of profiled offloading steps (caee_profile / caee_profile_read_offload): per slot
  // {first copy starts, last copy ends} on the side stream, {resident launch starts, ends} on the caller's
  std::vector<cudaEvent_t> prof_off_ev;  // 4 per slot
  int32_t* host_meta = nullptr;          // pinned: meta[16] then run_expert[max_runs]
  bool any_offload = false;

  // caee_moe_forward_host: double-buffered device staging and the two copy streams
  void* hx_d[2] = {nullptr, nullptr};
  void* hy_d[2] = {nullptr, nullptr};
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t ev_hin[2] = {nullptr, nullptr}, ev_hcmp[2] = {nullptr, nullptr}, ev_hout[2] = {nullptr, nullptr};
  unsigned host_step = 0;

  // LFU cache mode (cache.cu): residency, effective costs and image pointers change every step
  caee_cache* cache = nullptr;
  int cache_layer = -1;
  std::vector<uint8_t*> dptr_h;          // host copy of packed.dev_ptrs
  uint8_t* cache_up = nullptr;           // pinned staging: w_eff [E] int64 | dev_ptrs [E+S] | resident [E]
};

caee_status caee_fail(caee_ctx* c, caee_status code, const char* fmt, ...);
caee_status caee_check_cuda(caee_ctx* c, cudaError_t e, const char* what);

#define CAEE_CUDA(c, expr)                                             \
  do {                                                                 \
    cudaError_t _e = (expr);                                           \
    if (_e != cudaSuccess) return caee_check_cuda((c), _e, #expr);     \
  } while (0)

static inline int caee_ceil_div(int a, int b) { return (a + b - 1) / b; }

// router.cu
void caee_router_shape(const caee_ctx* c, int T, int* token_tile, int* ksplit, int* k_chunk);
caee_status caee_launch_router_logits(caee_ctx* c, const void* x, int T, cudaStream_t s);
// router_mma.cu
bool caee_router_mma_supported(const caee_ctx* c);
size_t caee_router_mma_image_bytes(const caee_ctx* c);
bool caee_router_uses_mma(const caee_ctx* c, int T);
void caee_router_mma_shape(const caee_ctx* c, int T, int* ksplit, int* stages_per_split);
void caee_launch_pack_router(caee_ctx* c, cudaStream_t s);
caee_status caee_launch_router_mma(caee_ctx* c, const void* x, int T, cudaStream_t s);
void caee_launch_route_topk(caee_ctx* c, const float* scores_in, int T, float* scores_out, int32_t* idx, float* gate,
                            cudaStream_t s);
// decide.cu
bool caee_decide_fits(const caee_ctx* c, int T);
size_t caee_decide_scratch_bytes(const caee_ctx* c);
bool caee_decide_splits_x(const caee_ctx* c, int T);   // the one-CTA decision kernel also does the e4m3 decode kernel's x split
cudaError_t caee_launch_decide(caee_ctx* c, const float* scores_in, int T, const caee_prune_params* p, caee_fwd_stats* stats,
                               cudaStream_t s, const void* x_split = nullptr);
// prune.cu
void caee_launch_prune(caee_ctx* c, int mode, int flags, double theta, double eps, int T, const int32_t* idx,
                       const float* gate, cudaStream_t s);
void caee_launch_compensate(caee_ctx* c, int flags, const float* scores, int T, int32_t* idx, float* gate,
                            cudaStream_t s);
// worklist.cu
void caee_launch_worklist(caee_ctx* c, int T, const int32_t* idx, const float* gate, cudaStream_t s);
size_t caee_wl_hist_ints(const caee_ctx* c);
void caee_launch_export_worklist(caee_ctx* c, int T, const caee_prune_out* out, cudaStream_t s);
// expert_simt.cu
void caee_launch_expert_simt(caee_ctx* c, const void* x, int T, cudaStream_t s);
// expert_umma.cu
caee_status caee_umma_supported(const caee_ctx* c, std::string* why);
size_t caee_umma_packed_bytes(const caee_ctx* c);
void caee_launch_pack_expert(caee_ctx* c, int e, uint8_t* dst_dev, const void* g, const void* u, const void* d,
                             const float* sg, const float* su, const float* sd, cudaStream_t s);
void caee_launch_umma_prepare(caee_ctx* c, const void* x, int T, cudaStream_t s);
caee_status caee_launch_expert_umma(caee_ctx* c, const void* x, int T, int run_begin, int run_count, int ticket, cudaStream_t s);
// expert_fp8.cu
caee_status caee_fp8_supported(const caee_ctx* c, std::string* why);
size_t caee_fp8_packed_bytes(const caee_ctx* c);
size_t caee_fp8_norm_offset(const caee_ctx* c);
void caee_launch_pack_expert_fp8(caee_ctx* c, uint8_t* dst_dev, const void* g, const void* u, const void* d, const float* sg,
                                 const float* su, const float* sd, cudaStream_t s);
void caee_launch_fp8_prepare(caee_ctx* c, const void* x, int T, cudaStream_t s);
caee_status caee_fp8_make_tensor_maps(caee_ctx* c);
void caee_launch_expert_fp8(caee_ctx* c, int T, int run_begin, int run_count, int ticket, cudaStream_t s);
// expert_fp8_wide.cu
bool caee_fp8_wide_supported(const caee_ctx* c);
size_t caee_fp8_wide_xg_bytes(const caee_ctx* c);
void caee_launch_fp8_wide_prepare(caee_ctx* c, const void* x, int T, cudaStream_t s);
void caee_launch_expert_fp8_wide(caee_ctx* c, int T, int run_begin, int run_count, int ticket, cudaStream_t s);
// expert_fp8_ts.cu
void caee_launch_expert_fp8_ts(caee_ctx* c, int T, int run_begin, int run_count, int ticket, cudaStream_t s);
// cache.cu
caee_status caee_cache_prepare_layer(caee_ctx* c, size_t slot_bytes);
void caee_cache_detach(caee_ctx* c);
caee_status caee_cache_step(caee_ctx* c, const int32_t* executed, int n_executed, std::vector<uint8_t*>* miss_slots);
// combine.cu
void caee_launch_combine(caee_ctx* c, int T, const int32_t* idx, const float* gate, void* y, cudaStream_t s, int t_lo = 0, int t_hi = -1);
void caee_launch_stats(caee_ctx* c, caee_fwd_stats* stats, int pruned, int n_fetch, cudaStream_t s);
long long caee_expert_bytes(const caee_ctx* c);
// ep.cu
void caee_launch_ep_plan(caee_ctx* c, const int32_t* owner_dev, int world, int32_t* counts, int32_t* offs, int32_t* tok,
                         int32_t* slot, int32_t* expert, cudaStream_t s);
// calibrate.cu
caee_status caee_calibrate_impl(caee_ctx* c, const caee_calib_opts* o, caee_cost_fit fit[2]);
