// caee_api.cu — the C ABI of include/caee.h: context, validation, tables, and the enqueue
// sequences of the per-layer hot path.  No torch types, no exceptions across the boundary.
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "umma_common.cuh"

static thread_local std::string g_create_err;

caee_status caee_fail(caee_ctx* c, caee_status code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) c->err = buf;
  else g_create_err = buf;
  return code;
}

caee_status caee_check_cuda(caee_ctx* c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return CAEE_OK;
  if (c) c->cuda_failed = true;
  if (e == cudaErrorMemoryAllocation) {
    cudaGetLastError();
    return caee_fail(c, CAEE_ENOMEM, "%s: %s", what, cudaGetErrorString(e));
  }
  return caee_fail(c, CAEE_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

namespace {

template <typename T>
caee_status dev_alloc(caee_ctx* c, T** p, size_t n) {
  CAEE_CUDA(c, cudaMalloc(reinterpret_cast<void**>(p), sizeof(T) * (n ? n : 1)));
  return CAEE_OK;
}

struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) {
    cudaGetDevice(&prev);
    if (prev != dev) cudaSetDevice(dev);
    else prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

caee_status validate_desc(const caee_layer_desc* d) {
  if (!d) return caee_fail(nullptr, CAEE_EINVAL, "desc is NULL");
  if (d->H < 8 || d->I < 8 || d->H % 8 || d->I % 8) return caee_fail(nullptr, CAEE_ESHAPE, "H and I must be positive multiples of 8");
  if (d->E < 1 || d->E > CAEE_MAX_E) return caee_fail(nullptr, CAEE_EINVAL, "E must be in 1..%d", CAEE_MAX_E);
  if (d->S < 0 || d->S > 16) return caee_fail(nullptr, CAEE_EINVAL, "S must be in 0..16");
  if (d->k < 1 || d->k > d->E || d->k > 32) return caee_fail(nullptr, CAEE_EINVAL, "k must be in 1..min(E,32)");
  if (d->n_group < 1 || d->n_group > 32 || d->E % d->n_group) return caee_fail(nullptr, CAEE_EINVAL, "n_group must divide E and be <= 32");
  if (d->topk_group < 1 || d->topk_group > d->n_group) return caee_fail(nullptr, CAEE_EINVAL, "topk_group must be in 1..n_group");
  if ((long long)d->topk_group * (d->E / d->n_group) < d->k) return caee_fail(nullptr, CAEE_EINVAL, "topk_group*(E/n_group) < k");
  if (d->score_fn != CAEE_SCORE_SOFTMAX && d->score_fn != CAEE_SCORE_SIGMOID) return caee_fail(nullptr, CAEE_EINVAL, "unknown score_fn");
  if (d->act_dtype != CAEE_F32 && d->act_dtype != CAEE_BF16) return caee_fail(nullptr, CAEE_EDTYPE, "act_dtype must be F32 or BF16");
  if (d->w_dtype != CAEE_F32 && d->w_dtype != CAEE_BF16 && d->w_dtype != CAEE_E4M3) return caee_fail(nullptr, CAEE_EDTYPE, "unknown w_dtype");
  if (d->D < 1 || d->D > CAEE_MAX_D) return caee_fail(nullptr, CAEE_EINVAL, "D must be in 1..%d", CAEE_MAX_D);
  if (d->max_tokens < 1 || d->max_tokens > 65536) return caee_fail(nullptr, CAEE_EINVAL, "max_tokens must be in 1..65536");
  if (d->expert_kernel < CAEE_KERNEL_AUTO || d->expert_kernel > CAEE_KERNEL_UMMA) return caee_fail(nullptr, CAEE_EINVAL, "unknown expert_kernel");
  if (!(d->routed_scale == d->routed_scale)) return caee_fail(nullptr, CAEE_EINVAL, "routed_scale is NaN");
  return CAEE_OK;
}

caee_status validate_prune(caee_ctx* c, const caee_prune_params* p) {
  if (!p) return CAEE_OK;
  switch (p->mode) {
    case CAEE_PRUNE_NONE: break;
    case CAEE_PRUNE_THRESH:
      if (!(p->theta >= 0.0) || p->theta > 1e6) return caee_fail(c, CAEE_EINVAL, "THRESH: theta must be in [0, 1e6]");
      break;
    case CAEE_PRUNE_CIR:
      if (!(p->theta > 0.0 && p->theta <= 1.0)) return caee_fail(c, CAEE_EINVAL, "CIR: theta_imp must be in (0,1]");
      break;
    case CAEE_PRUNE_RANK:
      if (!(p->theta >= 0.0 && p->theta <= c->d.k) || p->theta != (double)(int)p->theta)
        return caee_fail(c, CAEE_EINVAL, "RANK: budget must be an integer in 0..k");
      break;
    case CAEE_PRUNE_FRAC:
      if (!(p->theta >= 0.0 && p->theta <= 1.0)) return caee_fail(c, CAEE_EINVAL, "FRAC: p must be in [0,1]");
      break;
    default: return caee_fail(c, CAEE_EINVAL, "unknown prune mode %d", p->mode);
  }
  if (p->flags & ~(CAEE_COMP_ALL_TOKENS | CAEE_KEEP_TOP1 | CAEE_COMP_RANDOM | CAEE_IMP_BOUND)) return caee_fail(c, CAEE_EINVAL, "unknown prune flags");
  if ((p->flags & CAEE_IMP_BOUND) && (!(p->eps >= 0.0) || p->eps > 1e6)) return caee_fail(c, CAEE_EINVAL, "IMP_BOUND: eps must be in [0, 1e6]");
  return CAEE_OK;
}

// E_d as lists: experts grouped by partition, ascending id inside a partition
caee_status upload_partitions(caee_ctx* c) {
  const int E = c->d.E, D = c->d.D;
  std::vector<int32_t> start(D + 1, 0), list(E);
  for (int e = 0; e < E; ++e) ++start[c->part_h[e] + 1];
  c->part_max = 0;
  for (int d = 0; d < D; ++d) { c->part_max = std::max(c->part_max, start[d + 1]); start[d + 1] += start[d]; }
  std::vector<int32_t> fill(start.begin(), start.end() - 1);
  for (int e = 0; e < E; ++e) list[fill[c->part_h[e]]++] = e;
  CAEE_CUDA(c, cudaMemcpy(c->part, c->part_h.data(), sizeof(int32_t) * E, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->pl_experts, list.data(), sizeof(int32_t) * E, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->pl_start, start.data(), sizeof(int32_t) * (D + 1), cudaMemcpyHostToDevice));
  return CAEE_OK;
}

caee_status upload_costs(caee_ctx* c) {
  const int E = c->d.E;
  std::vector<int64_t> w(E);
  for (int e = 0; e < E; ++e) w[e] = c->resident_h[e] ? c->ticks_res_h[e] : c->ticks_miss_h[e];
  CAEE_CUDA(c, cudaMemcpy(c->w_eff, w.data(), sizeof(int64_t) * E, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->resident, c->resident_h.data(), E, cudaMemcpyHostToDevice));
  return CAEE_OK;
}

caee_status check_call(caee_ctx* c, int T) {
  if (!c) return CAEE_EINVAL;
  if (c->cuda_failed) return CAEE_ECUDA;
  if (T < 0) return caee_fail(c, CAEE_EINVAL, "T < 0");
  if (T > c->d.max_tokens) return caee_fail(c, CAEE_ESHAPE, "T=%d exceeds max_tokens=%d", T, c->d.max_tokens);
  return CAEE_OK;
}

caee_status after_launch(caee_ctx* c, const char* what) {
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? CAEE_OK : caee_check_cuda(c, e, what);
}

void free_all(caee_ctx* c) {
  void* ptrs[] = {c->part, c->pl_experts, c->pl_start, c->resident, c->w_eff, c->wg, c->wu, c->wd, c->sg, c->su, c->sd, c->partial, c->decide_scratch, c->scores, c->idx,
                  c->gate, c->act, c->must, c->keep, c->I_fix, c->load, c->scalars, c->wl.counts, c->wl.estart, c->wl.offs,
                  c->wl.expert_ids, c->wl.ent_tok, c->wl.ent_slot, c->wl.ent_wt, c->wl.ent_dst, c->wl.run_expert,
                  c->wl.run_start, c->wl.run_n, c->wl.run_hrow, c->wl.meta, c->wl.sched, c->hbuf_f32, c->hbuf_b16, c->obuf,
                  c->packed.dev_ptrs, c->xq, c->xs, c->hq, c->hs, c->xg, c->wl_hist, c->wr_img, c->ks_part, c->ks_cnt, c->ep_owned, c->ep_owner};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (size_t e = 0; e < c->packed.base.size(); ++e) {
    if (!c->packed.base[e]) continue;
    if (c->packed.on_host[e]) cudaFreeHost(c->packed.base[e]);
    else cudaFree(c->packed.base[e]);
  }
  for (uint8_t* p : c->stage_ring)
    if (p) cudaFree(p);
  for (cudaEvent_t e : c->ring_free_ev) cudaEventDestroy(e);
  if (c->ring_ptr_pin) cudaFreeHost(c->ring_ptr_pin);
  for (cudaEvent_t e : c->prof_off_ev) cudaEventDestroy(e);
  c->prof_off_ev.clear();
  for (cudaEvent_t e : c->fetch_ev) cudaEventDestroy(e);
  if (c->host_meta) cudaFreeHost(c->host_meta);
  if (c->cache_up) cudaFreeHost(c->cache_up);
  for (int b = 0; b < 2; ++b) {
    if (c->hx_d[b]) cudaFree(c->hx_d[b]);
    if (c->hy_d[b]) cudaFree(c->hy_d[b]);
    if (c->ev_hin[b]) cudaEventDestroy(c->ev_hin[b]);
    if (c->ev_hcmp[b]) cudaEventDestroy(c->ev_hcmp[b]);
    if (c->ev_hout[b]) cudaEventDestroy(c->ev_hout[b]);
  }
  if (c->s_in) cudaStreamDestroy(c->s_in);
  if (c->s_out) cudaStreamDestroy(c->s_out);
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  c->prof_ev.clear();
  if (c->side_stream) cudaStreamDestroy(c->side_stream);
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
}

caee_status create_impl(caee_ctx* c) {
  const caee_layer_desc& d = c->d;
  const size_t Tm = d.max_tokens, E = d.E, k = d.k, S = d.S;
  caee_status rc;
  if (const char* v = getenv("CAEE_ROUTER_SMALL_WAVES")) c->router_small_waves = std::max(1, std::min(4, atoi(v)));   // tuning aid
  if (const char* v = getenv("CAEE_ROUTER_MMA_MIN_TOKENS")) c->router_mma_min_tokens = std::max(1, atoi(v));   // tuning aid
  if (caee_router_mma_supported(c) && d.max_tokens >= c->router_mma_min_tokens) {
    if ((rc = dev_alloc(c, &c->wr_img, caee_router_mma_image_bytes(c))) != CAEE_OK) return rc;
  }
  size_t prow = 1;
  for (int T = 1; T <= d.max_tokens; ++T) {
    int tt, ks;
    caee_router_shape(c, T, &tt, &ks, nullptr);
    prow = std::max(prow, (size_t)ks * T);
  }
#define A(ptr, n) if ((rc = dev_alloc(c, &(ptr), (n))) != CAEE_OK) return rc
  A(c->part, E); A(c->pl_experts, E); A(c->pl_start, CAEE_MAX_D + 1); A(c->resident, E); A(c->w_eff, E);
  A(c->wg, E + S); A(c->wu, E + S); A(c->wd, E + S); A(c->sg, E + S); A(c->su, E + S); A(c->sd, E + S);
  A(c->partial, prow * E); A(c->decide_scratch, caee_decide_scratch_bytes(c)); A(c->scores, Tm * E); A(c->idx, Tm * k); A(c->gate, Tm * k);
  A(c->act, E); A(c->must, E); A(c->keep, E); A(c->I_fix, E); A(c->load, CAEE_MAX_D); A(c->scalars, 8);
  c->wl.max_runs = (int)(E + (Tm * k + CAEE_RUN_TOKENS_MIN - 1) / CAEE_RUN_TOKENS_MIN +
                         S * ((Tm + CAEE_RUN_TOKENS_MIN - 1) / CAEE_RUN_TOKENS_MIN));
  c->wl.run_cap = CAEE_RUN_TOKENS;
  A(c->wl.counts, E); A(c->wl.estart, E); A(c->wl.offs, E + 1); A(c->wl.expert_ids, E);
  A(c->wl.ent_tok, Tm * (k + S)); A(c->wl.ent_slot, Tm * k); A(c->wl.ent_wt, Tm * k); A(c->wl.ent_dst, Tm * (k + S));
  A(c->wl.run_expert, c->wl.max_runs); A(c->wl.run_start, c->wl.max_runs); A(c->wl.run_n, c->wl.max_runs);
  c->wl.n_tickets = 2 * ((int)E + 2);    // per expert-kernel launch of a step: tile tickets, then (second half) reducer tickets (KSplit)
  A(c->wl.run_hrow, c->wl.max_runs); A(c->wl.meta, 16); A(c->wl.sched, c->wl.n_tickets + c->wl.max_runs);
  c->wl.ready = c->wl.sched + c->wl.n_tickets;
  if (caee_wl_hist_ints(c)) { A(c->wl_hist, caee_wl_hist_ints(c)); }
  c->h_rows_cap = Tm * k + 15 * std::min(E, Tm * k) + S * (Tm + 15) + 16;
  c->wl.ent_cap = (int32_t)(Tm * (k + S)); c->wl.hrow_cap = (int32_t)c->h_rows_cap;
  if (c->kernel == CAEE_KERNEL_SIMT) { A(c->hbuf_f32, c->h_rows_cap * d.I); }
  else { A(c->hbuf_b16, c->h_rows_cap * d.I); }
  if (c->kernel == CAEE_KERNEL_UMMA && d.w_dtype == CAEE_E4M3) {
    A(c->xq, 2 * Tm * d.H); A(c->xs, Tm * (d.H / 128));
    A(c->hq, 2 * c->h_rows_cap * d.I); A(c->hs, c->h_rows_cap * (d.I / 128));
    if ((rc = caee_fp8_make_tensor_maps(c)) != CAEE_OK) return rc;
    if (const char* v = getenv("CAEE_FP8_WIDE_MIN_TOKENS")) c->fp8_wide_min_tokens = std::max(1, atoi(v));   // tuning aid
    if (const char* v = getenv("CAEE_FP8_WIDE_PAIRS")) c->fp8_wide_pairs = atoi(v) != 0;                      // tuning aid
    if (const char* v = getenv("CAEE_TS_RUN_TOKENS")) c->ts_run_tokens = atoi(v) > CAEE_RUN_TOKENS ? CAEE_RUN_TOKENS_TS : CAEE_RUN_TOKENS;   // tuning aid
    if (const char* v = getenv("CAEE_FP8_TS")) c->fp8_ts = atoi(v) != 0;                                      // tuning aid
    if (!caee_fp8_wide_supported(c)) c->fp8_wide_min_tokens = 1 << 30;   // k range too long for its scale registers
    if (d.max_tokens >= c->fp8_wide_min_tokens) { A(c->xg, caee_fp8_wide_xg_bytes(c)); }
  }
  A(c->obuf, Tm * (k + S) * d.H);
  if (c->kernel == CAEE_KERNEL_UMMA && !(getenv("CAEE_NO_KSPLIT") && atoi(getenv("CAEE_NO_KSPLIT")) != 0)) {
    // steps of one or two tokens: split phase-1 tiles while a step has at most 2 of them per SM (umma_common.cuh:
    // KSplit; measured on C3 / C4: +3.5 / +5.6% at T = 1, +2.7 / 0% at T = 2, -1 / -3.6% at T = 4)
    c->ks_tile_cap = 2 * c->num_sms;
    A(c->ks_part, caee_umma::caee_ksplit_part_floats(c->ks_tile_cap)); A(c->ks_cnt, c->ks_tile_cap);
    CAEE_CUDA(c, cudaMemset(c->ks_cnt, 0, sizeof(int32_t) * c->ks_tile_cap));
  }
#undef A
  if (const char* v = getenv("CAEE_NO_PDL")) c->pdl = atoi(v) == 0;   // tuning aid
  CAEE_CUDA(c, cudaMemset(c->wl.meta, 0, sizeof(int32_t) * 16));
  CAEE_CUDA(c, cudaMemset(c->decide_scratch, 0, caee_decide_scratch_bytes(c)));
  CAEE_CUDA(c, cudaMemset(c->scalars, 0, sizeof(int64_t) * 8));
  CAEE_CUDA(c, cudaMemset(c->load, 0, sizeof(int64_t) * CAEE_MAX_D));
  // defaults: contiguous partitions, everything resident, unit costs
  c->part_h.resize(E); c->resident_h.assign(E, 1); c->ticks_res_h.assign(E, 1); c->ticks_miss_h.assign(E, 1);
  const int per = (int)((E + d.D - 1) / d.D);
  for (size_t e = 0; e < E; ++e) c->part_h[e] = (int32_t)(e / per);
  if ((rc = upload_partitions(c)) != CAEE_OK) return rc;
  if ((rc = upload_costs(c)) != CAEE_OK) return rc;
  CAEE_CUDA(c, cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking));
  CAEE_CUDA(c, cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
  CAEE_CUDA(c, cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
  CAEE_CUDA(c, cudaMallocHost((void**)&c->host_meta, sizeof(int32_t) * (16 + c->wl.max_runs)));
  return CAEE_OK;
}

// expert parallelism: home tokens of this device in a T-token step (contiguous blocks of ceil(T / world))
void ep_step_view(caee_ctx* c, int T) {
  if (!c->wl.ep_owned) return;
  c->wl.ep_per = std::max(1, caee_ceil_div(T, c->ep_world));
  c->wl.ep_tlo = std::min(T, c->ep_rank * c->wl.ep_per);
  c->wl.ep_thi = std::min(T, c->wl.ep_tlo + c->wl.ep_per);
}

// route -> [prune + compensate] -> work list.  scores_in == NULL: compute scores from x.
caee_status enqueue_decisions(caee_ctx* c, const void* x, const float* scores_in, int T, const caee_prune_params* p,
                              int32_t* idx, float* gate, float* scores_out, bool do_route, cudaStream_t st) {
  const float* scores = scores_in;
  if (T > 0 && do_route) {
    if (!scores_in) {
      caee_status rr = caee_launch_router_logits(c, x, T, st);
      if (rr != CAEE_OK) return rr;
      caee_launch_route_topk(c, nullptr, T, scores_out ? scores_out : c->scores, idx, gate, st);
      scores = scores_out ? scores_out : c->scores;
    } else {
      caee_launch_route_topk(c, scores_in, T, nullptr, idx, gate, st);
    }
  }
  const int mode = p ? p->mode : CAEE_PRUNE_NONE;
  if (p) {
    caee_launch_prune(c, mode, p->flags, p->theta, p->eps, T, idx, gate, st);
    if (mode != CAEE_PRUNE_NONE && T > 0) caee_launch_compensate(c, p->flags, scores, T, idx, gate, st);
  }
  caee_launch_worklist(c, T, idx, gate, st);
  return after_launch(c, "decision kernels");
}

}  // namespace

extern "C" {

const char* caee_version(void) { return "caee-b200 0.1 sm_100a"; }

const char* caee_last_error(const caee_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

caee_status caee_create(const caee_layer_desc* desc, caee_ctx** out) {
  if (!out) return caee_fail(nullptr, CAEE_EINVAL, "out is NULL");
  *out = nullptr;
  caee_status rc = validate_desc(desc);
  if (rc != CAEE_OK) return rc;
  int dev = desc->device;
  if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return caee_fail(nullptr, CAEE_EUNSUPPORTED, "no CUDA device: this library has no CPU fallback");
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    return caee_fail(nullptr, CAEE_EUNSUPPORTED, "cannot query CUDA device %d: this library has no CPU fallback", dev);
  }
  if (prop.major != 10) return caee_fail(nullptr, CAEE_EUNSUPPORTED, "device %d is sm_%d%d; libcaee is built for sm_100a only", dev, prop.major, prop.minor);
  caee_ctx* c = new (std::nothrow) caee_ctx();
  if (!c) return caee_fail(nullptr, CAEE_ENOMEM, "host allocation failed");
  c->d = *desc;
  c->d.device = dev;
  c->device = dev;
  c->num_sms = prop.multiProcessorCount;
  c->wl = caee_worklist{};
  c->kernel = desc->expert_kernel;
  if (c->kernel == CAEE_KERNEL_AUTO) {
    std::string why;
    c->kernel = caee_umma_supported(c, &why) == CAEE_OK ? CAEE_KERNEL_UMMA : CAEE_KERNEL_SIMT;
  }
  if (c->kernel == CAEE_KERNEL_UMMA) {
    std::string why;
    rc = caee_umma_supported(c, &why);
    if (rc != CAEE_OK) {
      g_create_err = why;
      delete c;
      return rc;
    }
  }
  DeviceGuard g(dev);
  rc = create_impl(c);
  if (rc != CAEE_OK) {
    g_create_err = c->err;
    free_all(c);
    delete c;
    return rc;
  }
  *out = c;
  return CAEE_OK;
}

caee_status caee_destroy(caee_ctx* c) {
  if (!c) return CAEE_EINVAL;
  DeviceGuard g(c->device);
  cudaDeviceSynchronize();
  caee_cache_detach(c);
  free_all(c);
  delete c;
  return CAEE_OK;
}

caee_status caee_set_router(caee_ctx* c, const float* W_r, const float* b_logit, const float* corr_bias) {
  if (!c) return CAEE_EINVAL;
  if (!W_r) return caee_fail(c, CAEE_EINVAL, "W_r is NULL");
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaDeviceSynchronize());
  c->Wr = W_r; c->b_logit = b_logit; c->corr_bias = corr_bias; c->have_router = true;
  if (c->wr_img) {
    // the tensor-core router's copy of W_r (three bf16 terms, router_mma.cu): made once, here
    caee_launch_pack_router(c, nullptr);
    CAEE_CUDA(c, cudaDeviceSynchronize());
  }
  return CAEE_OK;
}

caee_status caee_set_partitions(caee_ctx* c, const int32_t* part, int32_t D) {
  if (!c) return CAEE_EINVAL;
  if (!part) return caee_fail(c, CAEE_EINVAL, "part_of_expert is NULL");
  if (D != c->d.D) return caee_fail(c, CAEE_EINVAL, "D=%d differs from the descriptor's D=%d", D, c->d.D);
  for (int e = 0; e < c->d.E; ++e)
    if (part[e] < 0 || part[e] >= D) return caee_fail(c, CAEE_EINVAL, "part_of_expert[%d]=%d out of range", e, part[e]);
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaDeviceSynchronize());
  c->part_h.assign(part, part + c->d.E);
  return upload_partitions(c);
}

caee_status caee_set_residency(caee_ctx* c, const uint8_t* resident) {
  if (!c) return CAEE_EINVAL;
  if (!resident) return caee_fail(c, CAEE_EINVAL, "resident is NULL");
  if (c->cache) return caee_fail(c, CAEE_ESTATE, "the context is attached to an expert cache: its residency is the cache's state");
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaDeviceSynchronize());
  bool changed = false;
  for (int e = 0; e < c->d.E; ++e) {
    changed |= c->resident_h[e] != (resident[e] ? 1 : 0);
    c->resident_h[e] = resident[e] ? 1 : 0;
  }
  if (changed) c->have_weights = false;  // where an expert's image lives follows its residency: set the weights again
  return upload_costs(c);
}

caee_status caee_set_cost_table(caee_ctx* c, const int64_t* ticks_resident, const int64_t* ticks_miss) {
  if (!c) return CAEE_EINVAL;
  if (!ticks_resident) return caee_fail(c, CAEE_EINVAL, "ticks_resident is NULL");
  for (int e = 0; e < c->d.E; ++e) {
    if (ticks_resident[e] < 0 || (ticks_miss && ticks_miss[e] < 0)) return caee_fail(c, CAEE_EINVAL, "negative cost for expert %d", e);
    if (ticks_resident[e] > (1LL << 40) || (ticks_miss && ticks_miss[e] > (1LL << 40))) return caee_fail(c, CAEE_EINVAL, "cost for expert %d exceeds 2^40 ns", e);
  }
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaDeviceSynchronize());
  c->ticks_res_h.assign(ticks_resident, ticks_resident + c->d.E);
  if (ticks_miss) c->ticks_miss_h.assign(ticks_miss, ticks_miss + c->d.E);
  else c->ticks_miss_h = c->ticks_res_h;
  c->have_cost = true;
  return upload_costs(c);
}

caee_status caee_set_weights(caee_ctx* c, const caee_expert_weights* w, int32_t pack) {
  if (!c) return CAEE_EINVAL;
  if (!w || !w->gate || !w->up || !w->down) return caee_fail(c, CAEE_EINVAL, "weight pointer tables are NULL");
  const int n = c->d.E + c->d.S;
  const bool fp8 = c->d.w_dtype == CAEE_E4M3;
  if (fp8 && (!w->gate_scale || !w->up_scale || !w->down_scale)) return caee_fail(c, CAEE_EINVAL, "e4m3 weights need block scales");
  // expert parallelism set up first (caee_set_ep): a rank needs only the experts it owns (and the shared ones);
  // the others may be NULL and are skipped
  auto needed = [&](int e) { return e >= c->d.E || c->ep_owner_h.empty() || c->ep_owner_h[e] == c->ep_rank; };
  c->weights_partial = false;
  for (int e = 0; e < n; ++e) {
    if (!needed(e) && !w->gate[e] && !w->up[e] && !w->down[e]) { c->weights_partial = true; continue; }
    if (!w->gate[e] || !w->up[e] || !w->down[e]) return caee_fail(c, CAEE_EINVAL, "expert %d has a NULL weight pointer", e);
    if (fp8 && (!w->gate_scale[e] || !w->up_scale[e] || !w->down_scale[e])) return caee_fail(c, CAEE_EINVAL, "expert %d has a NULL scale pointer", e);
  }
  if (c->kernel == CAEE_KERNEL_UMMA && !pack) return caee_fail(c, CAEE_EINVAL, "the UMMA expert kernel needs pack != 0");
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaDeviceSynchronize());
  c->wg_h.assign(w->gate, w->gate + n); c->wu_h.assign(w->up, w->up + n); c->wd_h.assign(w->down, w->down + n);
  if (fp8) { c->sg_h.assign(w->gate_scale, w->gate_scale + n); c->su_h.assign(w->up_scale, w->up_scale + n); c->sd_h.assign(w->down_scale, w->down_scale + n); }
  else { c->sg_h.assign(n, nullptr); c->su_h.assign(n, nullptr); c->sd_h.assign(n, nullptr); }
  const size_t pb = sizeof(void*) * n;
  CAEE_CUDA(c, cudaMemcpy(c->wg, c->wg_h.data(), pb, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->wu, c->wu_h.data(), pb, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->wd, c->wd_h.data(), pb, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->sg, c->sg_h.data(), pb, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->su, c->su_h.data(), pb, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->sd, c->sd_h.data(), pb, cudaMemcpyHostToDevice));
  if (c->kernel == CAEE_KERNEL_UMMA) {
    // tile-major repack, once ("packed weight layout (done once at caee_set_weights)")
    caee_packed& P = c->packed;
    for (size_t e = 0; e < P.base.size(); ++e)
      if (P.base[e]) { if (P.on_host[e]) cudaFreeHost(P.base[e]); else cudaFree(P.base[e]); }
    P.base.assign(n, nullptr); P.on_host.assign(n, 0);
    P.bytes_per_expert = caee_umma_packed_bytes(c);
    if (!P.dev_ptrs) CAEE_CUDA(c, cudaMalloc((void**)&P.dev_ptrs, pb));
    for (uint8_t* q : c->stage_ring)
      if (q) cudaFree(q);
    for (cudaEvent_t ev : c->ring_free_ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : c->fetch_ev) cudaEventDestroy(ev);
    c->stage_ring.clear(); c->ring_free_ev.clear();
    c->ring_next = 0;
    c->fetch_ev.clear();
    c->any_offload = false;
    if (c->cache) {
      caee_status crc = caee_cache_prepare_layer(c, P.bytes_per_expert);
      if (crc != CAEE_OK) return crc;
      if (!c->cache_up) CAEE_CUDA(c, cudaMallocHost((void**)&c->cache_up, (size_t)c->d.E * 9 + sizeof(void*) * n));
    }
    std::vector<uint8_t*> dptr(n, nullptr);
    uint8_t* tmp = nullptr;  // device scratch for packing a host-resident expert
    for (int e = 0; e < n; ++e) {
      if (!c->wg_h[e]) continue;    // an expert this rank does not own (expert parallelism): no image
      const bool res = e >= c->d.E || (!c->cache && c->resident_h[e]);
      if (res) {
        CAEE_CUDA(c, cudaMalloc((void**)&P.base[e], P.bytes_per_expert));
        caee_launch_pack_expert(c, e, P.base[e], c->wg_h[e], c->wu_h[e], c->wd_h[e], c->sg_h[e], c->su_h[e], c->sd_h[e], 0);
        dptr[e] = P.base[e];
      } else {
        // S9: the image of a non-resident expert stays in pinned host memory; it is copied into
        // its device staging slot by caee_moe_forward only when the expert survives pruning
        if (!tmp) CAEE_CUDA(c, cudaMalloc((void**)&tmp, P.bytes_per_expert));
        caee_launch_pack_expert(c, e, tmp, c->wg_h[e], c->wu_h[e], c->wd_h[e], c->sg_h[e], c->su_h[e], c->sd_h[e], 0);
        CAEE_CUDA(c, cudaMallocHost((void**)&P.base[e], P.bytes_per_expert));
        P.on_host[e] = 1;
        CAEE_CUDA(c, cudaMemcpy(P.base[e], tmp, P.bytes_per_expert, cudaMemcpyDeviceToHost));
        // static offload: the image pointer is set per step to the ring slot the copy goes to; cache mode: the cache's slots
        cudaEvent_t ev;
        CAEE_CUDA(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        c->fetch_ev.push_back(ev);
        c->any_offload = true;
      }
    }
    CAEE_CUDA(c, cudaDeviceSynchronize());
    if (tmp) cudaFree(tmp);
    if (c->any_offload && !c->cache) {
      // the staging ring (caee_internal.cuh): a few slots, reused by the misses of every step
      const int n_ring = std::min<int>(CAEE_STAGE_RING, (int)c->fetch_ev.size());
      if (!c->ring_ptr_pin) CAEE_CUDA(c, cudaMallocHost((void**)&c->ring_ptr_pin, sizeof(uint8_t*) * CAEE_STAGE_RING));
      for (int i = 0; i < n_ring; ++i) {
        uint8_t* q = nullptr;
        CAEE_CUDA(c, cudaMalloc((void**)&q, P.bytes_per_expert));
        c->stage_ring.push_back(q);
        c->ring_ptr_pin[i] = q;
        cudaEvent_t ev;
        CAEE_CUDA(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        CAEE_CUDA(c, cudaEventRecord(ev, nullptr));       // nothing to wait for yet
        c->ring_free_ev.push_back(ev);
      }
    }
    CAEE_CUDA(c, cudaMemcpy(P.dev_ptrs, dptr.data(), pb, cudaMemcpyHostToDevice));
    CAEE_CUDA(c, cudaDeviceSynchronize());
    c->dptr_h = dptr;
    if (c->cache) { caee_status urc = upload_costs(c); if (urc != CAEE_OK) return urc; }
  } else {
    for (int e = 0; e < c->d.E; ++e)
      if (!c->resident_h[e]) return caee_fail(c, CAEE_EUNSUPPORTED, "the SIMT expert kernel needs every expert in device memory");
  }
  if (c->weights_partial && (c->any_offload || c->cache)) return caee_fail(c, CAEE_ESTATE, "expert parallelism does not combine with offloaded experts or the expert cache");
  c->have_weights = true;
  return CAEE_OK;
}

caee_status caee_calibrate_cost(caee_ctx* c, const caee_calib_opts* opts, caee_cost_fit out_fit[2]) {
  if (!c) return CAEE_EINVAL;
  if (!out_fit) return caee_fail(c, CAEE_EINVAL, "out_fit is NULL");
  if (c->cuda_failed) return CAEE_ECUDA;
  DeviceGuard g(c->device);
  caee_status rc = caee_calibrate_impl(c, opts, out_fit);
  if (rc != CAEE_OK) return rc;
  if (!opts || opts->apply) {
    const int64_t bytes = 3LL * c->d.H * c->d.I * (c->d.w_dtype == CAEE_F32 ? 4 : c->d.w_dtype == CAEE_BF16 ? 2 : 1) +
                          (c->d.w_dtype == CAEE_E4M3 ? 3LL * ((c->d.H + 127) / 128) * ((c->d.I + 127) / 128) * 4 : 0);
    std::vector<int64_t> tr(c->d.E), tm(c->d.E);
    for (int e = 0; e < c->d.E; ++e) {
      tr[e] = out_fit[0].valid ? llround(out_fit[0].slope_ns_per_byte * (double)bytes + out_fit[0].intercept_ns) : c->ticks_res_h[e];
      tm[e] = out_fit[1].valid ? llround(out_fit[1].slope_ns_per_byte * (double)bytes + out_fit[1].intercept_ns) : c->ticks_miss_h[e];
      if (tr[e] < 0) tr[e] = 0;
      if (tm[e] < 0) tm[e] = 0;
    }
    return caee_set_cost_table(c, tr.data(), tm.data());
  }
  return CAEE_OK;
}

caee_status caee_calibrate_points(const caee_ctx* c, int32_t tier, int32_t cap, double* bytes, double* ns, int32_t* n_out) {
  if (!c || !n_out || tier < 0 || tier > 1 || cap < 0 || (cap > 0 && (!bytes || !ns))) return CAEE_EINVAL;
  const int n = (int)c->calib_bytes[tier].size();
  *n_out = n;
  for (int i = 0; i < n && i < cap; ++i) { bytes[i] = c->calib_bytes[tier][i]; ns[i] = c->calib_ns[tier][i]; }
  return CAEE_OK;
}

caee_status caee_get_cost_table(const caee_ctx* c, int64_t* ticks_resident, int64_t* ticks_miss) {
  if (!c) return CAEE_EINVAL;
  for (int e = 0; e < c->d.E; ++e) {
    if (ticks_resident) ticks_resident[e] = c->ticks_res_h[e];
    if (ticks_miss) ticks_miss[e] = c->ticks_miss_h[e];
  }
  return CAEE_OK;
}

caee_status caee_launch_count(const caee_ctx* c, int64_t* n_out) {
  if (!c || !n_out) return CAEE_EINVAL;
  *n_out = c->n_launches;
  return CAEE_OK;
}

caee_status caee_route(caee_ctx* c, const void* x, int32_t T, float* scores, int32_t* idx, float* gate, void* stream) {
  caee_status rc = check_call(c, T);
  if (rc != CAEE_OK) return rc;
  if (!c->have_router) return caee_fail(c, CAEE_ESTATE, "caee_route before caee_set_router");
  if (T == 0) return CAEE_OK;
  if (!x || !idx || !gate) return caee_fail(c, CAEE_EINVAL, "x, idx or gate is NULL");
  DeviceGuard g(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  if ((rc = caee_launch_router_logits(c, x, T, st)) != CAEE_OK) return rc;
  caee_launch_route_topk(c, nullptr, T, scores, idx, gate, st);
  return after_launch(c, "caee_route");
}

caee_status caee_route_from_scores(caee_ctx* c, const float* scores, int32_t T, int32_t* idx, float* gate, void* stream) {
  caee_status rc = check_call(c, T);
  if (rc != CAEE_OK) return rc;
  if (T == 0) return CAEE_OK;
  if (!scores || !idx || !gate) return caee_fail(c, CAEE_EINVAL, "scores, idx or gate is NULL");
  DeviceGuard g(c->device);
  caee_launch_route_topk(c, scores, T, nullptr, idx, gate, (cudaStream_t)stream);
  return after_launch(c, "caee_route_from_scores");
}

caee_status caee_prune(caee_ctx* c, const caee_prune_params* p, const float* scores, int32_t T, int32_t* idx, float* gate,
                       const caee_prune_out* out, void* stream) {
  caee_status rc = check_call(c, T);
  if (rc != CAEE_OK) return rc;
  if ((rc = validate_prune(c, p)) != CAEE_OK) return rc;
  if (T > 0 && (!idx || !gate)) return caee_fail(c, CAEE_EINVAL, "idx or gate is NULL");
  const bool prunes = p && p->mode != CAEE_PRUNE_NONE;
  if (prunes && T > 0 && !scores) return caee_fail(c, CAEE_EINVAL, "scores is NULL but compensation needs them");
  DeviceGuard g(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  caee_prune_params none = {CAEE_PRUNE_NONE, 0, 0.0, 0.0};
  c->wl.run_cap = CAEE_RUN_TOKENS;
  ep_step_view(c, T);
  rc = enqueue_decisions(c, nullptr, scores, T, p ? p : &none, idx, gate, nullptr, false, st);
  if (rc != CAEE_OK) return rc;
  caee_launch_export_worklist(c, T, out, st);
  if (out) {
    const size_t E = c->d.E;
    if (out->act) CAEE_CUDA(c, cudaMemcpyAsync(out->act, c->act, E, cudaMemcpyDeviceToDevice, st));
    if (out->must) CAEE_CUDA(c, cudaMemcpyAsync(out->must, c->must, E, cudaMemcpyDeviceToDevice, st));
    if (out->keep) CAEE_CUDA(c, cudaMemcpyAsync(out->keep, c->keep, E, cudaMemcpyDeviceToDevice, st));
    if (out->importance) CAEE_CUDA(c, cudaMemcpyAsync(out->importance, c->I_fix, 8 * E, cudaMemcpyDeviceToDevice, st));
    if (out->load) CAEE_CUDA(c, cudaMemcpyAsync(out->load, c->load, 8 * (size_t)c->d.D, cudaMemcpyDeviceToDevice, st));
    if (out->scalars) CAEE_CUDA(c, cudaMemcpyAsync(out->scalars, c->scalars, 64, cudaMemcpyDeviceToDevice, st));
  }
  return after_launch(c, "caee_prune");
}

static caee_status forward_impl(caee_ctx* c, const void* x, const float* scores, int32_t T, const caee_prune_params* p,
                                void* y, caee_fwd_stats* stats, void* stream) {
  caee_status rc = check_call(c, T);
  if (rc != CAEE_OK) return rc;
  if ((rc = validate_prune(c, p)) != CAEE_OK) return rc;
  if (!c->have_weights) return caee_fail(c, CAEE_ESTATE, "caee_moe_forward before caee_set_weights");
  if (!scores && !c->have_router) return caee_fail(c, CAEE_ESTATE, "caee_moe_forward before caee_set_router");
  if (p && p->mode != CAEE_PRUNE_NONE && !c->have_cost) return caee_fail(c, CAEE_ESTATE, "pruning requested before caee_set_cost_table / caee_calibrate_cost");
  if (T == 0) return CAEE_OK;
  const bool ep = c->wl.ep_owned != nullptr;
  if (!x || (!y && !ep)) return caee_fail(c, CAEE_EINVAL, "x or y is NULL");
  if (((uintptr_t)x | (uintptr_t)y) & 15) return caee_fail(c, CAEE_EINVAL, "x and y must be 16-byte aligned");
  if (ep && (c->any_offload || c->cache)) return caee_fail(c, CAEE_ESTATE, "expert parallelism does not combine with offloaded experts or the expert cache");
  DeviceGuard g(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  // decode steps (T <= 128) use 64-token runs: the smaller token operand leaves room for a deeper
  // weight ring (only the shared experts and the few hottest experts are split and streamed twice),
  // and the e4m3 kernel's hi/lo terms share one MMA (expert_fp8.cu); larger steps keep 128 for weight reuse
  c->wl.run_cap = (c->kernel == CAEE_KERNEL_UMMA && T <= 128) ? CAEE_RUN_TOKENS_MIN : CAEE_RUN_TOKENS;
  // e4m3 prefill-size steps: the A-from-TMEM kernel on 192-token runs (expert_fp8_ts.cu), or the shared-memory converter
  // kernel on 256-token runs (expert_fp8_wide.cu; also for CTA pairs)
  c->step_prefill = 0;
  if (c->kernel == CAEE_KERNEL_UMMA && c->d.w_dtype == CAEE_E4M3 && T >= c->fp8_wide_min_tokens) {
    c->step_prefill = (c->fp8_ts && !c->fp8_wide_pairs) ? 2 : 1;
    c->wl.run_cap = c->step_prefill == 2 ? c->ts_run_tokens : CAEE_RUN_TOKENS_WIDE;
  }
  if (c->cache) {
    // R33: the step's cost model and run order see the cache as it is now (other layers' misses
    // may have evicted this layer's experts since its last step).  The pinned staging buffer is
    // free to rewrite: every cached step ends its decision part with a stream synchronisation.
    const int E = c->d.E, n = E + c->d.S;
    int64_t* w = reinterpret_cast<int64_t*>(c->cache_up);
    uint8_t** dp = reinterpret_cast<uint8_t**>(c->cache_up + (size_t)E * 8);
    uint8_t* rs = c->cache_up + (size_t)E * 8 + sizeof(void*) * n;
    for (int e = 0; e < E; ++e) { w[e] = c->resident_h[e] ? c->ticks_res_h[e] : c->ticks_miss_h[e]; rs[e] = c->resident_h[e]; }
    for (int e = 0; e < n; ++e) dp[e] = c->dptr_h[e];
    CAEE_CUDA(c, cudaMemcpyAsync(c->w_eff, w, sizeof(int64_t) * E, cudaMemcpyHostToDevice, st));
    CAEE_CUDA(c, cudaMemcpyAsync(c->resident, rs, E, cudaMemcpyHostToDevice, st));
    CAEE_CUDA(c, cudaMemcpyAsync(c->packed.dev_ptrs, dp, sizeof(void*) * n, cudaMemcpyHostToDevice, st));
  }
  ep_step_view(c, T);
  const bool fused = caee_decide_fits(c, T);
  // e4m3 decode steps: the split of x into its two e4m3 terms depends on x alone, so it goes first and
  // the chain router GEMM -> decision kernel -> expert kernel stays free for programmatic dependent launches
  const bool early_prep = c->kernel == CAEE_KERNEL_UMMA && c->d.w_dtype == CAEE_E4M3 && c->step_prefill == 0;
  // ... and in steps of <= 16 tokens the one-CTA decision kernel does the split itself, ahead of its wait for the router
  const bool split_in_decide = early_prep && fused && caee_decide_splits_x(c, T);
  if (early_prep && !split_in_decide) caee_launch_umma_prepare(c, x, T, st);
  if (fused) {
    // decode-size step: router GEMM, then ONE kernel for S1-S6 + stats (decide.cu)
    if (!scores && (rc = caee_launch_router_logits(c, x, T, st)) != CAEE_OK) return rc;
    CAEE_CUDA(c, caee_launch_decide(c, scores, T, p, c->any_offload ? nullptr : stats, st, split_in_decide ? x : nullptr));
    if ((rc = after_launch(c, "decision kernel")) != CAEE_OK) return rc;
  } else {
    rc = enqueue_decisions(c, x, scores, T, p, c->idx, c->gate, nullptr, true, st);
    if (rc != CAEE_OK) return rc;
  }
  const bool prof = (size_t)c->prof_used * 2 + 1 < c->prof_ev.size();
  int n_fetch = 0;
  if (c->kernel == CAEE_KERNEL_SIMT) {
    if (prof) cudaEventRecord(c->prof_ev[2 * c->prof_used], st);
    caee_launch_expert_simt(c, x, T, st);
  } else if (!c->any_offload) {
    if (!early_prep) caee_launch_umma_prepare(c, x, T, st);
    if (prof) cudaEventRecord(c->prof_ev[2 * c->prof_used], st);
    if ((rc = caee_launch_expert_umma(c, x, T, 0, -1, 0, st)) != CAEE_OK) return rc;
  } else {
    // S9 (Fig. 8): only the non-resident experts that survived pruning are
    // fetched, one cudaMemcpyAsync each on the side stream, while the resident experts (first
    // in the run list) are already computing on the caller's stream.  The host has to learn
    // which experts survived: this is the one host synchronisation of an offloading step.
    if (!early_prep) caee_launch_umma_prepare(c, x, T, st);
    CAEE_CUDA(c, cudaMemcpyAsync(c->host_meta, c->wl.meta, sizeof(int32_t) * 16, cudaMemcpyDeviceToHost, st));
    CAEE_CUDA(c, cudaMemcpyAsync(c->host_meta + 16, c->wl.run_expert, sizeof(int32_t) * c->wl.max_runs, cudaMemcpyDeviceToHost, st));
    CAEE_CUDA(c, cudaStreamSynchronize(st));
    const int n_runs = c->host_meta[1], n_res = c->host_meta[4];
    const int32_t* run_expert = c->host_meta + 16;
    CAEE_CUDA(c, cudaEventRecord(c->ev_fork, st));                 // staging slots may still be read by the previous step
    CAEE_CUDA(c, cudaStreamWaitEvent(c->side_stream, c->ev_fork, 0));
    struct Seg { int e, begin, count; };
    std::vector<Seg> segs;
    for (int r = n_res; r < n_runs; ++r) {
      if (!segs.empty() && segs.back().e == run_expert[r]) ++segs.back().count;
      else segs.push_back({run_expert[r], r, 1});
    }
    std::vector<uint8_t*> miss_slots;
    if (c->cache) {
      // LFU cache (cache.cu, R30-R32): count the step's routed experts, give every miss a slot
      std::vector<int32_t> executed;
      for (int r = 0; r < n_runs; ++r)
        if (run_expert[r] < c->d.E && (executed.empty() || executed.back() != run_expert[r])) executed.push_back(run_expert[r]);
      std::sort(executed.begin(), executed.end());
      executed.erase(std::unique(executed.begin(), executed.end()), executed.end());
      if ((rc = caee_cache_step(c, executed.data(), (int)executed.size(), &miss_slots)) != CAEE_OK) return rc;
      if (miss_slots.size() != segs.size()) return caee_fail(c, CAEE_ESTATE, "expert cache out of step with the run list (%zu misses, %zu non-resident experts)", miss_slots.size(), segs.size());
      // the misses' image pointers, before any expert kernel of this step (second half of the staging buffer is not
      // needed: write the few changed entries straight from dptr_h, pageable -> staged at call time)
      for (size_t i = 0; i < segs.size(); ++i)
        CAEE_CUDA(c, cudaMemcpyAsync(c->packed.dev_ptrs + segs[i].e, &c->dptr_h[segs[i].e], sizeof(void*), cudaMemcpyHostToDevice, st));
    }
    const int n_ring = (int)c->stage_ring.size();
    cudaEvent_t* pev = (prof && (size_t)c->prof_used * 4 + 3 < c->prof_off_ev.size()) ? &c->prof_off_ev[(size_t)c->prof_used * 4] : nullptr;
    n_fetch = (int)segs.size();
    if (prof) cudaEventRecord(c->prof_ev[2 * c->prof_used], st);
    if (pev) { cudaEventRecord(pev[0], c->side_stream); cudaEventRecord(pev[2], st); }
    if (n_res > 0 && (rc = caee_launch_expert_umma(c, x, T, 0, n_res, 0, st)) != CAEE_OK) return rc;
    if (pev) cudaEventRecord(pev[3], st);
    // Fetched experts run in groups of consecutive misses: the group's copies (side stream, back to back with the
    // previous group's), then ONE expert-kernel launch behind the group's last copy.  Static offload stages the
    // images in the ring: a slot is free again once the launch that last read it is done, so the copy train runs at
    // most one ring ahead of the launches — enqueued in this order, which is what makes the slot events valid.
    const size_t G = c->cache ? 1 : (size_t)std::max(1, std::min<int>(CAEE_FETCH_GROUP, n_ring / 2));
    int ticket = 1;
    std::vector<int> slot_of(G, -1);
    for (size_t i = 0; i < segs.size(); i += G) {
      const size_t j = std::min(segs.size(), i + G) - 1;          // last miss of the group
      for (size_t q = i; q <= j; ++q) {
        const int e = segs[q].e;
        uint8_t* dst;
        if (c->cache) {
          dst = miss_slots[q];
        } else {
          const int sl = (int)(c->ring_next++ % (unsigned)n_ring);
          slot_of[q - i] = sl;
          dst = c->stage_ring[sl];
          CAEE_CUDA(c, cudaStreamWaitEvent(c->side_stream, c->ring_free_ev[sl], 0));
          // the expert's image pointer follows the slot (pinned source: nothing here waits for the stream)
          CAEE_CUDA(c, cudaMemcpyAsync(c->packed.dev_ptrs + e, &c->ring_ptr_pin[sl], sizeof(void*), cudaMemcpyHostToDevice, st));
        }
        CAEE_CUDA(c, cudaMemcpyAsync(dst, c->packed.base[e], c->packed.bytes_per_expert, cudaMemcpyHostToDevice, c->side_stream));
      }
      CAEE_CUDA(c, cudaEventRecord(c->fetch_ev[j], c->side_stream));
      CAEE_CUDA(c, cudaStreamWaitEvent(st, c->fetch_ev[j], 0));
      const int begin = segs[i].begin, count = segs[j].begin + segs[j].count - begin;
      if ((rc = caee_launch_expert_umma(c, x, T, begin, count, ticket++, st)) != CAEE_OK) return rc;
      if (!c->cache)
        for (size_t q = i; q <= j; ++q) CAEE_CUDA(c, cudaEventRecord(c->ring_free_ev[slot_of[q - i]], st));
    }
    if (pev) cudaEventRecord(pev[1], c->side_stream);
  }
  if (prof) cudaEventRecord(c->prof_ev[2 * c->prof_used++ + 1], st);
  // expert parallelism: the o rows of this device's home tokens are still arriving from its peers; the caller
  // synchronises the group and then calls caee_ep_combine
  if (!c->wl.ep_owned) caee_launch_combine(c, T, c->idx, c->gate, y, st);
  if (!fused || c->any_offload) caee_launch_stats(c, stats, p != nullptr, n_fetch, st);
  return after_launch(c, "caee_moe_forward");
}

caee_status caee_moe_forward(caee_ctx* c, const void* x, int32_t T, const caee_prune_params* p, void* y,
                             caee_fwd_stats* stats, void* stream) {
  return forward_impl(c, x, nullptr, T, p, y, stats, stream);
}

caee_status caee_moe_forward_from_scores(caee_ctx* c, const void* x, const float* scores, int32_t T,
                                         const caee_prune_params* p, void* y, caee_fwd_stats* stats, void* stream) {
  if (c && !scores && T > 0) return caee_fail(c, CAEE_EINVAL, "scores is NULL");
  return forward_impl(c, x, scores, T, p, y, stats, stream);
}

caee_status caee_moe_forward_host(caee_ctx* c, const void* x_host, int32_t T, const caee_prune_params* p, void* y_host,
                                  caee_fwd_stats* stats, void* stream) {
  caee_status rc = check_call(c, T);
  if (rc != CAEE_OK) return rc;
  if (T == 0) return CAEE_OK;
  if (!x_host || !y_host) return caee_fail(c, CAEE_EINVAL, "x_host or y_host is NULL");
  DeviceGuard g(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  const size_t esz = c->d.act_dtype == CAEE_F32 ? 4 : 2;
  if (!c->s_in) {
    const size_t cap = (size_t)c->d.max_tokens * c->d.H * esz;
    for (int b = 0; b < 2; ++b) {
      CAEE_CUDA(c, cudaMalloc(&c->hx_d[b], cap));
      CAEE_CUDA(c, cudaMalloc(&c->hy_d[b], cap));
      CAEE_CUDA(c, cudaEventCreateWithFlags(&c->ev_hin[b], cudaEventDisableTiming));
      CAEE_CUDA(c, cudaEventCreateWithFlags(&c->ev_hcmp[b], cudaEventDisableTiming));
      CAEE_CUDA(c, cudaEventCreateWithFlags(&c->ev_hout[b], cudaEventDisableTiming));
      CAEE_CUDA(c, cudaEventRecord(c->ev_hcmp[b], st));     // nothing to wait for yet
      CAEE_CUDA(c, cudaEventRecord(c->ev_hout[b], st));
    }
    CAEE_CUDA(c, cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
    CAEE_CUDA(c, cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
  }
  const int b = (int)(c->host_step++ & 1u);
  const size_t bytes = (size_t)T * c->d.H * esz;
  CAEE_CUDA(c, cudaStreamWaitEvent(c->s_in, c->ev_hcmp[b], 0));      // the step that last read this x buffer is done
  CAEE_CUDA(c, cudaMemcpyAsync(c->hx_d[b], x_host, bytes, cudaMemcpyHostToDevice, c->s_in));
  CAEE_CUDA(c, cudaEventRecord(c->ev_hin[b], c->s_in));
  CAEE_CUDA(c, cudaStreamWaitEvent(st, c->ev_hin[b], 0));
  CAEE_CUDA(c, cudaStreamWaitEvent(st, c->ev_hout[b], 0));           // this y buffer's previous copy-out is done
  rc = forward_impl(c, c->hx_d[b], nullptr, T, p, c->hy_d[b], stats, stream);
  if (rc != CAEE_OK) return rc;
  CAEE_CUDA(c, cudaEventRecord(c->ev_hcmp[b], st));
  CAEE_CUDA(c, cudaStreamWaitEvent(c->s_out, c->ev_hcmp[b], 0));
  CAEE_CUDA(c, cudaMemcpyAsync(y_host, c->hy_d[b], bytes, cudaMemcpyDeviceToHost, c->s_out));
  CAEE_CUDA(c, cudaEventRecord(c->ev_hout[b], c->s_out));
  return CAEE_OK;
}

caee_status caee_host_flush(caee_ctx* c, void* stream) {
  if (!c) return CAEE_EINVAL;
  if (!c->s_out) return CAEE_OK;
  DeviceGuard g(c->device);
  for (int b = 0; b < 2; ++b) CAEE_CUDA(c, cudaStreamWaitEvent((cudaStream_t)stream, c->ev_hout[b], 0));
  return CAEE_OK;
}

// ---------------------------------------------------------------- expert parallelism (include/caee.h)
caee_status caee_set_ep(caee_ctx* c, int32_t rank, int32_t world, const int32_t* owner, void* const* obuf_peers) {
  if (!c) return CAEE_EINVAL;
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaDeviceSynchronize());
  if (world <= 1 || !owner) {                 // back to one device
    c->ep_rank = 0; c->ep_world = 1; c->wl.ep_owned = nullptr; c->wl.ep_world = 1;
    c->ep_owner_h.clear();
    if (c->weights_partial) c->have_weights = false;    // only this rank's experts were loaded: set the weights again
    return CAEE_OK;
  }
  if (world > CAEE_EP_MAX) return caee_fail(c, CAEE_EINVAL, "world=%d exceeds CAEE_EP_MAX=%d", world, CAEE_EP_MAX);
  if (rank < 0 || rank >= world) return caee_fail(c, CAEE_EINVAL, "rank=%d out of range for world=%d", rank, world);
  if (!obuf_peers) return caee_fail(c, CAEE_EINVAL, "obuf_peers is NULL");
  const int E = c->d.E;
  std::vector<uint8_t> owned(E);
  for (int e = 0; e < E; ++e) {
    if (owner[e] < 0 || owner[e] >= world) return caee_fail(c, CAEE_EINVAL, "owner[%d]=%d out of range", e, owner[e]);
    owned[e] = owner[e] == rank;
  }
  for (int r = 0; r < world; ++r)
    if (!obuf_peers[r]) return caee_fail(c, CAEE_EINVAL, "obuf_peers[%d] is NULL", r);
  if (obuf_peers[rank] != (void*)c->obuf) return caee_fail(c, CAEE_EINVAL, "obuf_peers[rank] must be this context's own buffer (caee_ep_obuf)");
  caee_status rc;
  if (!c->ep_owned && (rc = dev_alloc(c, &c->ep_owned, (size_t)E)) != CAEE_OK) return rc;
  if (!c->ep_owner && (rc = dev_alloc(c, &c->ep_owner, (size_t)E)) != CAEE_OK) return rc;
  CAEE_CUDA(c, cudaMemcpy(c->ep_owned, owned.data(), E, cudaMemcpyHostToDevice));
  CAEE_CUDA(c, cudaMemcpy(c->ep_owner, owner, sizeof(int32_t) * E, cudaMemcpyHostToDevice));
  if (c->weights_partial && c->have_weights)
    for (int e = 0; e < E; ++e)
      if (owner[e] == rank && !c->wg_h[e]) { c->have_weights = false; break; }   // a newly owned expert was never loaded
  c->ep_owner_h.assign(owner, owner + E);
  c->ep_rank = rank; c->ep_world = world;
  c->wl.ep_owned = c->ep_owned; c->wl.ep_world = world;
  for (int r = 0; r < CAEE_EP_MAX; ++r) c->wl.ep_obuf[r] = r < world ? (float*)obuf_peers[r] : nullptr;
  return CAEE_OK;
}

caee_status caee_ep_obuf(caee_ctx* c, void** out, int64_t* bytes) {
  if (!c) return CAEE_EINVAL;
  if (!out) return caee_fail(c, CAEE_EINVAL, "out is NULL");
  *out = c->obuf;
  if (bytes) *bytes = (int64_t)sizeof(float) * c->d.max_tokens * (c->d.k + c->d.S) * c->d.H;
  return CAEE_OK;
}

caee_status caee_ep_ipc_export(caee_ctx* c, void* handle64) {
  if (!c) return CAEE_EINVAL;
  if (!handle64) return caee_fail(c, CAEE_EINVAL, "handle64 is NULL");
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaIpcGetMemHandle(reinterpret_cast<cudaIpcMemHandle_t*>(handle64), c->obuf));
  return CAEE_OK;
}

caee_status caee_ep_ipc_open(caee_ctx* c, const void* handle64, void** out) {
  if (!c) return CAEE_EINVAL;
  if (!handle64 || !out) return caee_fail(c, CAEE_EINVAL, "handle64 or out is NULL");
  DeviceGuard g(c->device);
  cudaIpcMemHandle_t h;
  memcpy(&h, handle64, sizeof(h));
  CAEE_CUDA(c, cudaIpcOpenMemHandle(out, h, cudaIpcMemLazyEnablePeerAccess));
  return CAEE_OK;
}

caee_status caee_ep_ipc_close(caee_ctx* c, void* peer_ptr) {
  if (!c) return CAEE_EINVAL;
  DeviceGuard g(c->device);
  if (peer_ptr) CAEE_CUDA(c, cudaIpcCloseMemHandle(peer_ptr));
  return CAEE_OK;
}

caee_status caee_ep_combine(caee_ctx* c, int32_t T, void* y, void* stream) {
  caee_status rc = check_call(c, T);
  if (rc != CAEE_OK) return rc;
  if (!c->wl.ep_owned) return caee_fail(c, CAEE_ESTATE, "caee_ep_combine before caee_set_ep");
  if (T == 0) return CAEE_OK;
  if (!y) return caee_fail(c, CAEE_EINVAL, "y is NULL");
  DeviceGuard g(c->device);
  const int per = caee_ceil_div(T, c->ep_world), lo = std::min(T, c->ep_rank * per), hi = std::min(T, lo + per);
  caee_launch_combine(c, T, c->idx, c->gate, y, (cudaStream_t)stream, lo, hi);
  return after_launch(c, "caee_ep_combine");
}

caee_status caee_ep_plan(caee_ctx* c, int32_t* counts, int32_t* offs, int32_t* tok, int32_t* slot, int32_t* expert, void* stream) {
  if (!c) return CAEE_EINVAL;
  if (!c->wl.ep_owned) return caee_fail(c, CAEE_ESTATE, "caee_ep_plan before caee_set_ep");
  if (!counts || !offs || !tok || !slot || !expert) return caee_fail(c, CAEE_EINVAL, "an output pointer is NULL");
  DeviceGuard g(c->device);
  caee_launch_ep_plan(c, c->ep_owner, c->ep_world, counts, offs, tok, slot, expert, (cudaStream_t)stream);
  return after_launch(c, "caee_ep_plan");
}

caee_status caee_profile(caee_ctx* c, int32_t n_slots) {
  if (!c) return CAEE_EINVAL;
  if (n_slots < 0 || n_slots > 65536) return caee_fail(c, CAEE_EINVAL, "n_slots must be in 0..65536");
  DeviceGuard g(c->device);
  CAEE_CUDA(c, cudaDeviceSynchronize());
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  c->prof_ev.assign((size_t)n_slots * 2, nullptr);
  c->prof_used = 0;
  for (auto& e : c->prof_ev) CAEE_CUDA(c, cudaEventCreate(&e));
  for (cudaEvent_t e : c->prof_off_ev) cudaEventDestroy(e);
  c->prof_off_ev.assign(c->any_offload ? (size_t)n_slots * 4 : 0, nullptr);
  for (auto& e : c->prof_off_ev) CAEE_CUDA(c, cudaEventCreate(&e));
  return CAEE_OK;
}

caee_status caee_profile_read_offload(caee_ctx* c, int32_t cap, float* copy_ms, float* resident_ms, float* lead_ms, int32_t* n_out) {
  if (!c) return CAEE_EINVAL;
  if (!copy_ms || !resident_ms || !lead_ms || !n_out) return caee_fail(c, CAEE_EINVAL, "an output pointer is NULL");
  DeviceGuard g(c->device);
  const int n = std::min<int>({c->prof_used, cap, (int)(c->prof_off_ev.size() / 4)});
  for (int i = 0; i < n; ++i) {
    cudaEvent_t* ev = &c->prof_off_ev[(size_t)i * 4];
    CAEE_CUDA(c, cudaEventSynchronize(ev[1]));
    CAEE_CUDA(c, cudaEventSynchronize(ev[3]));
    CAEE_CUDA(c, cudaEventElapsedTime(&copy_ms[i], ev[0], ev[1]));       // the step's copy train, first copy .. last copy
    CAEE_CUDA(c, cudaEventElapsedTime(&resident_ms[i], ev[2], ev[3]));   // the resident experts' launch
    CAEE_CUDA(c, cudaEventElapsedTime(&lead_ms[i], ev[0], ev[3]));       // copy train start .. resident launch done
  }
  *n_out = n;
  return CAEE_OK;
}

caee_status caee_profile_read(caee_ctx* c, float* expert_ms, int32_t* n_out) {
  if (!c) return CAEE_EINVAL;
  if (!expert_ms || !n_out) return caee_fail(c, CAEE_EINVAL, "expert_ms or n_out is NULL");
  DeviceGuard g(c->device);
  for (int i = 0; i < c->prof_used; ++i) {
    CAEE_CUDA(c, cudaEventSynchronize(c->prof_ev[2 * i + 1]));
    CAEE_CUDA(c, cudaEventElapsedTime(&expert_ms[i], c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
  }
  *n_out = c->prof_used;
  c->prof_used = 0;
  return CAEE_OK;
}

caee_status caee_last_routing(caee_ctx* c, int32_t T, int32_t* idx, float* gate, void* stream) {
  caee_status rc = check_call(c, T);
  if (rc != CAEE_OK) return rc;
  if (T == 0) return CAEE_OK;
  DeviceGuard g(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  if (idx) CAEE_CUDA(c, cudaMemcpyAsync(idx, c->idx, sizeof(int32_t) * T * c->d.k, cudaMemcpyDeviceToDevice, st));
  if (gate) CAEE_CUDA(c, cudaMemcpyAsync(gate, c->gate, sizeof(float) * T * c->d.k, cudaMemcpyDeviceToDevice, st));
  return CAEE_OK;
}

}  // extern "C"
