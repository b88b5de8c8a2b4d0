"""Thin ctypes binding over libcaee.so: same names as include/caee.h, argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; PyTorch is used by callers
for device memory and streams.  Importing this module fails loudly when the library has not
been built (python -m paper_2606_29982_b200.build): there is no CPU fallback.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcaee.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_29982_b200.build` "
                      "(libcaee has no CPU fallback)")
_lib = C.CDLL(LIB_PATH)

CAEE_OK, CAEE_EINVAL, CAEE_ESHAPE, CAEE_EDTYPE, CAEE_ENOMEM, CAEE_ECUDA, CAEE_ESTATE, CAEE_EUNSUPPORTED = 0, -1, -2, -3, -4, -5, -6, -7
CAEE_F32, CAEE_BF16, CAEE_E4M3 = 0, 1, 2
CAEE_SCORE_SOFTMAX, CAEE_SCORE_SIGMOID = 0, 1
CAEE_PRUNE_NONE, CAEE_PRUNE_THRESH, CAEE_PRUNE_CIR, CAEE_PRUNE_RANK, CAEE_PRUNE_FRAC = 0, 1, 2, 3, 4
CAEE_COMP_ALL_TOKENS, CAEE_KEEP_TOP1, CAEE_COMP_RANDOM, CAEE_IMP_BOUND = 1, 2, 4, 8
CAEE_KERNEL_AUTO, CAEE_KERNEL_SIMT, CAEE_KERNEL_UMMA = 0, 1, 2

EXPORTS = ["caee_create", "caee_destroy", "caee_last_error", "caee_set_router", "caee_set_weights",
           "caee_set_partitions", "caee_set_residency", "caee_set_cost_table", "caee_calibrate_cost", "caee_calibrate_points",
           "caee_get_cost_table", "caee_launch_count", "caee_route", "caee_route_noalloc",
           "caee_route_from_scores", "caee_prune", "caee_moe_forward", "caee_moe_forward_from_scores",
           "caee_moe_forward_host", "caee_host_flush", "caee_last_routing", "caee_profile", "caee_profile_read", "caee_profile_read_offload", "caee_version",
           "caee_cache_create", "caee_cache_destroy", "caee_cache_attach", "caee_cache_read_stats", "caee_cache_snapshot",
           "caee_set_ep", "caee_ep_obuf", "caee_ep_ipc_export", "caee_ep_ipc_open", "caee_ep_ipc_close", "caee_ep_combine",
           "caee_ep_plan"]


class caee_layer_desc(C.Structure):
    _fields_ = [("H", C.c_int32), ("I", C.c_int32), ("E", C.c_int32), ("S", C.c_int32), ("k", C.c_int32),
                ("n_group", C.c_int32), ("topk_group", C.c_int32), ("score_fn", C.c_int32), ("norm_topk", C.c_int32),
                ("routed_scale", C.c_float), ("act_dtype", C.c_int32), ("w_dtype", C.c_int32), ("D", C.c_int32),
                ("max_tokens", C.c_int32), ("expert_kernel", C.c_int32), ("device", C.c_int32)]


class caee_expert_weights(C.Structure):
    _fields_ = [(n, C.POINTER(C.c_void_p)) for n in ("gate", "up", "down", "gate_scale", "up_scale", "down_scale")]


class caee_prune_params(C.Structure):
    _fields_ = [("mode", C.c_int32), ("flags", C.c_int32), ("theta", C.c_double), ("eps", C.c_double)]


class caee_prune_out(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("act", "must", "keep", "importance", "load", "scalars", "n_run", "expert_ids",
                                          "offs", "tok", "slot", "wt")]


class caee_fwd_stats(C.Structure):
    _fields_ = [("F_base", C.c_int64), ("F_cost_dense", C.c_int64), ("F_cost", C.c_int64), ("F_imp", C.c_int64),
                ("weight_bytes", C.c_int64), ("h2d_bytes", C.c_int64), ("n_act", C.c_int32), ("n_keep", C.c_int32),
                ("n_run", C.c_int32), ("n_fetch", C.c_int32), ("load", C.c_int64 * 64)]


class caee_calib_opts(C.Structure):
    _fields_ = [("n_sizes", C.c_int32), ("iters", C.c_int32), ("min_bytes", C.c_int64), ("max_bytes", C.c_int64),
                ("apply", C.c_int32), ("reserved", C.c_int32)]


class caee_cost_fit(C.Structure):
    _fields_ = [("slope_ns_per_byte", C.c_double), ("intercept_ns", C.c_double), ("r2", C.c_double),
                ("gbytes_per_s", C.c_double), ("n_points", C.c_int32), ("valid", C.c_int32)]


class caee_cache_stats(C.Structure):
    _fields_ = [("hits", C.c_int64), ("misses", C.c_int64), ("evictions", C.c_int64), ("h2d_bytes", C.c_int64)]


_ctx_p = C.c_void_p
_lib.caee_cache_create.argtypes = [C.c_int32, C.POINTER(C.c_void_p)]
_lib.caee_cache_destroy.argtypes = [C.c_void_p]
_lib.caee_cache_destroy.restype = None
_lib.caee_cache_attach.argtypes = [C.c_void_p, _ctx_p, C.c_int32]
_lib.caee_cache_read_stats.argtypes = [C.c_void_p, C.POINTER(caee_cache_stats)]
_lib.caee_cache_snapshot.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_create.argtypes = [C.POINTER(caee_layer_desc), C.POINTER(_ctx_p)]
_lib.caee_destroy.argtypes = [_ctx_p]
_lib.caee_last_error.argtypes = [_ctx_p]
_lib.caee_last_error.restype = C.c_char_p
_lib.caee_version.restype = C.c_char_p
_lib.caee_set_router.argtypes = [_ctx_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_set_weights.argtypes = [_ctx_p, C.POINTER(caee_expert_weights), C.c_int32]
_lib.caee_set_partitions.argtypes = [_ctx_p, C.c_void_p, C.c_int32]
_lib.caee_set_residency.argtypes = [_ctx_p, C.c_void_p]
_lib.caee_set_cost_table.argtypes = [_ctx_p, C.c_void_p, C.c_void_p]
_lib.caee_calibrate_cost.argtypes = [_ctx_p, C.POINTER(caee_calib_opts), C.POINTER(caee_cost_fit)]
_lib.caee_calibrate_points.argtypes = [_ctx_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_get_cost_table.argtypes = [_ctx_p, C.c_void_p, C.c_void_p]
_lib.caee_launch_count.argtypes = [_ctx_p, C.c_void_p]
_lib.caee_route.argtypes = [_ctx_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_route_noalloc.argtypes = ([C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p] + [C.c_int32] * 8 +
                                    [C.c_void_p] * 4)
_lib.caee_route_from_scores.argtypes = [_ctx_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_prune.argtypes = [_ctx_p, C.POINTER(caee_prune_params), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p,
                            C.POINTER(caee_prune_out), C.c_void_p]
_lib.caee_moe_forward.argtypes = [_ctx_p, C.c_void_p, C.c_int32, C.POINTER(caee_prune_params), C.c_void_p, C.c_void_p,
                                  C.c_void_p]
_lib.caee_moe_forward_from_scores.argtypes = [_ctx_p, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(caee_prune_params),
                                              C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_moe_forward_host.argtypes = [_ctx_p, C.c_void_p, C.c_int32, C.POINTER(caee_prune_params), C.c_void_p, C.c_void_p,
                                       C.c_void_p]
_lib.caee_host_flush.argtypes = [_ctx_p, C.c_void_p]
_lib.caee_last_routing.argtypes = [_ctx_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_profile.argtypes = [_ctx_p, C.c_int32]
_lib.caee_profile_read.argtypes = [_ctx_p, C.c_void_p, C.c_void_p]
_lib.caee_profile_read_offload.argtypes = [_ctx_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.caee_set_ep.argtypes = [_ctx_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
_lib.caee_ep_obuf.argtypes = [_ctx_p, C.c_void_p, C.c_void_p]
_lib.caee_ep_ipc_export.argtypes = [_ctx_p, C.c_void_p]
_lib.caee_ep_ipc_open.argtypes = [_ctx_p, C.c_void_p, C.c_void_p]
_lib.caee_ep_ipc_close.argtypes = [_ctx_p, C.c_void_p]
_lib.caee_ep_combine.argtypes = [_ctx_p, C.c_int32, C.c_void_p, C.c_void_p]
_lib.caee_ep_plan.argtypes = [_ctx_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
for _n in EXPORTS:
    if _n not in ("caee_last_error", "caee_version", "caee_cache_destroy"):
        getattr(_lib, _n).restype = C.c_int32


class CaeeError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"caee error {code}: {msg}")
        self.code = code


def _ptr(t):
    """Device/host address of a tensor, numpy array or raw int (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        return t.data_ptr()
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return int(t)


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if isinstance(stream, torch.cuda.Stream) else int(stream)


def _check(rc, ctx=None):
    if rc != CAEE_OK:
        raise CaeeError(rc, (_lib.caee_last_error(ctx) or b"").decode())


# ---- the ABI, name for name -------------------------------------------------------------
def caee_version():
    return _lib.caee_version().decode()


def caee_create(desc: caee_layer_desc):
    ctx = _ctx_p()
    _check(_lib.caee_create(C.byref(desc), C.byref(ctx)))
    return ctx


def caee_destroy(ctx):
    _check(_lib.caee_destroy(ctx))


def caee_last_error(ctx=None):
    return (_lib.caee_last_error(ctx) or b"").decode()


def caee_set_router(ctx, W_r, b_logit=None, corr_bias=None):
    _check(_lib.caee_set_router(ctx, _ptr(W_r), _ptr(b_logit), _ptr(corr_bias)), ctx)


def _table(items):
    if items is None:
        return None
    arr = (C.c_void_p * len(items))()
    for i, t in enumerate(items):
        arr[i] = _ptr(t)
    return arr


def caee_set_weights(ctx, gate, up, down, gate_scale=None, up_scale=None, down_scale=None, pack=1):
    tabs = [_table(v) for v in (gate, up, down, gate_scale, up_scale, down_scale)]
    w = caee_expert_weights(*[C.cast(t, C.POINTER(C.c_void_p)) if t is not None else None for t in tabs])
    _check(_lib.caee_set_weights(ctx, C.byref(w), int(pack)), ctx)


def caee_set_partitions(ctx, part_of_expert, D):
    p = np.ascontiguousarray(part_of_expert, dtype=np.int32)
    _check(_lib.caee_set_partitions(ctx, _ptr(p), int(D)), ctx)


def caee_set_residency(ctx, resident):
    r = np.ascontiguousarray(resident, dtype=np.uint8)
    _check(_lib.caee_set_residency(ctx, _ptr(r)), ctx)


def caee_set_cost_table(ctx, ticks_resident, ticks_miss=None):
    tr = np.ascontiguousarray(ticks_resident, dtype=np.int64)
    tm = None if ticks_miss is None else np.ascontiguousarray(ticks_miss, dtype=np.int64)
    _check(_lib.caee_set_cost_table(ctx, _ptr(tr), _ptr(tm)), ctx)


def caee_calibrate_cost(ctx, opts: caee_calib_opts = None):
    fits = (caee_cost_fit * 2)()
    _check(_lib.caee_calibrate_cost(ctx, C.byref(opts) if opts is not None else None, fits), ctx)
    return fits[0], fits[1]


def caee_calibrate_points(ctx, tier, cap=16):
    """(bytes[n], ns[n]) of the last calibration's timed points for a tier."""
    b, t = np.zeros(cap, np.float64), np.zeros(cap, np.float64)
    n = C.c_int32(0)
    _check(_lib.caee_calibrate_points(ctx, int(tier), int(cap), _ptr(b), _ptr(t), C.addressof(n)), ctx)
    return b[:n.value].copy(), t[:n.value].copy()


def caee_get_cost_table(ctx, E):
    tr, tm = np.zeros(E, np.int64), np.zeros(E, np.int64)
    _check(_lib.caee_get_cost_table(ctx, _ptr(tr), _ptr(tm)), ctx)
    return tr, tm


def caee_launch_count(ctx):
    n = C.c_int64(0)
    _check(_lib.caee_launch_count(ctx, C.addressof(n)), ctx)
    return n.value


def caee_route(ctx, x, T, scores, idx, gate, stream=None):
    _check(_lib.caee_route(ctx, _ptr(x), int(T), _ptr(scores), _ptr(idx), _ptr(gate), _stream(stream)), ctx)


def caee_route_noalloc(device, x, act_dtype, Wr, b_logit, corr_bias, T, H, E, k, n_group, topk_group, score_fn, norm_topk,
                       scores, idx, gate, stream=None):
    _check(_lib.caee_route_noalloc(int(device), _ptr(x), int(act_dtype), _ptr(Wr), _ptr(b_logit), _ptr(corr_bias), int(T), int(H),
                                   int(E), int(k), int(n_group), int(topk_group), int(score_fn), int(norm_topk), _ptr(scores),
                                   _ptr(idx), _ptr(gate), _stream(stream)))


def caee_route_from_scores(ctx, scores, T, idx, gate, stream=None):
    _check(_lib.caee_route_from_scores(ctx, _ptr(scores), int(T), _ptr(idx), _ptr(gate), _stream(stream)), ctx)


def caee_prune(ctx, params, scores, T, idx, gate, out: caee_prune_out = None, stream=None):
    _check(_lib.caee_prune(ctx, C.byref(params) if params is not None else None, _ptr(scores), int(T), _ptr(idx),
                           _ptr(gate), C.byref(out) if out is not None else None, _stream(stream)), ctx)


def caee_moe_forward(ctx, x, T, params, y, stats=None, stream=None):
    _check(_lib.caee_moe_forward(ctx, _ptr(x), int(T), C.byref(params) if params is not None else None, _ptr(y),
                                 _ptr(stats), _stream(stream)), ctx)


def caee_moe_forward_from_scores(ctx, x, scores, T, params, y, stats=None, stream=None):
    _check(_lib.caee_moe_forward_from_scores(ctx, _ptr(x), _ptr(scores), int(T),
                                             C.byref(params) if params is not None else None, _ptr(y), _ptr(stats),
                                             _stream(stream)), ctx)


def caee_moe_forward_host(ctx, x_host, T, params, y_host, stats=None, stream=None):
    _check(_lib.caee_moe_forward_host(ctx, _ptr(x_host), int(T), C.byref(params) if params is not None else None,
                                      _ptr(y_host), _ptr(stats), _stream(stream)), ctx)


def caee_host_flush(ctx, stream=None):
    _check(_lib.caee_host_flush(ctx, _stream(stream)), ctx)


def caee_last_routing(ctx, T, idx, gate, stream=None):
    _check(_lib.caee_last_routing(ctx, int(T), _ptr(idx), _ptr(gate), _stream(stream)), ctx)


def caee_profile(ctx, n_slots):
    _check(_lib.caee_profile(ctx, int(n_slots)), ctx)


def caee_profile_read(ctx, n_slots):
    ms = np.zeros(max(int(n_slots), 1), np.float32)
    n = C.c_int32(0)
    _check(_lib.caee_profile_read(ctx, _ptr(ms), C.addressof(n)), ctx)
    return ms[:n.value].copy()


def caee_profile_read_offload(ctx, n_slots):
    """(copy_ms, resident_ms, lead_ms) per recorded offloading step; call before caee_profile_read."""
    cap = max(int(n_slots), 1)
    a, b, c_ = (np.zeros(cap, np.float32) for _ in range(3))
    n = C.c_int32(0)
    _check(_lib.caee_profile_read_offload(ctx, cap, _ptr(a), _ptr(b), _ptr(c_), C.addressof(n)), ctx)
    return a[:n.value].copy(), b[:n.value].copy(), c_[:n.value].copy()


def caee_cache_create(n_slots):
    cache = C.c_void_p()
    _check(_lib.caee_cache_create(int(n_slots), C.byref(cache)))
    return cache


def caee_cache_destroy(cache):
    _lib.caee_cache_destroy(cache)


def caee_cache_attach(cache, ctx, layer_id):
    _check(_lib.caee_cache_attach(cache, ctx, int(layer_id)), ctx)


def caee_cache_read_stats(cache):
    st = caee_cache_stats()
    _check(_lib.caee_cache_read_stats(cache, C.byref(st)))
    return st


def caee_cache_snapshot(cache, n_slots):
    """[(layer, expert, freq) or None] per slot."""
    layer, expert = np.zeros(n_slots, np.int32), np.zeros(n_slots, np.int32)
    freq = np.zeros(n_slots, np.int64)
    _check(_lib.caee_cache_snapshot(cache, _ptr(layer), _ptr(expert), _ptr(freq)))
    return [None if layer[s] < 0 else (int(layer[s]), int(expert[s]), int(freq[s])) for s in range(n_slots)]


def caee_set_ep(ctx, rank, world, owner=None, obuf_peers=None):
    """owner: int32 [E] (None: expert parallelism off); obuf_peers: one device address per rank."""
    o = None if owner is None else np.ascontiguousarray(owner, dtype=np.int32)
    peers = None
    if obuf_peers is not None:
        peers = (C.c_void_p * len(obuf_peers))(*[int(p) for p in obuf_peers])
    _check(_lib.caee_set_ep(ctx, int(rank), int(world), _ptr(o), C.cast(peers, C.c_void_p) if peers is not None else None), ctx)


def caee_ep_obuf(ctx):
    """(device address, bytes) of this context's o buffer (the target of its peers' stores)."""
    p, n = C.c_void_p(), C.c_int64(0)
    _check(_lib.caee_ep_obuf(ctx, C.addressof(p), C.addressof(n)), ctx)
    return p.value, n.value


def caee_ep_ipc_export(ctx):
    h = (C.c_ubyte * 64)()
    _check(_lib.caee_ep_ipc_export(ctx, C.addressof(h)), ctx)
    return bytes(h)


def caee_ep_ipc_open(ctx, handle):
    h = (C.c_ubyte * 64)(*handle)
    p = C.c_void_p()
    _check(_lib.caee_ep_ipc_open(ctx, C.addressof(h), C.addressof(p)), ctx)
    return p.value


def caee_ep_ipc_close(ctx, peer_ptr):
    _check(_lib.caee_ep_ipc_close(ctx, int(peer_ptr)), ctx)


def caee_ep_combine(ctx, T, y, stream=None):
    _check(_lib.caee_ep_combine(ctx, int(T), _ptr(y), _stream(stream)), ctx)


def caee_ep_plan(ctx, counts, offs, tok, slot, expert, stream=None):
    _check(_lib.caee_ep_plan(ctx, _ptr(counts), _ptr(offs), _ptr(tok), _ptr(slot), _ptr(expert), _stream(stream)), ctx)


# ---- small conveniences for tests / bench (marshalling only) -----------------------------
def layer_desc(cfg, max_tokens, expert_kernel=CAEE_KERNEL_AUTO, device=-1):
    """caee_layer_desc from a workloads.LayerConfig."""
    return caee_layer_desc(cfg.H, cfg.I, cfg.E, cfg.S, cfg.k, cfg.n_group, cfg.topk_group, cfg.score_fn,
                           int(cfg.norm_topk), cfg.routed_scale, cfg.act_dtype, cfg.w_dtype, cfg.D, int(max_tokens),
                           expert_kernel, device)


def caee_kernel_is_simt(cfg, kernel):
    """Mirror of caee_create's AUTO rule: which expert kernel a descriptor resolves to."""
    umma_ok = (cfg.w_dtype in (CAEE_BF16, CAEE_E4M3) and cfg.act_dtype == CAEE_BF16 and cfg.H % 256 == 0
               and cfg.I % 128 == 0)
    return kernel == CAEE_KERNEL_SIMT or (kernel == CAEE_KERNEL_AUTO and not umma_ok)


def prune_params(mode, theta=0.0, flags=0, eps=None):
    """eps (a bound on F_imp in gate units) switches CAEE_IMP_BOUND on."""
    if eps is not None:
        flags |= CAEE_IMP_BOUND
    return caee_prune_params(int(mode), int(flags), float(theta), 0.0 if eps is None else float(eps))


class PruneOut:
    """Device buffers for every optional output of caee_prune."""

    def __init__(self, E, D, T, k, device):
        o = dict(act=torch.zeros(E, dtype=torch.uint8, device=device), must=torch.zeros(E, dtype=torch.uint8, device=device),
                 keep=torch.zeros(E, dtype=torch.uint8, device=device), importance=torch.zeros(E, dtype=torch.int64, device=device),
                 load=torch.zeros(D, dtype=torch.int64, device=device), scalars=torch.zeros(8, dtype=torch.int64, device=device),
                 n_run=torch.zeros(1, dtype=torch.int32, device=device), expert_ids=torch.zeros(E, dtype=torch.int32, device=device),
                 offs=torch.zeros(E + 1, dtype=torch.int32, device=device), tok=torch.zeros(max(T * k, 1), dtype=torch.int32, device=device),
                 slot=torch.zeros(max(T * k, 1), dtype=torch.int32, device=device), wt=torch.zeros(max(T * k, 1), dtype=torch.float32, device=device))
        self.t = o
        self.struct = caee_prune_out(*[o[n].data_ptr() for n, _ in caee_prune_out._fields_])


def read_stats(stats_tensor):
    """Decode a uint8 device tensor of sizeof(caee_fwd_stats) bytes."""
    raw = stats_tensor.cpu().numpy().tobytes()
    return caee_fwd_stats.from_buffer_copy(raw)


def stats_buffer(device):
    return torch.zeros(C.sizeof(caee_fwd_stats), dtype=torch.uint8, device=device)
