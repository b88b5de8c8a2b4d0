"""ctypes loader for the CPU oracle (oracle/caee_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  Nothing under
paper_2606_29982_b200/ imports this module and this module imports nothing
from there.  All arrays are numpy; bf16 travels as uint16 bit patterns and
e4m3 as uint8 codes.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

DT_F32, DT_BF16, DT_E4M3 = 0, 1, 2
SCORE_SOFTMAX, SCORE_SIGMOID = 0, 1
MODE_NONE, MODE_THRESH, MODE_CIR, MODE_RANK, MODE_FRAC = 0, 1, 2, 3, 4
FLAG_COMP_ALL_TOKENS, FLAG_KEEP_TOP1, FLAG_COMP_RANDOM, FLAG_IMP_BOUND = 1, 2, 4, 8
FIX_ONE = float(2 ** 40)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_f_cost.restype = C.c_int64
        _lib.oracle_cost_ticks.restype = C.c_int64
        _lib.oracle_cost_ticks.argtypes = [C.c_double, C.c_double, C.c_int64]
        _lib.oracle_e4m3_value.restype = C.c_double
        _lib.oracle_fmix32.restype = C.c_uint32
        _lib.oracle_fmix32.argtypes = [C.c_uint32]
        _lib.oracle_unit_draw.restype = C.c_float
        _lib.oracle_unit_draw.argtypes = [C.c_int, C.c_int]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


def act_dtype_of(x):
    return DT_F32 if x.dtype == np.float32 else DT_BF16


def w_dtype_of(w):
    return {np.dtype(np.float32): DT_F32, np.dtype(np.uint16): DT_BF16, np.dtype(np.uint8): DT_E4M3}[w.dtype]


def scores(x, Wr, b_logit, score_fn):
    T, H = x.shape
    E = Wr.shape[0]
    x = np.ascontiguousarray(x)
    Wr = _c(Wr, np.float32)
    b = _c(b_logit, np.float32)
    s = np.empty((T, E), np.float32)
    rc = lib().oracle_scores(_p(x), act_dtype_of(x), _p(Wr), _p(b), T, H, E, score_fn, _p(s))
    assert rc == 0
    return s


def route(s, corr_bias, k, n_group=1, topk_group=1, norm_topk=True):
    s = _c(s, np.float32)
    T, E = s.shape
    cb = _c(corr_bias, np.float32)
    idx = np.empty((T, k), np.int32)
    gate = np.empty((T, k), np.float32)
    rc = lib().oracle_route(_p(s), _p(cb), T, E, k, n_group, topk_group, int(norm_topk), _p(idx), _p(gate))
    assert rc == 0, "invalid route arguments"
    return idx, gate


def importance(idx, gate, E):
    idx = _c(idx, np.int32)
    gate = _c(gate, np.float32)
    T, k = idx.shape
    act = np.empty(E, np.uint8)
    I_fix = np.empty(E, np.int64)
    lib().oracle_importance(_p(idx), _p(gate), T, E, k, _p(act), _p(I_fix))
    return act, I_fix


def effective_cost(resident, ticks_resident, ticks_miss):
    resident = _c(resident, np.uint8)
    tr = _c(ticks_resident, np.int64)
    tm = _c(ticks_miss, np.int64)
    w = np.empty(resident.shape[0], np.int64)
    lib().oracle_effective_cost(_p(resident), _p(tr), _p(tm), resident.shape[0], _p(w))
    return w


def f_cost(mask, w, part, D):
    mask = _c(mask, np.uint8)
    w = _c(w, np.int64)
    part = _c(part, np.int32)
    load = np.empty(D, np.int64)
    F = lib().oracle_f_cost(_p(mask), _p(w), _p(part), mask.shape[0], D, _p(load))
    return int(F), load


def cost_ticks(slope_ns_per_byte, intercept_ns, nbytes):
    return int(lib().oracle_cost_ticks(float(slope_ns_per_byte), float(intercept_ns), int(nbytes)))


def prune(mode, theta, flags, idx, gate, E, w, part, D, eps=0.0):
    idx = _c(idx, np.int32)
    gate = _c(gate, np.float32)
    w = _c(w, np.int64)
    part = _c(part, np.int32)
    T, k = idx.shape
    act = np.empty(E, np.uint8)
    I_fix = np.empty(E, np.int64)
    must = np.empty(E, np.uint8)
    keep = np.empty(E, np.uint8)
    load = np.empty(D, np.int64)
    sc = np.empty(7, np.int64)
    rc = lib().oracle_prune(int(mode), C.c_double(theta), int(flags), C.c_double(eps), _p(idx), _p(gate), T, E, k, _p(w),
                            _p(part), D, _p(act), _p(I_fix), _p(must), _p(keep), _p(load), _p(sc))
    assert rc == 0
    return dict(act=act, I_fix=I_fix, must=must, keep=keep, load=load, F_base=int(sc[0]),
                F_cost_dense=int(sc[1]), F_cost=int(sc[2]), F_imp_fix=int(sc[3]), n_act=int(sc[4]),
                n_must=int(sc[5]), n_keep=int(sc[6]))


def compensate(s, corr_bias, keep, idx, gate, norm_topk=True, flags=0):
    s = _c(s, np.float32)
    cb = _c(corr_bias, np.float32)
    keep = _c(keep, np.uint8)
    idx = np.array(idx, dtype=np.int32, order="C", copy=True)
    gate = np.array(gate, dtype=np.float32, order="C", copy=True)
    T, E = s.shape
    k = idx.shape[1]
    lib().oracle_compensate(_p(s), _p(cb), _p(keep), T, E, k, int(norm_topk), int(flags), _p(idx), _p(gate))
    return idx, gate


def compact(idx, gate, E):
    idx = _c(idx, np.int32)
    gate = _c(gate, np.float32)
    T, k = idx.shape
    n_run = C.c_int32(0)
    expert_ids = np.empty(E, np.int32)
    offs = np.empty(E + 1, np.int32)
    tok = np.empty(T * k, np.int32)
    slot = np.empty(T * k, np.int32)
    wt = np.empty(T * k, np.float32)
    lib().oracle_compact(_p(idx), _p(gate), T, E, k, C.byref(n_run), _p(expert_ids), _p(offs), _p(tok),
                         _p(slot), _p(wt))
    r = n_run.value
    n = int(offs[r])
    return dict(n_run=r, expert_ids=expert_ids[:r].copy(), offs=offs[:r + 1].copy(), tok=tok[:n].copy(),
                slot=slot[:n].copy(), wt=wt[:n].copy())


def expert_ffn(x_row, Wg, Wu, Wd, sg=None, su=None, sd=None):
    """One expert on one token -> o[H] fp64.  Wg, Wu: [I,H]; Wd: [H,I]."""
    x_row = np.ascontiguousarray(x_row)
    I, H = Wg.shape
    Wg, Wu, Wd = (np.ascontiguousarray(a) for a in (Wg, Wu, Wd))
    sg, su, sd = (_c(a, np.float32) for a in (sg, su, sd))
    o = np.empty(H, np.float64)
    lib().oracle_expert_ffn(_p(x_row), act_dtype_of(x_row), _p(Wg), _p(Wu), _p(Wd), w_dtype_of(Wg), _p(sg),
                            _p(su), _p(sd), H, I, _p(o))
    return o


def moe_tokens(x, tokens, idx, gate, Wg, Wu, Wd, E, S, routed_scale, sg=None, su=None, sd=None):
    """y rows (fp64, unrounded) for the listed tokens.

    Wg/Wu/Wd (and sg/su/sd) are lists of E+S arrays; entries may be None for
    experts no listed token uses.
    """
    x = np.ascontiguousarray(x)
    T, H = x.shape
    idx = _c(idx, np.int32)
    gate = _c(gate, np.float32)
    k = idx.shape[1]
    tokens = _c(tokens, np.int32)
    if all(a is None for a in Wg):          # no listed token uses any expert (everything pruned, S = 0): empty sums
        return np.zeros((len(tokens), H), np.float64)
    first = next(a for a in Wg if a is not None)
    I = first.shape[0]
    wdt = w_dtype_of(first)
    keepalive = []

    def table(lst, dt=None):
        if lst is None:
            return None
        arr = (C.c_void_p * (E + S))()
        for i, a in enumerate(lst):
            if a is None:
                arr[i] = None
            else:
                a = np.ascontiguousarray(a) if dt is None else _c(a, dt)
                keepalive.append(a)
                arr[i] = a.ctypes.data
        return arr

    tg, tu, td = table(Wg), table(Wu), table(Wd)
    tsg, tsu, tsd = table(sg, np.float32), table(su, np.float32), table(sd, np.float32)
    y = np.empty((len(tokens), H), np.float64)
    rc = lib().oracle_moe_tokens(_p(x), act_dtype_of(x), _p(tokens), len(tokens), _p(idx), _p(gate), k, tg, tu,
                                 td, wdt, tsg, tsu, tsd, E, S, H, I, C.c_double(routed_scale), _p(y))
    assert rc == 0, f"oracle_moe_tokens rc={rc} (missing expert weights?)"
    return y


def fit(sizes, times):
    S = _c(sizes, np.float64)
    t = _c(times, np.float64)
    a, b, r2 = C.c_double(), C.c_double(), C.c_double()
    rc = lib().oracle_fit(_p(S), _p(t), len(S), C.byref(a), C.byref(b), C.byref(r2))
    assert rc == 0
    return a.value, b.value, r2.value


def e4m3_value(code):
    return float(lib().oracle_e4m3_value(int(code)))
