"""CPU oracle for expert-parallel (EP) execution of one CAEE layer.

TEST INFRASTRUCTURE ONLY (see oracle/oracle.py).  Plain numpy / Python loops, fp64, in the order of
PAPER.md:57 (II-B: "token dispatch -> expert activation -> computation -> result aggregation ...
across devices"):

  ep_plan          which (token, slot) entry goes to which device, in which order
  ep_layer         the literal data flow over D devices: every device computes E_e(x_t) for the entries
                   it receives (experts of its own E_d only), the rows travel back to the token's home
                   device and are combined there in slot order
  ep_latency       Latency_total = max_d Latency_d with Latency_d = sum of R C~ over the
                   experts device d executes: the quantity F_cost models

Readings: R38 — a device receives its entries ordered by (expert, token) ascending, i.e.
each device's slice of the single-device expert-major work list (S6); R39 — shared experts are
replicated: a token's shared-expert rows are computed on its home device (R21: always run, gate 1);
R40 — the pruning decision of an EP step is taken on the GLOBAL batch (x_e is one bit per expert for
all devices' tokens, PAPER.md:111 "each Process_i", :127): every device all-gathers K_t and the gates
and takes the same integer decision.

Pins (tests/test_oracle_ep.py): ep_layer == the single-device oracle_moe_tokens bit for bit (the
combine adds the same fp64 terms in the same order), for any partition table and any token->home map;
ep_plan is a permutation of the valid entries whose per-device segments are sorted and hit only that
device's experts; counts = bincount of part[idx]; ep_latency == oracle_f_cost.
"""
import numpy as np

from . import oracle as orc


def ep_plan(idx, part, D):
    """Send order of the valid (token, slot) entries: ascending (device, expert, token).
    Returns dict(counts[D], offs[D+1], tok[n], slot[n], expert[n])."""
    idx = np.asarray(idx, np.int32)
    T, k = idx.shape
    ent = []
    for t in range(T):
        for j in range(k):
            e = int(idx[t, j])
            if e >= 0:
                ent.append((int(part[e]), e, t, j))
    ent.sort()
    counts = np.zeros(D, np.int32)
    for d, _, _, _ in ent:
        counts[d] += 1
    offs = np.zeros(D + 1, np.int32)
    offs[1:] = np.cumsum(counts)
    return dict(counts=counts, offs=offs, tok=np.array([e[2] for e in ent], np.int32),
                slot=np.array([e[3] for e in ent], np.int32), expert=np.array([e[1] for e in ent], np.int32))


def ep_layer(x, idx, gate, Wg, Wu, Wd, part, D, E, S, routed_scale, sg=None, su=None, sd=None):
    """y [T,H] fp64 computed the EP way.  Wg/Wu/Wd (sg/su/sd): lists of E+S arrays as in oracle.moe_tokens."""
    x = np.ascontiguousarray(x)
    T, H = x.shape
    k = idx.shape[1]
    plan = ep_plan(idx, part, D)

    def ffn(t, e):
        return orc.expert_ffn(x[t], Wg[e], Wu[e], Wd[e], None if sg is None else sg[e], None if su is None else su[e],
                              None if sd is None else sd[e])

    # dispatch + computation: device d works through its received entries in order
    back = np.zeros((T, k, H), np.float64)           # rows as they arrive back at the home device
    for d in range(D):
        for i in range(plan["offs"][d], plan["offs"][d + 1]):
            t, j, e = int(plan["tok"][i]), int(plan["slot"][i]), int(plan["expert"][i])
            assert part[e] == d
            back[t, j] = ffn(t, e)
    # aggregation at the home device, slot order, then the replicated shared experts (R39)
    y = np.zeros((T, H), np.float64)
    for t in range(T):
        for j in range(k):
            if idx[t, j] >= 0:
                y[t] += float(gate[t, j]) * back[t, j]
        y[t] *= routed_scale
        for s in range(S):
            y[t] += ffn(t, E + s)
    return y


def ep_latency(keep, w, part, D):
    """(Latency_total, per-device Latency_d): PAPER.md:97 max over devices of PAPER.md:127's sums."""
    load = np.zeros(D, np.int64)
    for e in range(len(keep)):
        if keep[e]:
            load[part[e]] += int(w[e])
    return int(load.max()) if D else 0, load
