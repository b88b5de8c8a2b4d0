"""Pins for oracle O3 (cost, F_cost), O4 (prune), O5 (compensate), O6 (compact), O9 (fit):
closed forms the paper / BASELINE.json fix, brute force over all expert subsets on tiny
instances, special-case reductions and the hand-worked fixture.  CPU only."""
import itertools

import numpy as np
import pytest
import torch

from tests.golden_io import read_golden

MODE_NONE, MODE_THRESH, MODE_CIR, MODE_RANK, MODE_FRAC = 0, 1, 2, 3, 4
FIX = 2.0 ** 40


def tiny_instance(rng, E=8, D=2, T=None, k=2, uniform_cost=True, residency=False, softmax=True):
    T = T or int(rng.integers(1, 7))
    z = rng.normal(size=(T, E)) * 1.5
    if softmax:
        p = np.exp(z - z.max(1, keepdims=True))
        s = (p / p.sum(1, keepdims=True)).astype(np.float32)
    else:
        s = (1 / (1 + np.exp(-z))).astype(np.float32)
    part = (np.arange(E) // (E // D)).astype(np.int32)
    if uniform_cost:
        per_part = rng.integers(1, 20, size=D)
        w = per_part[part].astype(np.int64)
    else:
        w = rng.integers(1, 20, size=E).astype(np.int64)
    if residency:
        w = np.where(rng.random(E) < 0.4, 0, w).astype(np.int64)   # cache hits cost nothing
    return s, part, w, T


def F_literal(mask, w, part, D):
    """PAPER.md:127 written as a library call: max over d of bincount-weighted sums."""
    return int(np.bincount(part, weights=np.asarray(mask, np.float64) * w, minlength=D).max())


# ---------------------------------------------------------------- O3 / O9 closed forms
def test_paper_and_config_constants(orc):
    g = read_golden("paper_constants.txt")
    a, b, c = (int(v) for v in g["expert_weight_shape"])
    assert a * b * c == 44_040_192 and round(a * b * c / 2 ** 20) == 42      # the paper rounds to "43 MB"
    assert abs(a * b * c / 1e6 - g["expert_size_MB_W8"][0]) < 1.1
    assert int(g["moe_layers"][0] * g["experts_per_layer"][0]) == int(g["experts_total"][0])
    for base, new, gain in (("table2_bs8_tpot_base", "table2_bs8_tpot_08", "table2_bs8_gain_pct"),
                            ("table2_bs1_tpot_base", "table2_bs1_tpot_09", "table2_bs1_gain_pct")):
        assert abs((g[base][0] - g[new][0]) / g[base][0] * 100 - g[gain][0]) < 0.01
    # C~ = S_e / B_d + overhead at config 1's numbers: 1,572,864 B / 1 TB/s + 2 us
    assert orc.cost_ticks(1e-3, 2000.0, int(g["c1_expert_bytes"][0])) == int(g["c1_cost_ticks_ns"][0]) == 3573
    # R1-shaped bf16 expert at a nominal 8 TB/s: 88,080,384 B -> 11.010 us (+ 2 us)
    assert orc.cost_ticks(1 / 8000.0, 0.0, 88_080_384) == 11010
    assert orc.cost_ticks(1 / 8000.0, 2000.0, 88_080_384) == 13010
    from paper_2606_29982_b200 import workloads as wl
    assert wl.C1.expert_bytes == 1_572_864 and wl.C3.expert_bytes == 88_080_384
    assert wl.C4.expert_bytes == 44_040_192 + 3 * 56 * 16 * 4
    for cfg, bw in ((wl.C1, 1000.0), (wl.C2, 8000.0), (wl.C3, 8000.0), (wl.C4, 8000.0)):
        assert orc.cost_ticks(1 / bw, 2000.0, cfg.expert_bytes) == cfg.cost_ticks_ns


def test_fit_recovers_a_line_and_matches_polyfit(orc):
    S = np.array([1e6, 4e6, 16e6, 64e6, 88e6])
    a, b, r2 = orc.fit(S, 0.000125 * S + 2000.0)
    assert abs(a - 0.000125) < 1e-12 and abs(b - 2000.0) < 1e-6 and abs(r2 - 1) < 1e-12
    rng = np.random.default_rng(0)
    t = 0.018 * S + 9000 + rng.normal(scale=500, size=S.size)
    a, b, r2 = orc.fit(S, t)
    pa, pb = np.polyfit(S, t, 1)
    assert abs(a - pa) < 1e-9 * abs(pa) + 1e-15 and abs(b - pb) < 1e-6 * abs(pb)
    assert 0.99 < r2 <= 1.0


def test_effective_cost_two_tier(orc):
    res = np.array([1, 0, 1, 0], np.uint8)
    w = orc.effective_cost(res, np.array([5, 5, 0, 0]), np.array([90, 91, 92, 93]))
    assert list(w) == [5, 91, 0, 93]       # R(e,d) gates which tier applies


def test_f_cost_is_max_over_partitions_of_sums(orc):
    rng = np.random.default_rng(1)
    for _ in range(200):
        E, D = 12, int(rng.choice([1, 2, 3, 4, 6]))
        part = rng.integers(0, D, size=E).astype(np.int32)
        w = rng.integers(0, 50, size=E).astype(np.int64)
        mask = (rng.random(E) < 0.5).astype(np.uint8)
        F, load = orc.f_cost(mask, w, part, D)
        assert F == F_literal(mask, w, part, D) == load.max()
        assert load.sum() == int((mask * w).sum())
    # D = 1 is a plain sum; one expert per partition is a plain max (PAPER.md:97 straggler law)
    w = np.array([3, 9, 4, 7], np.int64)
    assert orc.f_cost(np.ones(4, np.uint8), w, np.zeros(4, np.int32), 1)[0] == 23
    assert orc.f_cost(np.ones(4, np.uint8), w, np.arange(4, dtype=np.int32), 4)[0] == 9


# ---------------------------------------------------------------- O4
def test_prune_hand_example(orc):
    g = read_golden("prune_hand_example.txt")
    E, D, k = int(g["E"][0]), int(g["D"][0]), int(g["k"][0])
    idx = np.array(g["idx"], np.int32).reshape(-1, k)
    gate = np.array(g["gate"], np.float32).reshape(-1, k)
    r = orc.prune(MODE_THRESH, g["theta"][0], 0, idx, gate, E, np.array(g["w"], np.int64), np.array(g["part"], np.int32), D)
    assert list(r["must"]) == [int(v) for v in g["must"]]
    assert list(r["keep"]) == [int(v) for v in g["keep"]]
    assert (r["F_base"], r["F_cost_dense"], r["F_cost"]) == (int(g["F_base"][0]), int(g["F_cost_dense"][0]), int(g["F_cost"][0]))
    assert abs(r["F_imp_fix"] / FIX - g["F_imp"][0]) < 1e-6
    # compensation for t1
    s = np.zeros((3, E), np.float32)
    for t in range(3):
        s[t, idx[t]] = gate[t]          # any full vector consistent with the top-2; t1 gets the stated one
    s[1] = np.array(g["s_t1"], np.float32)
    idx2, gate2 = orc.compensate(s, None, r["keep"], idx, gate)
    assert list(idx2[1]) == [int(v) for v in g["kfinal_t1"]]
    np.testing.assert_allclose(gate2[1], g["gate_t1"], rtol=1e-6)
    assert np.array_equal(idx2[[0, 2]], idx[[0, 2]]) and np.array_equal(gate2[[0, 2]], gate[[0, 2]])


def _must_reference(mode, theta, idx, gate, E):
    """A_must by mode, recomputed independently in float64 / numpy set operations."""
    T, k = idx.shape
    I = np.zeros(E)
    np.add.at(I, idx.ravel(), gate.ravel().astype(np.float64))
    act = np.isin(np.arange(E), idx)
    if mode == MODE_THRESH:
        return act & (I >= theta)
    # per-token rules see K_t sorted by gate (R36): an independent numpy sort
    order = np.stack([np.lexsort((idx[t], -gate[t].astype(np.float64))) for t in range(T)])
    idx_s, gate_s = np.take_along_axis(idx, order, 1), np.take_along_axis(gate, order, 1).astype(np.float64)
    if mode == MODE_RANK:
        return np.isin(np.arange(E), idx_s[:, :k - int(theta)])
    if mode == MODE_CIR:
        cir = np.cumsum(gate_s, 1) / gate_s.sum(1, keepdims=True)
        m = (cir >= theta).argmax(1) + 1
        keep = [idx_s[t, :m[t]] for t in range(T)]
        return np.isin(np.arange(E), np.concatenate(keep))
    if mode == MODE_FRAC:
        ids = np.flatnonzero(act)
        order = ids[np.lexsort((ids, I[ids]))]
        n_c = int(np.floor(theta * len(ids)))
        must = act.copy()
        must[order[:n_c]] = False
        return must
    return act


@pytest.mark.parametrize("mode,thetas", [(MODE_THRESH, [0.13, 0.37, 0.61, 0.93, 1.7]), (MODE_CIR, [0.97, 0.83, 0.71, 0.52]),
                                         (MODE_RANK, [0, 1, 2]), (MODE_FRAC, [0.0, 0.1, 0.25, 0.5, 1.0])])
@pytest.mark.parametrize("uniform_cost,residency", [(True, False), (True, True), (False, True)])
def test_prune_bruteforce_over_all_subsets(orc, mode, thetas, uniform_cost, residency):
    rng = np.random.default_rng(100 + mode * 7 + uniform_cost * 3 + residency)
    E, D, k = 8, 2, 2
    for trial in range(60):
        s, part, w, T = tiny_instance(rng, E, D, k=k, uniform_cost=uniform_cost, residency=residency)
        idx, gate = orc.route(s, None, k)
        prev_Fbase = None
        for theta in thetas:
            r = orc.prune(mode, theta, 0, idx, gate, E, w, part, D)
            act, must, keep = r["act"].astype(bool), r["must"].astype(bool), r["keep"].astype(bool)
            I = r["I_fix"]
            # step 1 against an independent float64 recomputation (thetas sit away from ties)
            ref_must = _must_reference(mode, theta, idx, gate, E)
            margin_ok = True
            if mode == MODE_THRESH:
                margin_ok = np.all(np.abs(I[act] / FIX - theta) > 1e-5)
            if mode == MODE_CIR:
                gs = -np.sort(-gate.astype(np.float64), 1)
                cir = np.cumsum(gs, 1) / gs.sum(1, keepdims=True)
                margin_ok = np.all(np.abs(cir - theta) > 1e-5)
            if mode == MODE_FRAC:
                margin_ok = len(set(I[act].tolist())) == act.sum()
            if margin_ok:
                assert np.array_equal(must, ref_must), (mode, theta)
            # A_must subset A_trans subset A_act
            assert not (must & ~keep).any() and not (keep & ~act).any()
            # F_cost(A_trans) = F_base exactly, both as literal max-of-sums
            assert r["F_base"] == F_literal(must, w, part, D)
            assert r["F_cost"] == F_literal(keep, w, part, D) == r["F_base"]
            assert r["F_cost_dense"] == F_literal(act, w, part, D)
            assert r["F_imp_fix"] == int(I[act & ~keep].sum())
            # brute force over every A with A_must <= A <= A_act
            cand = np.flatnonzero(act & ~must)
            best_imp, feasible_sets = -1, []
            for bits_ in itertools.product([0, 1], repeat=len(cand)):
                A = must.copy()
                A[cand[np.array(bits_, bool)]] = True
                F = F_literal(A, w, part, D)
                assert F >= r["F_base"]                     # F_base is the minimum of the objective
                if F == r["F_base"]:
                    feasible_sets.append(A)
                    best_imp = max(best_imp, int(I[A].sum()))
            assert any(np.array_equal(A, keep) for A in feasible_sets)
            # inclusion-maximal: no pruned candidate fits at F_base
            for e in np.flatnonzero(act & ~keep):
                A = keep.copy()
                A[e] = True
                assert F_literal(A, w, part, D) > r["F_base"]
            # zero-cost (cache-hit) candidates are never pruned
            assert keep[act & (w == 0)].all()
            # with per-partition uniform non-zero costs the greedy also retains the most importance
            if uniform_cost:
                assert int(I[keep].sum()) == best_imp
            # monotone in the knob
            if mode in (MODE_THRESH, MODE_RANK, MODE_FRAC) and prev_Fbase is not None:
                assert r["F_base"] <= prev_Fbase
            if mode == MODE_CIR and prev_Fbase is not None:
                assert r["F_base"] <= prev_Fbase             # thetas listed in decreasing theta_imp
            prev_Fbase = r["F_base"]


@pytest.mark.parametrize("mode,theta", [(MODE_NONE, 0.0), (MODE_THRESH, 0.0), (MODE_CIR, 1.0), (MODE_RANK, 0), (MODE_FRAC, 0.0)])
def test_zero_budget_keeps_everything(orc, mode, theta):
    rng = np.random.default_rng(5)
    for _ in range(30):
        s, part, w, T = tiny_instance(rng, 16, 4, k=3)
        idx, gate = orc.route(s, None, 3)
        r = orc.prune(mode, theta, 0, idx, gate, 16, w, part, 4)
        assert np.array_equal(r["keep"], r["act"]) and r["F_imp_fix"] == 0 and r["F_cost"] == r["F_cost_dense"]
        idx2, gate2 = orc.compensate(s, None, r["keep"], idx, gate)
        assert np.array_equal(idx2, idx) and np.array_equal(gate2, gate)


def test_single_partition_keeps_must_plus_free(orc):
    rng = np.random.default_rng(6)
    for _ in range(50):
        s, part, w, T = tiny_instance(rng, 8, 1, k=2, uniform_cost=False, residency=True)
        idx, gate = orc.route(s, None, 2)
        r = orc.prune(MODE_THRESH, 0.4, 0, idx, gate, 8, w, part, 1)
        expect = r["must"].astype(bool) | (r["act"].astype(bool) & (w == 0))
        assert np.array_equal(r["keep"].astype(bool), expect)


def test_straggler_partition_only_shrinks(orc):
    """Doubling one partition's costs can only shrink that partition's kept set (SURVEY §8(c) vii)."""
    rng = np.random.default_rng(7)
    for _ in range(200):
        s, part, w, T = tiny_instance(rng, 8, 2, k=2)
        idx, gate = orc.route(s, None, 2)
        theta = float(rng.choice([0.2, 0.4, 0.6]))
        r1 = orc.prune(MODE_THRESH, theta, 0, idx, gate, 8, w, part, 2)
        w2 = np.where(part == 1, 2 * w, w)
        r2 = orc.prune(MODE_THRESH, theta, 0, idx, gate, 8, w2, part, 2)
        k1, k2 = r1["keep"].astype(bool), r2["keep"].astype(bool)
        assert not (k2 & ~k1 & (part == 1)).any()


def test_keep_top1_flag(orc):
    rng = np.random.default_rng(8)
    s, part, w, T = tiny_instance(rng, 8, 2, T=1, k=2)
    idx, gate = orc.route(s, None, 2)
    r = orc.prune(MODE_THRESH, 5.0, 0, idx, gate, 8, w, part, 2)
    assert r["n_must"] == 0 and r["n_keep"] == int((w[idx[0]] == 0).sum())       # faithful: may empty A_must (reading R23)
    r = orc.prune(MODE_THRESH, 5.0, 2, idx, gate, 8, w, part, 2)
    assert r["must"][idx[0, 0]] == 1


def _golden_case(name):
    g = read_golden(name)
    E, D, k = int(g["E"][0]), int(g["D"][0]), int(g["k"][0])
    idx = np.array(g["idx"], np.int32).reshape(-1, k)
    gate = np.array(g["gate"], np.float32).reshape(-1, k)
    return g, E, D, idx, gate, np.array(g["w"], np.int64), np.array(g["part"], np.int32)


def _check_golden(r, g, keep_key="keep"):
    assert list(r["must"]) == [int(v) for v in g["must"]]
    assert list(r["keep"]) == [int(v) for v in g[keep_key]]


def test_cir_boundary_and_gate_order_hand_example(orc):
    """R9 (the boundary is '>=') and R36 (K_t sorted by gate, equal gates -> lower id)."""
    g, E, D, idx, gate, w, part = _golden_case("cir_boundary_example.txt")
    r = orc.prune(MODE_CIR, g["theta_imp"][0], 0, idx, gate, E, w, part, D)
    _check_golden(r, g)
    assert (r["F_base"], r["F_cost_dense"], r["F_cost"]) == (int(g["F_base"][0]), int(g["F_cost_dense"][0]), int(g["F_cost"][0]))
    assert r["F_imp_fix"] == int(g["F_imp"][0] * FIX)
    r = orc.prune(MODE_RANK, g["rank_budget"][0], 0, idx, gate, E, w, part, D)
    assert list(r["must"]) == [int(v) for v in g["must"]]
    r = orc.prune(MODE_THRESH, 5.0, 2, idx, gate, E, w, part, D)
    assert list(r["must"]) == [int(v) for v in g["top1_must"]]


def test_equal_importance_tie_hand_example(orc):
    """R7 / R22: equal I(e) -> the lower expert id is visited (and promoted) first."""
    g, E, D, idx, gate, w, part = _golden_case("prune_tie_example.txt")
    r = orc.prune(MODE_THRESH, g["theta"][0], 0, idx, gate, E, w, part, D)
    assert r["I_fix"][1] == r["I_fix"][2]
    _check_golden(r, g)
    assert (r["F_base"], r["F_cost_dense"], r["F_cost"]) == (int(g["F_base"][0]), int(g["F_cost_dense"][0]), int(g["F_cost"][0]))
    assert r["F_imp_fix"] == int(g["F_imp"][0] * FIX)


def test_per_token_rules_use_gate_order_not_list_order(orc):
    """With a selection bias the route lists K_t by s' = s + corr_bias; CIR / RANK / KEEP_TOP1 must
    still see it sorted by the gate (R36).  The reference sorts independently with numpy."""
    rng = np.random.default_rng(77)
    E, D, k = 16, 4, 4
    differs = 0
    for trial in range(120):
        s, part, w, T = tiny_instance(rng, E, D, T=int(rng.integers(1, 9)), k=k, softmax=False)
        cb = rng.normal(scale=0.3, size=E).astype(np.float32)
        idx, gate = orc.route(s, cb, k)
        differs += int((np.diff(gate, axis=1) > 0).any())
        for mode, theta in ((MODE_CIR, 0.83), (MODE_CIR, 0.61), (MODE_RANK, 1), (MODE_RANK, 3)):
            if mode == MODE_CIR:
                gs = -np.sort(-gate.astype(np.float64), 1)
                if not np.all(np.abs(np.cumsum(gs, 1) / gs.sum(1, keepdims=True) - theta) > 1e-5):
                    continue
            r = orc.prune(mode, theta, 0, idx, gate, E, w, part, D)
            assert np.array_equal(r["must"].astype(bool), _must_reference(mode, theta, idx, gate, E)), (trial, mode, theta)
        r = orc.prune(MODE_THRESH, 100.0, 2, idx, gate, E, w, part, D)
        top = idx[np.arange(T), np.argmax(gate, 1)]          # np.argmax: first maximum
        assert np.array_equal(r["must"].astype(bool), np.isin(np.arange(E), top))
    assert differs > 60          # the instances really do have non-descending gate lists


# ---------------------------------------------------------------- importance bound (R37)
def test_importance_bound_hand_example(orc):
    g, E, D, idx, gate, w, part = _golden_case("imp_bound_example.txt")
    r0 = orc.prune(MODE_THRESH, g["theta"][0], 0, idx, gate, E, w, part, D)
    _check_golden(r0, g, "keep_unbounded")
    assert r0["F_imp_fix"] == int(g["F_imp_unbounded"][0] * FIX)
    for eps in (g["eps"][0], g["eps_boundary"][0]):
        r = orc.prune(MODE_THRESH, g["theta"][0], 8, idx, gate, E, w, part, D, eps=eps)
        _check_golden(r, g)
        assert (r["F_base"], r["F_cost"]) == (int(g["F_base"][0]), int(g["F_cost"][0]))
        assert r["F_imp_fix"] == int(g["F_imp"][0] * FIX)
    r = orc.prune(MODE_THRESH, g["theta"][0], 8, idx, gate, E, w, part, D, eps=0.0)
    assert np.array_equal(r["keep"], r["act"]) and r["F_imp_fix"] == 0 and r["F_cost"] == r["F_cost_dense"]


@pytest.mark.parametrize("mode,theta", [(MODE_THRESH, 0.9), (MODE_CIR, 0.6), (MODE_FRAC, 0.7), (MODE_RANK, 1)])
def test_importance_bound_bruteforce(orc, mode, theta):
    """F_imp <= eps holds; the bound only ever restores (A_trans grows); the restored
    set R is the smallest set of pruned experts whose return meets the bound (brute force over all
    subsets of the unbounded pruned set), hence the pruned set is inclusion-maximal under the bound;
    a bound that already holds changes nothing."""
    rng = np.random.default_rng(300 + mode)
    E, D, k = 8, 2, 2
    hit = 0
    for trial in range(80):
        s, part, w, T = tiny_instance(rng, E, D, T=int(rng.integers(2, 9)), k=k)
        idx, gate = orc.route(s, None, k)
        r0 = orc.prune(mode, theta, 0, idx, gate, E, w, part, D)
        I = r0["I_fix"]
        pruned0 = np.flatnonzero(r0["act"].astype(bool) & ~r0["keep"].astype(bool))
        for eps in (0.0, 0.05, 0.3, 0.8, 100.0):
            r = orc.prune(mode, theta, 8, idx, gate, E, w, part, D, eps=eps)
            eps_fix = int(np.floor(eps * FIX))
            assert r["F_imp_fix"] <= eps_fix
            keep0, keep1 = r0["keep"].astype(bool), r["keep"].astype(bool)
            assert not (keep0 & ~keep1).any() and np.array_equal(r["must"], r0["must"]) and r["F_base"] == r0["F_base"]
            assert r["F_cost"] == F_literal(keep1, w, part, D) >= r["F_base"]
            assert r["F_imp_fix"] == int(I[r["act"].astype(bool) & ~keep1].sum())
            restored = np.flatnonzero(keep1 & ~keep0)
            if r0["F_imp_fix"] <= eps_fix:
                assert len(restored) == 0
                continue
            hit += 1
            best = None
            for bits_ in itertools.product([0, 1], repeat=len(pruned0)):
                sel = pruned0[np.array(bits_, bool)]
                if int(I[pruned0].sum() - I[sel].sum()) <= eps_fix and (best is None or len(sel) < best):
                    best = len(sel)
            assert len(restored) == best
            # greedy by importance: every restored expert is at least as important as every expert left pruned
            left = np.setdiff1d(pruned0, restored)
            if len(left) and len(restored):
                assert I[restored].min() >= I[left].max()
            for e in restored:             # dropping any restored expert breaks the bound
                assert r["F_imp_fix"] + int(I[e]) > eps_fix
    assert hit > 40


# ---------------------------------------------------------------- O5
@pytest.mark.parametrize("grouped", [False, True])
def test_compensation_invariants_and_masked_topk(orc, grouped):
    rng = np.random.default_rng(9 + grouped)
    E, D, k = 16, 4, 3
    for trial in range(80):
        s, part, w, T = tiny_instance(rng, E, D, T=int(rng.integers(1, 12)), k=k, softmax=not grouped)
        cb = rng.normal(scale=0.05, size=E).astype(np.float32) if grouped else None
        ng, tg = (4, 2) if grouped else (1, 1)
        idx, gate = orc.route(s, cb, k, n_group=ng, topk_group=tg)
        r = orc.prune(MODE_THRESH, float(rng.choice([0.2, 0.5, 0.9])), 0, idx, gate, E, w, part, D)
        keep = r["keep"].astype(bool)
        idx2, gate2 = orc.compensate(s, cb, keep, idx, gate)
        sp = torch.from_numpy(s) + (torch.from_numpy(cb) if cb is not None else 0)
        n_keep = int(keep.sum())
        for t in range(T):
            affected = (~keep[idx[t]]).any()
            if not affected:                      # untouched, bit for bit (reading R14)
                assert np.array_equal(idx2[t], idx[t]) and np.array_equal(gate2[t], gate[t])
                continue
            sel = idx2[t][idx2[t] >= 0]
            assert keep[sel].all()                                   # K_final subset of A_trans
            assert len(sel) == min(k, n_keep)                        # output stays dense
            masked = sp[t].clone()
            masked[torch.from_numpy(~keep)] = -float("inf")          # Top-k(G_masked) as a library call
            ref = torch.topk(masked, min(k, n_keep)).indices.numpy()
            assert np.array_equal(sel, ref)
            if len(sel):
                np.testing.assert_allclose(gate2[t][:len(sel)], s[t][sel] / s[t][sel].astype(np.float64).sum(), rtol=1e-6)
                assert abs(gate2[t].sum() - 1) < 1e-5                # redistributed, still sums to 1
            assert (gate2[t][len(sel):] == 0).all() and (idx2[t][len(sel):] == -1).all()
        # literal reading (every token re-selected) coincides for ungrouped routers when |A_trans| >= k
        if not grouped and n_keep >= k:
            idx3, gate3 = orc.compensate(s, cb, keep, idx, gate, flags=1)
            assert np.array_equal(idx3, idx2)
            np.testing.assert_allclose(gate3, gate2, rtol=1e-6)


def test_compensation_with_empty_transferable_set(orc):
    s = np.array([[0.5, 0.3, 0.2, 0.0]], np.float32)
    idx, gate = orc.route(s, None, 2)
    idx2, gate2 = orc.compensate(s, None, np.zeros(4, np.uint8), idx, gate)
    assert (idx2 == -1).all() and (gate2 == 0).all()                 # reading R15: no division by zero


# ---------------------------------------------------------------- O6
def test_compact_inverts_idx(orc):
    rng = np.random.default_rng(11)
    for _ in range(30):
        T, E, k = int(rng.integers(1, 40)), 16, 3
        s, part, w, _ = tiny_instance(rng, E, 4, T=T, k=k)
        idx, gate = orc.route(s, None, k)
        keep = (rng.random(E) < 0.6).astype(np.uint8)
        idx, gate = orc.compensate(s, None, keep, idx, gate)
        c = orc.compact(idx, gate, E)
        assert c["offs"][0] == 0 and c["offs"][-1] == int((idx >= 0).sum()) == len(c["tok"])
        assert list(c["expert_ids"]) == sorted(set(idx[idx >= 0].tolist()))
        rebuilt = np.full_like(idx, -1)
        for r, e in enumerate(c["expert_ids"]):
            lo, hi = c["offs"][r], c["offs"][r + 1]
            assert hi > lo and list(c["tok"][lo:hi]) == sorted(c["tok"][lo:hi])
            for i in range(lo, hi):
                rebuilt[c["tok"][i], c["slot"][i]] = e
                assert c["wt"][i] == gate[c["tok"][i], c["slot"][i]]
        assert np.array_equal(rebuilt, idx)
