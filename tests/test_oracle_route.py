"""Pins for oracle O0 (scores), O1 (route), O2 (importance): library routines,
brute force, invariants and the hand-worked fixture.  CPU only."""
import itertools
import os

import numpy as np
import pytest
import torch

from tests.golden_io import read_golden

HERE = os.path.dirname(os.path.abspath(__file__))


def _rand_scores(rng, T, E, kind="sigmoid"):
    z = rng.normal(size=(T, E)).astype(np.float64)
    if kind == "sigmoid":
        return (1 / (1 + np.exp(-z))).astype(np.float32)
    e = np.exp(z - z.max(1, keepdims=True))
    return (e / e.sum(1, keepdims=True)).astype(np.float32)


# ---------------------------------------------------------------- O0
@pytest.mark.parametrize("score_fn", [0, 1])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_scores_vs_torch_fp64(orc, score_fn, dtype):
    g = torch.Generator().manual_seed(5)
    T, H, E = 7, 96, 24
    x = torch.randn(T, H, generator=g)
    Wr = 0.1 * torch.randn(E, H, generator=g)
    b = 0.3 * torch.randn(E, generator=g)
    if dtype == "bf16":
        xb = x.to(torch.bfloat16)
        x_in = xb.view(torch.int16).numpy().view(np.uint16)
        x64 = xb.double()
    else:
        x_in = x.numpy()
        x64 = x.double()
    logits = x64 @ Wr.double().T + b.double()
    ref = torch.sigmoid(logits) if score_fn == 1 else torch.softmax(logits, dim=1)
    s = orc.scores(x_in, Wr.numpy(), b.numpy(), score_fn)
    np.testing.assert_allclose(s, ref.numpy(), rtol=2e-7, atol=1e-30)
    if score_fn == 0:
        np.testing.assert_allclose(s.sum(1), 1.0, rtol=1e-6)
    # no bias pointer == zero bias
    s0 = orc.scores(x_in, Wr.numpy(), None, score_fn)
    s1 = orc.scores(x_in, Wr.numpy(), np.zeros(E, np.float32), score_fn)
    assert np.array_equal(s0, s1)


# ---------------------------------------------------------------- O1
def test_route_plain_topk_matches_torch(orc):
    rng = np.random.default_rng(0)
    s = _rand_scores(rng, 50, 64, "softmax")
    idx, gate = orc.route(s, None, 6)
    tv, ti = torch.topk(torch.from_numpy(s), 6, dim=1)  # library routine, sorted descending
    assert np.array_equal(idx, ti.numpy().astype(np.int32))
    ref = tv.double() / tv.double().sum(1, keepdim=True)
    np.testing.assert_allclose(gate, ref.numpy(), rtol=1e-6)
    np.testing.assert_allclose(gate.sum(1), 1.0, rtol=1e-6)


def test_route_all_groups_allowed_reduces_to_plain_topk(orc):
    rng = np.random.default_rng(1)
    s = _rand_scores(rng, 40, 32)
    cb = rng.normal(scale=0.05, size=32).astype(np.float32)
    a = orc.route(s, cb, 4, n_group=1, topk_group=1)
    b = orc.route(s, cb, 4, n_group=8, topk_group=8)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    _, ti = torch.topk(torch.from_numpy(s) + torch.from_numpy(cb), 4, dim=1)
    assert np.array_equal(a[0], ti.numpy().astype(np.int32))


def test_route_monotone_activation_gives_topk_of_logits(orc):
    rng = np.random.default_rng(2)
    z = rng.normal(size=(30, 16))
    s = (1 / (1 + np.exp(-z))).astype(np.float32)
    idx, _ = orc.route(s, None, 3)
    _, ti = torch.topk(torch.from_numpy(z), 3, dim=1)
    assert np.array_equal(idx, ti.numpy().astype(np.int32))


def test_route_group_limited_bruteforce(orc):
    """Best groups = argmax over group subsets of the summed group score; best experts =
    argmax over k-subsets inside them of the summed s' (no ties with random floats)."""
    rng = np.random.default_rng(3)
    E, ng, tg, k = 8, 4, 2, 3
    gs = E // ng
    for trial in range(200):
        s = _rand_scores(rng, 1, E)
        cb = rng.normal(scale=0.2, size=E).astype(np.float32)
        sp = (s[0] + cb).astype(np.float32)
        gscore = [np.sort(sp[g * gs:(g + 1) * gs])[-2:].astype(np.float64).sum() for g in range(ng)]
        best_groups = max(itertools.combinations(range(ng), tg), key=lambda c: sum(gscore[g] for g in c))
        allowed = [e for g in best_groups for e in range(g * gs, (g + 1) * gs)]
        best = max(itertools.combinations(allowed, k), key=lambda c: sum(float(sp[e]) for e in c))
        idx, gate = orc.route(s, cb, k, n_group=ng, topk_group=tg)
        assert set(idx[0]) == set(best)
        assert list(sp[idx[0]]) == sorted(sp[idx[0]], reverse=True)        # listed in descending s'
        assert len({e // gs for e in idx[0]}) <= tg
        # the gate uses the unbiased s, not s' (reading R1)
        np.testing.assert_allclose(gate[0], s[0][idx[0]] / s[0][idx[0]].astype(np.float64).sum(), rtol=1e-6)


def test_route_large_bias_changes_selection_not_gate_formula(orc):
    rng = np.random.default_rng(4)
    s = _rand_scores(rng, 5, 16)
    cb = np.zeros(16, np.float32)
    cb[11] = 10.0
    idx, gate = orc.route(s, cb, 2)
    assert (idx[:, 0] == 11).all()
    np.testing.assert_allclose(gate, np.take_along_axis(s, idx, 1) / np.take_along_axis(s, idx, 1).sum(1, keepdims=True), rtol=1e-6)


def test_route_ties_go_to_lower_index(orc):
    s = np.full((1, 8), 0.25, np.float32)
    idx, gate = orc.route(s, None, 3)
    assert list(idx[0]) == [0, 1, 2]
    s[0, 5] = 0.5
    idx, _ = orc.route(s, None, 3)
    assert list(idx[0]) == [5, 0, 1]
    # group ties -> lower group id
    idx, _ = orc.route(np.full((1, 8), 0.25, np.float32), None, 2, n_group=4, topk_group=1)
    assert list(idx[0]) == [0, 1]


def test_route_no_norm_gives_raw_scores(orc):
    rng = np.random.default_rng(6)
    s = _rand_scores(rng, 4, 16)
    idx, gate = orc.route(s, None, 4, norm_topk=False)
    assert np.array_equal(gate, np.take_along_axis(s, idx, 1))


def test_route_hand_example(orc):
    g = read_golden("route_hand_example.txt")
    s = np.array([g["s"]], np.float32)
    idx, gate = orc.route(s, None, int(g["k"][0]), n_group=int(g["n_group"][0]), topk_group=int(g["topk_group"][0]))
    assert list(idx[0]) == [int(v) for v in g["idx"]]
    np.testing.assert_allclose(gate[0], g["gate"], rtol=2e-6)
    plain, _ = orc.route(s, None, 3)
    assert list(plain[0]) == [int(v) for v in g["idx_plain_top3"]]


# ---------------------------------------------------------------- O2
def test_importance_sums_to_T_and_is_order_independent(orc):
    rng = np.random.default_rng(7)
    T, E, k = 64, 32, 4
    s = _rand_scores(rng, T, E, "softmax")
    idx, gate = orc.route(s, None, k)
    act, I = orc.importance(idx, gate, E)
    # sum_e I(e) = sum_t sum_j G = T, up to the fp32 rounding of each gate
    # (<= 2^-25, i.e. 2^15 fixed-point units) and the floor (< 1 unit)
    assert abs(int(I.sum()) - T * 2 ** 40) <= T * k * 2 ** 16
    perm = rng.permutation(T)
    act2, I2 = orc.importance(idx[perm], gate[perm], E)
    assert np.array_equal(I, I2) and np.array_equal(act, act2)
    ref = np.zeros(E)
    np.add.at(ref, idx.ravel(), gate.ravel().astype(np.float64))
    np.testing.assert_allclose(I / 2.0 ** 40, ref, atol=1e-9)
    assert np.array_equal(act.astype(bool), np.isin(np.arange(E), idx))
