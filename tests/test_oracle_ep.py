"""Pins for the expert-parallel oracle (oracle/ep_oracle.py).
CPU only."""
import numpy as np
import pytest

from oracle import ep_oracle as ep


def tiny_layer(rng, T, H=16, I=8, E=8, S=1, k=2):
    x = rng.normal(size=(T, H)).astype(np.float32)
    W = lambda r, c: (0.3 * rng.normal(size=(r, c))).astype(np.float32)
    Wg, Wu, Wd = [W(I, H) for _ in range(E + S)], [W(I, H) for _ in range(E + S)], [W(H, I) for _ in range(E + S)]
    z = rng.normal(size=(T, E))
    s = (np.exp(z) / np.exp(z).sum(1, keepdims=True)).astype(np.float32)
    return x, Wg, Wu, Wd, s


@pytest.mark.parametrize("D", [1, 2, 4, 8])
def test_ep_layer_is_the_single_device_layer(orc, D):
    """EP over D devices computes exactly the single-device layer (the combine adds the same fp64 terms
    in the same order), for contiguous and for scattered partition tables, with pruned / empty slots."""
    rng = np.random.default_rng(40 + D)
    E, S, k = 8, 1, 3
    for trial in range(6):
        T = int(rng.integers(1, 9))
        x, Wg, Wu, Wd, s = tiny_layer(rng, T, E=E, S=S, k=k)
        idx, gate = orc.route(s, None, k)
        keep = (rng.random(E) < 0.6).astype(np.uint8)
        idx, gate = orc.compensate(s, None, keep, idx, gate)            # leaves -1 slots when < k experts survive
        part = (np.arange(E) // (E // D)).astype(np.int32) if trial % 2 == 0 else rng.integers(0, D, size=E).astype(np.int32)
        y_ep = ep.ep_layer(x, idx, gate, Wg, Wu, Wd, part, D, E, S, 2.5)
        y_1 = orc.moe_tokens(x, list(range(T)), idx, gate, Wg, Wu, Wd, E, S, 2.5)
        assert np.array_equal(y_ep, y_1)


def test_ep_plan_invariants(orc):
    rng = np.random.default_rng(7)
    E, k = 16, 4
    for trial in range(50):
        T, D = int(rng.integers(1, 20)), int(rng.choice([1, 2, 4, 8]))
        z = rng.normal(size=(T, E)).astype(np.float32)
        idx, gate = orc.route(z, None, k)
        idx[rng.random(idx.shape) < 0.15] = -1                           # pruned slots
        part = rng.integers(0, D, size=E).astype(np.int32)
        p = ep.ep_plan(idx, part, D)
        n = int((idx >= 0).sum())
        assert len(p["tok"]) == n == p["offs"][-1] and p["offs"][0] == 0
        valid = idx[idx >= 0]
        assert np.array_equal(p["counts"], np.bincount(part[valid], minlength=D))      # counts as a library call
        seen = set()
        for d in range(D):
            lo, hi = p["offs"][d], p["offs"][d + 1]
            seg = list(zip(p["expert"][lo:hi], p["tok"][lo:hi]))
            assert seg == sorted(seg)                                     # (expert, token) ascending inside a device (R38)
            assert all(part[e] == d for e, _ in seg)
        for i in range(n):                                                # a permutation of the valid entries
            t, j, e = p["tok"][i], p["slot"][i], p["expert"][i]
            assert idx[t, j] == e and (t, j) not in seen
            seen.add((t, j))
        # with contiguous partitions the send order is the single-device expert-major work list (S6) itself
        partc = (np.arange(E) // (E // D)).astype(np.int32)
        pc = ep.ep_plan(idx, partc, D)
        c = orc.compact(idx, gate, E)
        assert np.array_equal(pc["tok"], c["tok"]) and np.array_equal(pc["slot"], c["slot"])


def test_ep_latency_is_f_cost(orc):
    """Latency_total = max_d Latency_d is the F_cost of PAPER.md:127."""
    rng = np.random.default_rng(3)
    for _ in range(100):
        E, D = 12, int(rng.choice([1, 2, 3, 4]))
        part = rng.integers(0, D, size=E).astype(np.int32)
        w = rng.integers(0, 50, size=E).astype(np.int64)
        keep = (rng.random(E) < 0.5).astype(np.uint8)
        tot, load = ep.ep_latency(keep, w, part, D)
        F, l2 = orc.f_cost(keep, w, part, D)
        assert tot == F and np.array_equal(load, l2)
