"""Pins for the random-selection compensation baseline (FLAG_COMP_RANDOM; Fig. 9;
reading R35): the counter-based generator against murmur3's published finalizer values, the
uniformity of its draws, and the invariants / distribution of the re-selection."""
import numpy as np

from oracle import oracle as orc


def test_fmix32_is_murmur3s_finalizer():
    f = orc.lib().oracle_fmix32
    assert f(0) == 0
    assert f(1) == 0x514E28B7          # MurmurHash3 fmix32(1), the published avalanche test value
    assert len({f(i) for i in range(1 << 16)}) == 1 << 16      # a bijection: no collisions


def test_unit_draws_are_uniform():
    u = np.array([[orc.lib().oracle_unit_draw(t, e) for e in range(64)] for t in range(512)], np.float64)
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1 / 12) < 0.005
    hist, _ = np.histogram(u, bins=16, range=(0, 1))
    exp = u.size / 16
    assert ((hist - exp) ** 2 / exp).sum() < 40.0               # chi-square, 15 dof: P(> 40) ~ 4e-4
    # rows and columns are not copies of one another
    assert abs(np.corrcoef(u[0], u[1])[0, 1]) < 0.5 and abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.2


def _setup(T=3000, E=16, k=3, seed=0):
    rng = np.random.default_rng(seed)
    s = rng.random((T, E)).astype(np.float32)
    idx, gate = orc.route(s, None, k, 1, 1, True)
    keep = np.ones(E, np.uint8)
    keep[[1, 6, 11, 12]] = 0
    return s, idx, gate, keep


def test_random_compensation_invariants():
    s, idx, gate, keep = _setup()
    E, k = s.shape[1], idx.shape[1]
    idx2, gate2 = orc.compensate(s, None, keep, idx, gate, True, orc.FLAG_COMP_RANDOM)
    n_aff = 0
    for t in range(s.shape[0]):
        orig, new = [int(e) for e in idx[t]], [int(e) for e in idx2[t]]
        lost = [e for e in orig if not keep[e]]
        if not lost:
            assert new == orig and np.array_equal(gate2[t].view(np.uint32), gate[t].view(np.uint32))   # untouched
            continue
        n_aff += 1
        assert all(keep[e] for e in new) and len(set(new)) == k                  # K_final in A_trans, k distinct
        assert set(e for e in orig if keep[e]) <= set(new)                       # surviving picks stay
        assert abs(float(gate2[t].sum()) - 1.0) < 1e-6                           # R16
        w = s[t, new] / s[t, new].sum(dtype=np.float32)
        assert np.allclose(gate2[t], w, rtol=1e-6)                               # gates from the unbiased scores
    assert n_aff > 1000


def test_random_replacements_are_uniform_and_not_the_top_scores():
    s, idx, gate, keep = _setup(T=6000)
    E = s.shape[1]
    idx_r, _ = orc.compensate(s, None, keep, idx, gate, True, orc.FLAG_COMP_RANDOM)
    idx_m, _ = orc.compensate(s, None, keep, idx, gate, True, 0)
    counts = np.zeros(E)
    same = tot = 0
    for t in range(s.shape[0]):
        orig = set(int(e) for e in idx[t])
        if all(keep[e] for e in orig):
            continue
        surv = set(e for e in orig if keep[e])
        repl = set(int(e) for e in idx_r[t]) - surv
        elig = [e for e in range(E) if keep[e] and e not in surv]
        for e in repl:
            counts[e] += 1.0 / len(repl) * len(repl)            # one count per replacement
        # expected share of every eligible expert for this token: |repl| / |elig|
        tot += 1
        same += set(int(e) for e in idx_m[t]) == set(int(e) for e in idx_r[t])
    kept = np.flatnonzero(keep)
    share = counts[kept] / counts[kept].sum()
    assert counts[keep == 0].sum() == 0
    assert np.abs(share - 1.0 / len(kept)).max() < 0.02          # each of the 12 survivors gets ~1/12 of the refills
    assert same / tot < 0.5                                      # it is not the masked top-k in disguise
