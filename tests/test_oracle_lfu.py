"""Pins for the LFU cache oracle (oracle/lfu_cache.py): a hand-worked example, the cases that
reduce to set arithmetic, and invariants checked on random traces."""
import random

import pytest

from oracle.lfu_cache import CacheFull, LFUCache
from tests.golden_io import read_golden


def _ints(v):
    return [int(x) for x in v]


def test_hand_example():
    g = read_golden("lfu_hand_example.txt")
    c = LFUCache(int(g["n_slots"][0]))
    for i in range(1, 6):
        fetched, evicted = c.step(0, _ints(g[f"step{i}"]))
        assert fetched == _ints(g[f"fetched{i}"]), i
        assert [-1 if v is None else v[1] for v in evicted] == _ints(g[f"evicted{i}"]), i
    snap = c.snapshot()
    assert [s[1] for s in snap] == _ints(g["slots_expert"])
    assert [s[2] for s in snap] == _ints(g["slots_freq"])
    assert (c.hits, c.misses, c.evictions) == (int(g["hits"][0]), int(g["misses"][0]), int(g["evictions"][0]))
    with pytest.raises(CacheFull):
        c.step(0, _ints(g["step6"]))


def test_two_layer_tie_goes_to_the_smaller_key():
    g = read_golden("lfu_hand_example.txt")
    c = LFUCache(2)
    c.step(0, [5])
    c.step(1, [2])
    _, evicted = c.step(0, [1])
    assert evicted == [tuple(_ints(g["two_layer_victim"]))]
    assert c.resident_mask(0, 8) == [0, 1, 0, 0, 0, 0, 0, 0] and c.resident_mask(1, 4) == [0, 0, 1, 0]


def test_large_cache_has_only_compulsory_misses():
    """n_slots >= number of distinct keys: no eviction ever; misses = distinct keys, hits = the rest."""
    rng = random.Random(1)
    c = LFUCache(3 * 16)
    seen, touches = set(), 0
    for _ in range(200):
        layer = rng.randrange(3)
        ex = rng.sample(range(16), rng.randint(1, 6))
        c.step(layer, ex)
        seen |= {(layer, e) for e in ex}
        touches += len(ex)
    assert c.evictions == 0 and c.misses == len(seen) and c.hits == touches - len(seen)


@pytest.mark.parametrize("seed", range(4))
def test_invariants_on_random_traces(seed):
    rng = random.Random(seed)
    L, E, n_slots = 3, 12, 9
    c = LFUCache(n_slots)
    count = {}
    for step in range(300):
        layer = rng.randrange(L)
        ex = sorted(rng.sample(range(E), rng.randint(1, 5)))
        before = {s[:2]: s[2] for s in c.snapshot() if s is not None}
        free_before = sum(1 for s in c.snapshot() if s is None)
        fetched, evicted = c.step(layer, ex)
        for e in ex:
            count[(layer, e)] = count.get((layer, e), 0) + 1
        snap = [s for s in c.snapshot() if s is not None]
        keys = [s[:2] for s in snap]
        assert len(keys) == len(set(keys)) <= n_slots                      # one slot per key, capacity
        assert all((layer, e) in keys for e in ex)                         # executed => cached afterwards
        assert fetched == [e for e in ex if (layer, e) not in before]      # misses, ascending
        assert all(s[2] == count[s[:2]] for s in snap)                     # R31: f = executions so far
        assert sum(v is None for v in evicted) == min(free_before, len(fetched))   # free slots first
        in_use = {(layer, e) for e in ex}
        survivors = set(before) - {v for v in evicted if v is not None}
        for v in evicted:
            if v is None:
                continue
            assert v not in in_use and v in before
            # nothing that stayed (and was evictable) was less frequently used than a victim
            for k in survivors - in_use:
                assert (before[k], k) > (before[v], v) or k in {x for x in evicted if x is not None}


def test_frequency_survives_eviction():
    c = LFUCache(1)
    c.step(0, [0]); c.step(0, [0]); c.step(0, [1])       # 0 evicted with f = 2
    c.step(0, [0])                                       # back in: f = 3, not 1
    assert c.snapshot() == [(0, 0, 3)]
