"""Oracle for the LFU expert cache of the offloading system (Fig. 8).

TEST INFRASTRUCTURE ONLY (same rule as oracle/oracle.py): imported by tests/ and by bench.py's
cpu_baseline leg, never by the product; it imports nothing from paper_2606_29982_b200/.

The paper fixes only this much: "each HBM caches only a subset of 1024 experts [of the 58 layers'
14848], managed by a Least Frequently Used (LFU) eviction policy"; a cache hit
costs nothing to move, a miss is one full H2D transfer of the expert.
Everything else is a reading, listed as R30-R34 in DESIGN.md §3 and followed here step by step:

  R30  keys are (layer, expert) pairs of ROUTED experts; shared experts never enter the cache.
  R31  frequency f(layer, expert) = number of steps in which that expert was executed (it is in
       the step's run list after pruning and compensation), hit or miss, counted from the
       creation of the cache and kept when the expert is evicted.
  R32  one step of one layer, given the ascending list of executed experts: (1) every listed
       expert's frequency goes up by one; (2) the listed experts that are not cached are
       inserted in ascending expert order, each into the lowest-numbered free slot if there is
       one, else into the slot of the victim; (3) the victim is the cached key with the smallest
       frequency among the keys that are not executed by this step, ties to the smaller
       (layer, expert).  No victim and no free slot: the step's working set does not fit, an error.
  R33  the cost model sees the cache as it is when the step starts (R(e,d) = 0 for a hit).
  R34  the cache starts empty.

PARITY UNPINNED by PAPER.md beyond the word "LFU": the paper prints no trace, count or rule to
check these readings against.  What pins this file is tests/test_oracle_lfu.py (a trace worked by
hand from R30-R34, the slots >= keys special case, invariants).

Plain Python on purpose: dictionaries and a linear scan, no heap, so that it can be checked against
the rules above by eye.
"""


class CacheFull(Exception):
    pass


class LFUCache:
    def __init__(self, n_slots):
        self.n_slots = int(n_slots)
        self.slot_key = [None] * self.n_slots      # slot -> (layer, expert) or None
        self.slot_of = {}                          # (layer, expert) -> slot
        self.freq = {}                             # (layer, expert) -> count (R31: never reset)
        self.hits = self.misses = self.evictions = 0

    def resident_mask(self, layer, E):
        """R33: 1 for the experts of `layer` that are cached right now."""
        return [1 if (layer, e) in self.slot_of else 0 for e in range(E)]

    def step(self, layer, experts):
        """R32.  experts: the routed experts executed by this step of `layer`.
        Returns (fetched, evicted): the misses in insertion order and the keys they displaced
        (None where a free slot was used)."""
        experts = sorted(set(int(e) for e in experts))
        in_use = set((layer, e) for e in experts)
        for key in in_use:
            self.freq[key] = self.freq.get(key, 0) + 1
        fetched, evicted = [], []
        for e in experts:
            key = (layer, e)
            if key in self.slot_of:
                self.hits += 1
                continue
            self.misses += 1
            slot, victim = None, None
            for s in range(self.n_slots):
                if self.slot_key[s] is None:
                    slot = s
                    break
            if slot is None:
                best = None
                for s in range(self.n_slots):
                    k = self.slot_key[s]
                    if k in in_use:
                        continue
                    cand = (self.freq.get(k, 0), k[0], k[1])
                    if best is None or cand < best[0]:
                        best = (cand, s)
                if best is None:
                    raise CacheFull(f"layer {layer}: {len(experts)} executed experts do not fit {self.n_slots} slots")
                slot = best[1]
                victim = self.slot_key[slot]
                del self.slot_of[victim]
                self.evictions += 1
            self.slot_key[slot] = key
            self.slot_of[key] = slot
            fetched.append(e)
            evicted.append(victim)
        return fetched, evicted

    def snapshot(self):
        """[(layer, expert, freq) or None] per slot."""
        return [None if k is None else (k[0], k[1], self.freq[k]) for k in self.slot_key]
