"""Oracle for the memory-pool / LRU residency policy of SURVEY.md 8(f) row f4: a plain Python model
of the policy stated in include/qdp_b200.h, sharing no code with csrc/pool.cu.  TEST INFRASTRUCTURE ONLY.

Policy.  Allocation granularity 256 bytes.  First fit: the free block with the lowest offset that is large enough; the
allocation takes the front of that block.  A freed block merges with free neighbours.  When nothing fits, the resident
cached object with no outstanding acquire that was least recently acquired (an object never acquired is older than
any acquired one; among those, registration order) is spilled, and the search is repeated; if no such object exists
the allocation fails.  acquire() of a resident object only locks it and makes it the most recently used.

Pinned (tests/test_oracle_pool.py): the textbook LRU page-replacement example (equal-size objects: reference string
7 0 1 2 0 3 0 4 2 3 0 3 2 1 2 0 1 7 0 1 with three frames gives 12 faults), and allocator invariants (no overlap,
alignment, conservation of bytes, full coalescing)."""
GRAN = 256


def round_up(n):
    return (max(n, 1) + GRAN - 1) // GRAN * GRAN


class PoolModel:
    def __init__(self, capacity):
        self.cap = capacity // GRAN * GRAN
        self.free = [(0, self.cap)]          # (offset, size), sorted by offset
        self.used = {}                       # offset -> size
        self.objs = []                       # cached objects: dicts
        self.lru = []                        # ids, most recently acquired first
        self.evictions = []

    # ---- allocator -------------------------------------------------------
    def _first_fit(self, need):
        for i, (off, size) in enumerate(self.free):
            if size >= need:
                if size == need:
                    del self.free[i]
                else:
                    self.free[i] = (off + need, size - need)
                self.used[off] = need
                return off
        return None

    def _give_back(self, off):
        size = self.used.pop(off)
        self.free.append((off, size))
        self.free.sort()
        merged = []
        for o, s in self.free:
            if merged and merged[-1][0] + merged[-1][1] == o:
                merged[-1] = (merged[-1][0], merged[-1][1] + s)
            else:
                merged.append((o, s))
        self.free = merged

    def _spill_one(self):
        for oid in reversed(self.lru):
            ob = self.objs[oid]
            if ob["off"] is not None and ob["locks"] == 0:
                self._give_back(ob["off"])
                ob["off"] = None
                self.evictions.append(oid)
                return True
        return False

    def alloc(self, nbytes):
        need = round_up(nbytes)
        while True:
            off = self._first_fit(need)
            if off is not None:
                return off
            if not self._spill_one():
                return None          # out of memory

    def free_(self, off):
        self._give_back(off)

    # ---- cached objects ----------------------------------------------------
    def register(self, nbytes):
        oid = len(self.objs)
        self.objs.append({"bytes": nbytes, "off": None, "locks": 0, "alive": True})
        self.lru.append(oid)         # never acquired: least recently used
        return oid

    def acquire(self, oid):
        ob = self.objs[oid]
        faulted = False
        if ob["off"] is None:
            off = self.alloc(ob["bytes"])
            if off is None:
                return None, False
            ob["off"] = off
            faulted = True
        ob["locks"] += 1
        self.lru.remove(oid)
        self.lru.insert(0, oid)
        return ob["off"], faulted

    def release(self, oid):
        self.objs[oid]["locks"] -= 1

    def unregister(self, oid):
        ob = self.objs[oid]
        if ob["off"] is not None:
            self._give_back(ob["off"])
            ob["off"] = None
        ob["alive"] = False
        self.lru.remove(oid)

    def stats(self):
        return {"capacity": self.cap, "in_use": sum(self.used.values()),
                "largest_free": max([s for _, s in self.free], default=0), "free_blocks": len(self.free)}
