"""Pins for the pool / LRU model (oracle/pool_model.py) and, without a GPU, the C++ pool of csrc/pool.cu run as an
address-range-only pool (device = -1) against that model on random traces."""
import random

import pytest

from oracle.pool_model import GRAN, PoolModel


def test_textbook_lru_reference_string():
    """Equal-size objects in a pool of three frames: the classic page-replacement example (reference string
    7 0 1 2 0 3 0 4 2 3 0 3 2 1 2 0 1 7 0 1) has 12 faults under LRU, with this victim sequence."""
    refs = [7, 0, 1, 2, 0, 3, 0, 4, 2, 3, 0, 3, 2, 1, 2, 0, 1, 7, 0, 1]
    m = PoolModel(3 * 4096)
    ids = {}
    faults = 0
    for page in refs:
        if page not in ids:
            ids[page] = m.register(4096)
        off, faulted = m.acquire(ids[page])
        assert off is not None
        m.release(ids[page])
        faults += faulted
    assert faults == 12
    back = {v: k for k, v in ids.items()}
    assert [back[i] for i in m.evictions] == [7, 1, 2, 3, 0, 4, 0, 3, 2]


def test_allocator_invariants_on_random_traces():
    rng = random.Random(5596)
    for _ in range(20):
        m = PoolModel(1 << 16)
        live = {}
        for _ in range(400):
            if live and rng.random() < 0.45:
                off = rng.choice(list(live))
                m.free_(off)
                del live[off]
            else:
                n = rng.choice([1, 100, 256, 257, 1000, 4096, 9000])
                off = m.alloc(n)
                if off is None:
                    assert max([s for _, s in m.free], default=0) < -(-n // GRAN) * GRAN     # really no block fits
                    continue
                assert off % GRAN == 0 and off not in live
                live[off] = -(-max(n, 1) // GRAN) * GRAN
            spans = sorted([(o, s) for o, s in live.items()] + list(m.free))
            assert spans[0][0] == 0 and sum(s for _, s in spans) == m.cap
            assert all(a[0] + a[1] == b[0] for a, b in zip(spans, spans[1:]))           # a partition: no overlap, no gap
            assert all(a[0] + a[1] != b[0] for a, b in zip(m.free, m.free[1:]))          # free neighbours are merged
            lowest = m.free[0][0] if m.free else None
            assert lowest is None or all(o != lowest for o in live)
        for off in list(live):
            m.free_(off)
        assert m.free == [(0, m.cap)]


def test_locked_objects_are_never_spilled_and_oom_is_reported():
    m = PoolModel(4 * 1024)
    a, b, c = m.register(2048), m.register(2048), m.register(2048)
    assert m.acquire(a)[0] == 0 and m.acquire(b)[0] == 2048
    assert m.acquire(c) == (None, False)                # both residents are locked
    m.release(a)
    assert m.acquire(c) == (0, True) and m.evictions == [a]
    m.release(b), m.release(c)
    assert m.acquire(a) == (2048, True) and m.evictions == [a, b]     # b was acquired before c


def _replay(qdp, seed, cap, nobj, steps):
    """The same random trace through the C++ pool (address-range-only) and the model."""
    rng = random.Random(seed)
    pool = qdp.qdp_pool_create(-1, cap)
    m = PoolModel(cap)
    base = None
    sizes = [rng.choice([300, 1024, 2000, 4096, 5000, 8192]) for _ in range(nobj)]
    objs = [qdp.qdp_cache_register(pool, None, s) for s in sizes]
    mids = [m.register(s) for s in sizes]
    locked = set()
    raw = {}
    for _ in range(steps):
        r = rng.random()
        if r < 0.55:
            i = rng.randrange(nobj)
            want, _ = m.acquire(mids[i])
            if want is None:
                with pytest.raises(qdp.QdpError) as e:
                    qdp.qdp_cache_acquire(objs[i], rng.random() < 0.5)
                assert e.value.code == -7
            else:
                ptr = qdp.qdp_cache_acquire(objs[i], rng.random() < 0.5)
                base = ptr - want if base is None else base
                assert ptr - base == want
                if i in locked or rng.random() < 0.7:
                    qdp.qdp_cache_release(objs[i])
                    m.release(mids[i])
                else:
                    locked.add(i)
        elif r < 0.7 and locked:
            i = locked.pop()
            qdp.qdp_cache_release(objs[i])
            m.release(mids[i])
        elif r < 0.9:
            n = rng.choice([256, 700, 3000])
            want = m.alloc(n)
            if want is None:
                with pytest.raises(qdp.QdpError):
                    qdp.qdp_pool_alloc(pool, n)
            else:
                ptr = qdp.qdp_pool_alloc(pool, n)
                base = ptr - want if base is None else base
                assert ptr - base == want
                raw[ptr] = want
        elif raw:
            ptr = rng.choice(list(raw))
            qdp.qdp_pool_free(pool, ptr)
            m.free_(raw.pop(ptr))
        assert qdp.qdp_pool_eviction_log(pool) == m.evictions
        assert qdp.qdp_pool_stats(pool) == m.stats()
        for i in range(nobj):
            assert qdp.qdp_cache_is_resident(objs[i]) == (m.objs[mids[i]]["off"] is not None)
    for i in locked:
        qdp.qdp_cache_release(objs[i])
    for ptr in raw:
        qdp.qdp_pool_free(pool, ptr)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_pool_destroy(pool)                      # objects still registered
    for o in objs:
        qdp.qdp_cache_unregister(o)
    assert qdp.qdp_pool_stats(pool)["in_use"] == 0 and qdp.qdp_pool_stats(pool)["free_blocks"] == 1
    qdp.qdp_pool_destroy(pool)


@pytest.mark.parametrize("seed", range(6))
def test_cpp_pool_follows_the_model_on_random_traces(qdp, seed):
    _replay(qdp, 1000 + seed, cap=rng_cap(seed), nobj=9, steps=600)


def rng_cap(seed):
    return [16 * 1024, 20 * 1024, 24 * 1024 + 100, 32 * 1024, 12 * 1024, 64 * 1024][seed]


def test_cpp_pool_textbook_lru(qdp):
    refs = [7, 0, 1, 2, 0, 3, 0, 4, 2, 3, 0, 3, 2, 1, 2, 0, 1, 7, 0, 1]
    pool = qdp.qdp_pool_create(-1, 3 * 4096)
    objs = {}
    for page in refs:
        if page not in objs:
            objs[page] = qdp.qdp_cache_register(pool, None, 4096)
        qdp.qdp_cache_acquire(objs[page])
        qdp.qdp_cache_release(objs[page])
    by_id = {qdp.qdp_cache_id(o): page for page, o in objs.items()}
    assert [by_id[i] for i in qdp.qdp_pool_eviction_log(pool)] == [7, 1, 2, 3, 0, 4, 0, 3, 2]
    for o in objs.values():
        qdp.qdp_cache_unregister(o)
    qdp.qdp_pool_destroy(pool)


def test_destroy_and_unregister_refuse_while_memory_is_in_use(qdp):
    """A pool with a live block is not destroyed (the block would dangle), and an unregister that is refused because the
    object is still acquired keeps the Python handle so that it can be retried."""
    pool = qdp.qdp_pool_create(-1, 16 * 1024)
    ptr = qdp.qdp_pool_alloc(pool, 1024)
    with pytest.raises(qdp.QdpError) as e:
        qdp.qdp_pool_destroy(pool)
    assert "still allocated" in str(e.value) and pool.handle
    qdp.qdp_pool_free(pool, ptr)
    obj = qdp.qdp_cache_register(pool, None, 4096)
    qdp.qdp_cache_acquire(obj)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_cache_unregister(obj)
    assert obj.handle
    qdp.qdp_cache_release(obj)
    qdp.qdp_cache_unregister(obj)
    assert obj.handle is None
    qdp.qdp_pool_destroy(pool)
    assert pool.handle is None
