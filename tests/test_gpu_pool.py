"""Row f4 on the device: the pool sub-allocates one cudaMalloc, cached fields survive spill and page-in bit-exactly
(including write-back of modified objects), evictions follow the LRU model, and the allocator hook draws fields from
the pool."""
import numpy as np
import pytest

import oracle
import synth
from oracle.pool_model import PoolModel

pytestmark = pytest.mark.gpu


def test_cached_fields_survive_spill_and_page_in(qdp):
    import torch
    dims = (8, 8, 8, 8)
    lat = qdp.qdp_lattice_create(dims)
    nbytes = qdp.qdp_field_bytes(lat, qdp.QDP_FERMION, qdp.QDP_F64)
    cap = 3 * nbytes + 4096                       # room for three of the five spinor fields
    pool = qdp.qdp_pool_create(0, cap)
    model = PoolModel(cap)
    hosts, objs, mids, norms = [], [], [], []
    for k in range(5):
        hp = synth.spinor(dims, 1201, k)
        f = qdp.field_from_host(lat, qdp.QDP_FERMION, hp)            # device layout of the field ...
        qdp.qdp_lattice_sync(lat)
        hosts.append(f.storage.cpu().pin_memory())                   # ... kept on the host as raw bytes
        objs.append(qdp.qdp_cache_register(pool, hosts[-1]))
        mids.append(model.register(nbytes))
        norms.append(oracle.norm2(dims, hp))
    scale = [1.0] * 5
    base = None
    rng = np.random.default_rng(7)
    for step in range(40):
        k = int(rng.integers(5))
        write = bool(rng.integers(2))
        ptr = qdp.qdp_cache_acquire(objs[k], write)
        want_off, _ = model.acquire(mids[k])
        base = ptr - want_off if base is None else base
        assert ptr - base == want_off
        f = qdp.qdp_field_wrap(lat, qdp.QDP_FERMION, qdp.QDP_F64, ptr, nbytes)
        n2 = qdp.qdp_norm2(f)
        assert abs(n2 - scale[k] ** 2 * norms[k]) <= 1e-12 * n2, (step, k)
        if write:
            qdp.qdp_axpby(f, 1.0, f, 1.0, f)                         # f <- 2 f on the device only
            scale[k] *= 2.0
        qdp.qdp_field_free(f)                                        # waits for the lattice's stream
        qdp.qdp_cache_release(objs[k])
        model.release(mids[k])
        assert qdp.qdp_pool_eviction_log(pool) == model.evictions
    assert len(model.evictions) > 5
    for k in range(5):                                               # unregister writes modified residents back
        qdp.qdp_cache_unregister(objs[k])
        g = qdp.qdp_field_alloc(lat, qdp.QDP_FERMION, qdp.QDP_F64)
        g.storage.copy_(hosts[k])
        got = qdp.field_to_host(g)
        assert np.array_equal(got, scale[k] * synth.spinor(dims, 1201, k)), k     # powers of two: exact in fp64
    assert qdp.qdp_pool_stats(pool)["in_use"] == 0
    qdp.qdp_pool_destroy(pool)


def test_allocator_hook_draws_fields_from_the_pool(qdp):
    dims = (4, 4, 4, 4)
    pool = qdp.qdp_pool_create(0, 64 << 20)
    alloc, free_ = qdp.qdp_pool_hook_alloc()
    qdp.qdp_set_allocator(alloc, free_, pool.handle)
    try:
        lat = qdp.qdp_lattice_create(dims)                           # its scratch comes from the pool too
        used0 = qdp.qdp_pool_stats(pool)["in_use"]
        assert used0 > 0
        hp = synth.spinor(dims, 1202)
        f = qdp.qdp_field_alloc(lat, qdp.QDP_FERMION, qdp.QDP_F64, use_torch=False)
        assert qdp.qdp_pool_stats(pool)["in_use"] >= used0 + qdp.qdp_field_bytes(lat, qdp.QDP_FERMION, qdp.QDP_F64)
        qdp.qdp_field_upload(f, hp)
        assert abs(qdp.qdp_norm2(f) - oracle.norm2(dims, hp)) <= 1e-12 * oracle.norm2(dims, hp)
        qdp.qdp_field_free(f)
        assert qdp.qdp_pool_stats(pool)["in_use"] == used0
        qdp.qdp_lattice_destroy(lat)
        assert qdp.qdp_pool_stats(pool)["in_use"] == 0
    finally:
        qdp.qdp_set_allocator(None, None)
    qdp.qdp_pool_destroy(pool)
