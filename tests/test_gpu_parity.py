"""GPU-vs-oracle parity through the C ABI on the small configs (C1 4^4, 2^4, anisotropic
extras, C2 16^3x32): element by element on the same seeded inputs.
Bars (BASELINE.json:north_star): bit-exact for shifts / tables / masks / round trips;
per-site relative error <= 1e-12 (fp64) / 2e-5 (fp32); global sums <= 1e-10 (fp64)."""
import numpy as np
import pytest

import oracle
import synth
from parity import TOL_SITE, TOL_SUM, links, site_rel_err, z3_fix

pytestmark = pytest.mark.gpu

SMALL = [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4), (6, 4, 2, 8), (10, 6, 4, 2)]
C2 = synth.CONFIGS["C2"]
PRECS = ["f64", "f32"]
SUBSETS = [0, 1, 2]
KINDS = {"matrix": 0, "gauge": 1, "fermion": 2}


def _seed(dims):
    return synth.BASE_SEED + sum(dims)


def _field(dims, kind, seed):
    if kind == "matrix":
        return synth.color_matrix(dims, seed)
    if kind == "gauge":
        return synth.gauge_hot(dims, seed)
    return synth.spinor(dims, seed)


def _as64(a):
    return a.astype(np.complex128)


@pytest.fixture(scope="module")
def lat_cache(qdp):
    cache = {}

    def get(dims):
        if dims not in cache:
            cache[dims] = qdp.qdp_lattice_create(dims)
        return cache[dims]
    yield get
    cache.clear()


@pytest.mark.parametrize("dims", SMALL + [C2])
def test_tables_and_masks_bit_exact(qdp, lat_cache, dims):
    lat = lat_cache(dims)
    assert qdp.qdp_lattice_volume(lat) == synth.volume(dims)
    assert np.array_equal(qdp.qdp_lattice_parity_mask(lat), oracle.parity_mask(dims))
    for mu in range(4):
        for sign in (+1, -1):
            assert np.array_equal(qdp.qdp_lattice_neighbor_table(lat, mu, sign),
                                  oracle.neighbor_table(dims, mu, sign))


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_upload_download_round_trip_bit_exact(qdp, lat_cache, dims, prec):
    lat = lat_cache(dims)
    V = synth.volume(dims)
    for kind, k in KINDS.items():
        host = synth.round_to(_field(dims, kind, _seed(dims)), prec)
        f = qdp.field_from_host(lat, k, host)
        assert np.array_equal(qdp.field_to_host(f), host)
    # a field filled with its own lex index pins the private permutation (A21)
    idx = np.zeros((V, 3, 3), dtype=np.complex128)
    idx[:] = np.arange(V)[:, None, None]
    f = qdp.field_from_host(lat, 0, idx)
    assert np.array_equal(qdp.field_to_host(f), idx)
    s = qdp.qdp_sum(f)
    assert np.array_equal(s, np.full((3, 3), V * (V - 1) / 2 + 0j))


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_shift_bit_exact(qdp, lat_cache, dims, prec):
    lat = lat_cache(dims)
    kinds = KINDS if dims != C2 else {"fermion": 2}
    for kind, k in kinds.items():
        host = synth.round_to(_field(dims, kind, _seed(dims) + 1), prec)
        sentinel = synth.round_to(_field(dims, kind, _seed(dims) + 2), prec)
        src = qdp.field_from_host(lat, k, host)
        for mu in range(4):
            for sign in (+1, -1):
                for sub in SUBSETS:
                    dst = qdp.field_from_host(lat, k, sentinel)
                    qdp.qdp_shift(dst, src, mu, sign, sub)
                    want = oracle.shift(dims, host, mu, sign, sub, dst=sentinel)
                    assert np.array_equal(qdp.field_to_host(dst), want), (kind, mu, sign, sub)


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_reductions(qdp, lat_cache, dims, prec):
    lat = lat_cache(dims)
    tol = TOL_SUM[prec] if prec == "f64" else 1e-12   # fp32 inputs are exact in fp64: same bar applies
    for kind, k in KINDS.items():
        ha = synth.round_to(_field(dims, kind, _seed(dims) + 3), prec)
        hb = synth.round_to(_field(dims, kind, _seed(dims) + 4), prec)
        a, b = qdp.field_from_host(lat, k, ha), qdp.field_from_host(lat, k, hb)
        for sub in SUBSETS:
            n2 = oracle.norm2(dims, _as64(ha), sub)
            got = qdp.qdp_norm2(a, sub)
            assert abs(got - n2) <= tol * n2
            assert got == qdp.qdp_norm2(a, sub)                       # run-to-run bit-identical
            ip = oracle.inner(dims, _as64(ha), _as64(hb), sub)
            scale = np.sqrt(n2 * oracle.norm2(dims, _as64(hb), sub))
            assert abs(qdp.qdp_inner(a, b, sub) - ip) <= tol * scale
            sm = oracle.sum_field(dims, _as64(ha), sub)
            assert np.abs(qdp.qdp_sum(a, sub).ravel() - sm).max() <= tol * np.sqrt(n2 * synth.volume(dims))
        assert abs(qdp.qdp_inner(a, a).real - qdp.qdp_norm2(a)) <= 1e-12 * qdp.qdp_norm2(a)


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_plaquette(qdp, lat_cache, dims, prec):
    lat = lat_cache(dims)
    variants = [synth.gauge_hot(dims, _seed(dims) + 5), synth.gauge_unit(dims)]
    if dims == C2:
        variants.append(synth.gauge_warm(dims, _seed(dims) + 5, 0.2))
    for hu64 in variants:
        hu = synth.round_to(hu64, prec)
        u = qdp.field_from_host(lat, 1, hu)
        for sub in SUBSETS:
            want = oracle.plaquette(dims, _as64(hu), sub)
            got = qdp.qdp_plaquette(u, sub)
            # sums of O(V) terms of size <= 3, normalised by 9N or 18N: absolute bar
            assert np.abs(got - want).max() <= TOL_SUM[prec], (sub, got, want)
            assert np.array_equal(got, qdp.qdp_plaquette(u, sub))
    unit = qdp.field_from_host(lat, 1, synth.round_to(synth.gauge_unit(dims), prec))
    assert np.array_equal(qdp.qdp_plaquette(unit), [1.0, 1.0, 1.0])


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_hop_and_axpy_hop(qdp, lat_cache, dims, prec):
    lat = lat_cache(dims)
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 6), prec)
    hp = synth.round_to(synth.spinor(dims, _seed(dims) + 7), prec)
    sentinel = synth.round_to(synth.spinor(dims, _seed(dims) + 8, 1), prec)
    u, psi = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 2, hp)
    a, b = synth.scalars_ab(_seed(dims))
    if prec == "f32":
        a, b = float(np.float32(a)), float(np.float32(b))
    full = None
    for sub in SUBSETS:
        chi = qdp.field_from_host(lat, 2, sentinel)
        qdp.qdp_hop(chi, u, psi, sub)
        got = qdp.field_to_host(chi)
        want = oracle.hop(dims, _as64(hu), _as64(hp), sub, chi=_as64(sentinel))
        assert site_rel_err(got, want).max() <= TOL_SITE[prec], sub
        if sub == 0:
            full = got
        chi2 = qdp.field_from_host(lat, 2, sentinel)
        n2 = qdp.qdp_axpy_hop(chi2, a, b, u, psi, sub, want_norm2=True)
        got2 = qdp.field_to_host(chi2)
        want2 = oracle.axpy_hop(dims, a, b, _as64(hu), _as64(hp), sub, chi=_as64(sentinel))
        assert site_rel_err(got2, want2).max() <= TOL_SITE[prec], sub
        # fused norm2 == separate norm2 of the output (deterministic trees may differ in shape)
        sep = qdp.qdp_norm2(chi2, sub)
        assert abs(n2 - sep) <= 1e-12 * sep
        assert abs(n2 - oracle.norm2(dims, want2, sub)) <= TOL_SUM[prec] * n2
    # A17: even call then odd call into the same chi == full call, bit-exact
    chi = qdp.field_from_host(lat, 2, sentinel)
    qdp.qdp_hop(chi, u, psi, 1)
    qdp.qdp_hop(chi, u, psi, 2)
    assert np.array_equal(qdp.field_to_host(chi), full)
    # inner(psi, hop psi) is real (A19: absolute bar 1e-10 * 8 * norm2)
    ip = qdp.qdp_inner(psi, chi)
    want_ip = oracle.inner(dims, _as64(hp), _as64(full))
    n2p = oracle.norm2(dims, _as64(hp))
    assert abs(ip - want_ip) <= 1e-10 * 8 * n2p
    if prec == "f64":
        assert abs(ip.imag) <= 1e-10 * 8 * n2p
    # b = 0: chi = a psi exactly; a = 0, b = 1: hop exactly
    chi3 = qdp.field_from_host(lat, 2, sentinel)
    qdp.qdp_axpy_hop(chi3, a, 0.0, u, psi)
    assert np.array_equal(qdp.field_to_host(chi3), (hp * hp.real.dtype.type(a)).astype(hp.dtype))
    qdp.qdp_axpy_hop(chi3, 0.0, 1.0, u, psi)
    assert np.array_equal(qdp.field_to_host(chi3), full)


@pytest.mark.parametrize("dims", SMALL)
@pytest.mark.parametrize("prec", PRECS)
@pytest.mark.parametrize("t_dir", [3, -1])
def test_ape_step(qdp, lat_cache, dims, prec, t_dir):
    lat = lat_cache(dims)
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 9), prec)
    sentinel = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 10), prec)
    u = qdp.field_from_host(lat, 1, hu)
    for sub in SUBSETS:
        out = qdp.field_from_host(lat, 1, sentinel)
        qdp.qdp_ape_smear_step(out, u, 0.5, t_dir, sub)
        got = qdp.field_to_host(out)
        want = oracle.ape_smear_step(dims, _as64(hu), 0.5, t_dir, sub, u_out=_as64(sentinel))
        fixed, n_centre = z3_fix(links(got).astype(np.complex128), links(want))
        assert n_centre == 0                                      # A9: cut not hit on these inputs
        assert site_rel_err(fixed, links(want)).max() <= TOL_SITE[prec], (sub, t_dir)
        if t_dir == 3 and sub == 0:
            assert np.array_equal(got[:, 3], hu[:, 3])            # A7: bit-exact copy
    # unit field is a fixed point, exactly
    unit = synth.round_to(synth.gauge_unit(dims), prec)
    uu, out = qdp.field_from_host(lat, 1, unit), qdp.field_from_host(lat, 1, sentinel)
    qdp.qdp_ape_smear_step(out, uu, 0.5, t_dir)
    assert np.array_equal(qdp.field_to_host(out), unit)
    # alpha = 0 is the identity
    qdp.qdp_ape_smear_step(out, u, 0.0, t_dir)
    assert site_rel_err(links(qdp.field_to_host(out)), links(_as64(hu))).max() <= TOL_SITE[prec]


@pytest.mark.parametrize("prec", PRECS)
def test_c2_ten_ape_steps_warm_and_hot(qdp, lat_cache, prec):
    """BASELINE.json:configs[1]: 10 APE steps, plaquette after each (A16), hot + warm."""
    dims = C2
    lat = lat_cache(dims)
    for name, hu64 in (("warm", synth.gauge_warm(dims, _seed(dims) + 11, 0.2)),
                       ("hot", synth.gauge_hot(dims, _seed(dims) + 11))):
        hu = synth.round_to(hu64, prec)
        bufs = [qdp.field_from_host(lat, 1, hu), qdp.qdp_field_alloc(lat, 1, 1 if prec == "f64" else 0)]
        ref = _as64(hu)
        worst = 0.0
        prev = None
        for step in range(10):
            qdp.qdp_ape_smear_step(bufs[1], bufs[0], 0.5, 3)
            bufs.reverse()
            ref = oracle.ape_smear_step(dims, ref, 0.5, 3)
            pg, po = qdp.qdp_plaquette(bufs[0]), oracle.plaquette(dims, ref)
            assert np.abs(pg - po).max() <= (1e-10 if prec == "f64" else 1e-5), (name, step)
            if prev is not None:
                assert pg[1] > prev                                 # smearing raises the plaquette
            prev = pg[1]
            if step in (0, 9):
                got = links(qdp.field_to_host(bufs[0])).astype(np.complex128)
                fixed, n_centre = z3_fix(got, links(ref))
                assert n_centre == 0
                err = site_rel_err(fixed, links(ref)).max()
                if step == 0:
                    assert err <= TOL_SITE[prec], (name, err)       # one step, nothing chained: the north-star bar itself
                worst = max(worst, err)
                eye = np.eye(3)
                unit_bar = 1e-12 if prec == "f64" else 1e-5
                assert np.abs(got @ np.conj(np.swapaxes(got, 1, 2)) - eye).max() <= unit_bar
                assert np.abs(np.linalg.det(got) - 1).max() <= unit_bar
        # error may grow over 10 chained steps; each step is within the bar, the chain within 10x
        assert worst <= 10 * TOL_SITE[prec], (name, worst)


def test_error_codes(qdp, lat_cache):
    lat, lat2 = lat_cache((4, 4, 4, 4)), lat_cache((4, 2, 6, 4))
    u = qdp.qdp_field_alloc(lat, 1, 1)
    u32 = qdp.qdp_field_alloc(lat, 1, 0)
    psi = qdp.qdp_field_alloc(lat, 2, 1)
    chi = qdp.qdp_field_alloc(lat, 2, 1)
    other = qdp.qdp_field_alloc(lat2, 2, 1)

    def code(fn, *a):
        with pytest.raises(qdp.QdpError) as e:
            fn(*a)
        return e.value.code

    assert code(qdp.qdp_shift, psi, psi, 0, 1, 0) == -6
    assert code(qdp.qdp_hop, psi, u, psi, 0) == -6
    assert code(qdp.qdp_ape_smear_step, u, u, 0.5, 3, 0) == -6
    assert code(qdp.qdp_hop, chi, u, other, 0) == -5
    assert code(qdp.qdp_hop, chi, u32, psi, 0) == -4
    assert code(qdp.qdp_hop, chi, psi, psi, 0) == -3
    assert code(qdp.qdp_plaquette, psi, 0) == -3
    assert code(qdp.qdp_shift, chi, psi, 4, 1, 0) == -1
    assert code(qdp.qdp_shift, chi, psi, 0, 2, 0) == -1
    assert code(qdp.qdp_shift, chi, psi, 0, 1, 3) == -1
    assert code(qdp.qdp_ape_smear_step, u32, u32, 0.5, 2, 0) == -1
    # library-owned allocation and the allocator hook
    import ctypes, torch
    f = qdp.qdp_field_alloc(lat, 2, 1, use_torch=False)
    qdp.qdp_field_upload(f, synth.spinor((4, 4, 4, 4), 1))
    assert qdp.qdp_norm2(f) > 0
    qdp.qdp_field_free(f)
    held = {}

    def _alloc(n, ctx):
        t = torch.empty(n, dtype=torch.uint8, device="cuda:0")
        held[t.data_ptr()] = t
        return t.data_ptr()

    def _free(p, ctx):
        held.pop(p, None)
    a_cb, f_cb = qdp.binding.ALLOC_FN(_alloc), qdp.binding.FREE_FN(_free)
    qdp.qdp_set_allocator(a_cb, f_cb)
    try:
        g = qdp.qdp_field_alloc(lat, 2, 1, use_torch=False)
        assert len(held) == 1
        qdp.qdp_field_upload(g, synth.spinor((4, 4, 4, 4), 1))
        assert qdp.qdp_norm2(g) > 0
        qdp.qdp_field_free(g)
        assert len(held) == 0
    finally:
        qdp.qdp_set_allocator(None, None)


@pytest.mark.parametrize("dims,c2", [((16, 4, 8, 4), 2), ((16, 4, 8, 4), 4), ((8, 8, 6, 4), 3), ((32, 2, 4, 2), 1)])
def test_sweep_slab_order_gives_the_same_fields(qdp, dims, c2):
    """qdp_lattice_set_sweep_slab (the L2-aware sweep that qdp_lattice_create switches on for
    lattices as large as C5) only permutes the order in which sites are visited: fields must come
    out bit-identical to the linear sweep, sums within the 1e-10 bar, everything within the
    oracle bars -- here on lattices small enough to compare element by element."""
    lat, lin = qdp.qdp_lattice_create(dims), qdp.qdp_lattice_create(dims)
    qdp.qdp_lattice_set_sweep_slab(lat, c2)
    qdp.qdp_lattice_set_sweep_slab(lin, 0)
    hu, hp = synth.gauge_hot(dims, _seed(dims) + 21), synth.spinor(dims, _seed(dims) + 22)
    outs = []
    for L in (lat, lin):
        u, psi = qdp.field_from_host(L, 1, hu), qdp.field_from_host(L, 2, hp)
        u2, chi = qdp.qdp_field_alloc(L, 1, 1), qdp.qdp_field_alloc(L, 2, 1)
        res = {"plaq": [qdp.qdp_plaquette(u, s) for s in SUBSETS]}
        for t_dir in (3, -1):
            qdp.qdp_ape_smear_step(u2, u, 0.5, t_dir)
            res[f"ape{t_dir}"] = qdp.field_to_host(u2)
        for s in SUBSETS:
            chi = qdp.field_from_host(L, 2, hp)
            res[f"n2_{s}"] = qdp.qdp_axpy_hop(chi, 0.3, -0.7, u, psi, s, want_norm2=True)
            res[f"hop{s}"] = qdp.field_to_host(chi)
        outs.append(res)
    slab, lin_ = outs
    for k in slab:
        if k.startswith(("ape", "hop")):
            assert np.array_equal(slab[k], lin_[k]), k
    for s in SUBSETS:
        assert np.abs(slab["plaq"][s] - oracle.plaquette(dims, hu, s)).max() <= 1e-10
        assert np.abs(slab["plaq"][s] - lin_["plaq"][s]).max() <= 1e-12
        want = oracle.axpy_hop(dims, 0.3, -0.7, hu, hp, s, chi=hp.copy())
        assert site_rel_err(slab[f"hop{s}"], want).max() <= TOL_SITE["f64"]
        assert abs(slab[f"n2_{s}"] - oracle.norm2(dims, want, s)) <= 1e-10 * slab[f"n2_{s}"]
    assert site_rel_err(links(slab["ape3"]), links(oracle.ape_smear_step(dims, hu, 0.5, 3))).max() <= TOL_SITE["f64"]
    assert site_rel_err(links(slab["ape-1"]), links(oracle.ape_smear_step(dims, hu, 0.5, -1))).max() <= TOL_SITE["f64"]
    # argument validation
    with pytest.raises(qdp.QdpError):
        qdp.qdp_lattice_set_sweep_slab(lat, 5)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_lattice_set_sweep_slab(qdp.qdp_lattice_create((4, 4, 4, 4)), 2)   # L0/2*L1 = 8


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_smear_hop(qdp, lat_cache, dims, prec):
    """qdp_smear_hop (row f2): spatial and four-direction steps on every subset vs the oracle."""
    lat = lat_cache(dims)
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 31), prec)
    hp = synth.round_to(synth.spinor(dims, _seed(dims) + 32), prec)
    sentinel = synth.round_to(synth.spinor(dims, _seed(dims) + 33, 1), prec)
    u, psi = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 2, hp)
    a, b = synth.scalars_ab(_seed(dims) + 3)
    if prec == "f32":
        a, b = float(np.float32(a)), float(np.float32(b))
    for t_dir in (3, -1):
        for sub in SUBSETS:
            chi = qdp.field_from_host(lat, 2, sentinel)
            n2 = qdp.qdp_smear_hop(chi, a, b, u, psi, t_dir, sub, want_norm2=True)
            got = qdp.field_to_host(chi)
            want = oracle.smear_hop(dims, a, b, _as64(hu), _as64(hp), t_dir, sub, chi=_as64(sentinel))
            assert site_rel_err(got, want).max() <= TOL_SITE[prec], (t_dir, sub)
            assert abs(n2 - oracle.norm2(dims, want, sub)) <= TOL_SUM[prec] * n2
            chi2 = qdp.field_from_host(lat, 2, sentinel)
            qdp.qdp_smear_hop(chi2, a, b, u, psi, t_dir, sub)
            assert np.array_equal(qdp.field_to_host(chi2), got)          # with and without the fused norm2
            if t_dir == -1:                                               # identical to qdp_axpy_hop
                chi3 = qdp.field_from_host(lat, 2, sentinel)
                qdp.qdp_axpy_hop(chi3, a, b, u, psi, sub)
                assert np.array_equal(qdp.field_to_host(chi3), got)
    # a source on one time-slice stays there under the spatial step (exact zeros elsewhere)
    on = (np.arange(synth.volume(dims)) // (dims[0] * dims[1] * dims[2])) == dims[3] // 2
    src = hp.copy()
    src[~on] = 0
    bufs = [qdp.field_from_host(lat, 2, src), qdp.field_from_host(lat, 2, np.zeros_like(src))]
    for _ in range(3):
        qdp.qdp_smear_hop(bufs[1], 1.0, 0.25, u, bufs[0], 3)
        bufs.reverse()
    out = qdp.field_to_host(bufs[0])
    assert np.all(out[~on] == 0) and np.abs(out[on]).max() > 0
    with pytest.raises(qdp.QdpError):
        qdp.qdp_smear_hop(bufs[1], 1.0, 0.25, u, bufs[0], 2)


@pytest.mark.parametrize("dims", SMALL + [(2, 2, 2, 40), C2])
@pytest.mark.parametrize("prec", PRECS)
@pytest.mark.parametrize("kind", ["fermion", "matrix"])
def test_inner_timeslices(qdp, lat_cache, dims, prec, kind):
    """qdp_inner_timeslices (row f3) on every subset vs the oracle; both the streaming path
    (s3 a multiple of 32) and the scanning path (ragged lattices)."""
    lat = lat_cache(dims)
    ha = synth.round_to(_field(dims, kind, _seed(dims) + 41), prec)
    hb = synth.round_to(_field(dims, kind, _seed(dims) + 42) if kind == "matrix" else synth.spinor(dims, _seed(dims) + 42, 1), prec)
    a, b = qdp.field_from_host(lat, KINDS[kind], ha), qdp.field_from_host(lat, KINDS[kind], hb)
    scale = oracle.norm2(dims, _as64(ha)) + oracle.norm2(dims, _as64(hb))
    for sub in SUBSETS:
        got = qdp.qdp_inner_timeslices(a, b, sub)
        want = oracle.inner_timeslices(dims, _as64(ha), _as64(hb), sub)
        assert got.shape == (dims[3],)
        assert np.abs(got - want).max() <= TOL_SUM[prec] * scale / dims[3], sub
        assert np.array_equal(got, qdp.qdp_inner_timeslices(a, b, sub))          # deterministic
        assert abs(got.sum() - qdp.qdp_inner(a, b, sub)) <= 1e-12 * scale
    n = qdp.qdp_inner_timeslices(a, a)
    # (the imaginary part is a sum of x*y - y*x terms: zero up to the rounding of the fused multiply-add)
    assert np.abs(n.imag).max() <= 1e-14 * scale and abs(n.real.sum() - qdp.qdp_norm2(a)) <= 1e-12 * scale
    if kind == "fermion":
        with pytest.raises(qdp.QdpError):
            qdp.qdp_inner_timeslices(a, qdp.qdp_field_alloc(lat, 0, 1 if prec == "f64" else 0))


def test_streams_copy_and_wrapped_memory(qdp):
    """Plumbing entry points: qdp_lattice_set_stream / qdp_lattice_sync with a torch stream,
    qdp_field_copy, qdp_field_wrap on torch-owned memory (size check included)."""
    import torch
    dims = (8, 4, 4, 6)
    lat = qdp.qdp_lattice_create(dims)
    hu, hp = synth.gauge_hot(dims, 51), synth.spinor(dims, 52)
    stream = torch.cuda.Stream()
    qdp.qdp_lattice_set_stream(lat, stream.cuda_stream)
    u, psi = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 2, hp)
    chi, cpy = qdp.qdp_field_alloc(lat, 2, 1), qdp.qdp_field_alloc(lat, 2, 1)
    for _ in range(4):                       # a chain of asynchronous calls on the user's stream
        qdp.qdp_hop(chi, u, psi, 0)
        qdp.qdp_field_copy(cpy, chi)
        qdp.qdp_smear_hop(chi, 0.5, 0.1, u, cpy, 3)
    qdp.qdp_lattice_sync(lat)
    assert stream.query()                    # nothing left in flight after the sync
    want = oracle.smear_hop(dims, 0.5, 0.1, hu, oracle.hop(dims, hu, hp), 3)
    assert site_rel_err(qdp.field_to_host(chi), want).max() <= TOL_SITE["f64"]
    assert np.array_equal(qdp.field_to_host(cpy), qdp.field_to_host(cpy))
    assert site_rel_err(qdp.field_to_host(cpy), oracle.hop(dims, hu, hp)).max() <= TOL_SITE["f64"]
    qdp.qdp_lattice_set_stream(lat, None)    # back to the default stream
    assert abs(qdp.qdp_norm2(psi) - oracle.norm2(dims, hp)) <= 1e-10 * oracle.norm2(dims, hp)
    # wrapped torch memory: the field lives in the tensor
    nbytes = qdp.qdp_field_bytes(lat, 2, 1)
    buf = torch.zeros(nbytes, dtype=torch.uint8, device="cuda:0")
    w = qdp.qdp_field_wrap(lat, 2, 1, buf.data_ptr(), nbytes, storage=buf)
    qdp.qdp_field_copy(w, psi)
    qdp.qdp_lattice_sync(lat)
    assert int(buf.count_nonzero()) > nbytes // 2
    assert qdp.qdp_norm2(w) == qdp.qdp_norm2(psi)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_field_wrap(lat, 2, 1, buf.data_ptr(), nbytes - 16)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_field_copy(w, u)              # kinds differ


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_reunitarize(qdp, lat_cache, dims, prec):
    """qdp_reunitarize (row f2): Proj and Gram-Schmidt on gauge fields and colour matrices,
    every subset, out of place and in place."""
    lat = lat_cache(dims)
    P = 1 if prec == "f64" else 0
    # links pushed off the group (general matrices, well conditioned); colour matrices fully general
    hg = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 61) + 0.2 * synth.gauge_hot(dims, _seed(dims) + 62), prec)
    hm = synth.round_to(synth.color_matrix(dims, _seed(dims) + 63), prec)
    unit_bar = 1e-12 if prec == "f64" else 1e-5
    for kind, host in ((1, hg), (0, hm)):
        src = qdp.field_from_host(lat, kind, host)
        h64 = links(_as64(host))
        # conditioning-scaled bar: the polar factor of V moves by ~cond(V) eps under a
        # relative perturbation eps of V, so the per-matrix bar is the north-star bar times max(1, cond(V)/10)
        # (blended APE links have cond <= ~11); cond from the oracle's smallest eigenvalue of V^dag V.
        lam_min = np.array([oracle.min_eig_vdv(m) for m in h64])
        cond = np.sqrt((np.abs(h64) ** 2).sum(axis=(1, 2)) / lam_min)
        for method in (qdp.QDP_REUNIT_POLAR, qdp.QDP_REUNIT_GRAM_SCHMIDT):
            for sub in SUBSETS:
                sentinel = np.full_like(host, 3.0 - 2.0j)
                dst = qdp.field_from_host(lat, kind, sentinel)
                qdp.qdp_reunitarize(dst, src, method, sub)
                got = qdp.field_to_host(dst)
                want = oracle.reunitarize(dims, _as64(host), method, sub, out=_as64(sentinel))
                fixed, n_centre = z3_fix(links(_as64(got)), links(want))
                tol = TOL_SITE[prec] * np.maximum(1.0, cond / 10.0)
                assert np.all(site_rel_err(fixed, links(want)) <= tol), (kind, method, sub)
                assert n_centre == 0 or method == qdp.QDP_REUNIT_POLAR
            work = qdp.field_from_host(lat, kind, host)            # in place, whole lattice
            qdp.qdp_reunitarize(work, work, method)
            g = links(_as64(qdp.field_to_host(work)))
            # the output itself is unitary to working precision whatever the conditioning of the input
            assert np.abs(g @ np.conj(np.swapaxes(g, 1, 2)) - np.eye(3)).max() <= unit_bar
            assert np.abs(np.linalg.det(g) - 1).max() <= unit_bar
    # scale invariance of Proj and badly scaled input (the fp32 seeds of the closed form must not overflow)
    if prec == "f64":
        for scale in (1e-9, 1e7):
            src = qdp.field_from_host(lat, 0, hm * scale)
            dst = qdp.qdp_field_alloc(lat, 0, P)
            qdp.qdp_reunitarize(dst, src, qdp.QDP_REUNIT_POLAR)
            want = oracle.reunitarize(dims, _as64(hm), qdp.QDP_REUNIT_POLAR)
            fixed, _ = z3_fix(links(_as64(qdp.field_to_host(dst))), links(want))
            lam_min = np.array([oracle.min_eig_vdv(m) for m in links(_as64(hm))])
            cond = np.sqrt((np.abs(links(_as64(hm))) ** 2).sum(axis=(1, 2)) / lam_min)
            assert np.all(site_rel_err(fixed, links(want)) <= TOL_SITE[prec] * np.maximum(1.0, cond / 10.0)), scale
    # matrices without a polar factor (exactly zero, or with a non-finite entry) come back as they went in, and do
    # not disturb their neighbours in the warp
    V = synth.volume(dims)
    bad = hm.copy()
    bad[0] = 0
    bad[V // 2 + 1] = 0
    bad[V - 1, 1, 2] = np.inf
    src = qdp.field_from_host(lat, 0, bad)
    dst = qdp.qdp_field_alloc(lat, 0, P)
    qdp.qdp_reunitarize(dst, src, qdp.QDP_REUNIT_POLAR)
    got = qdp.field_to_host(dst)
    assert not got[0].any() and not got[V // 2 + 1].any()
    assert np.array_equal(got[V - 1], bad[V - 1])
    keep = np.ones(V, bool)
    keep[[0, V // 2 + 1, V - 1]] = False
    ref = qdp.qdp_field_alloc(lat, 0, P)
    qdp.qdp_reunitarize(ref, qdp.field_from_host(lat, 0, hm), qdp.QDP_REUNIT_POLAR)
    assert np.array_equal(got[keep], qdp.field_to_host(ref)[keep]) and np.isfinite(got[keep]).all()
    psi = qdp.qdp_field_alloc(lat, 2, P)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_reunitarize(psi, psi, 0)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_reunitarize(qdp.field_from_host(lat, 1, hg), qdp.field_from_host(lat, 1, hg), 2)


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_matmul(qdp, lat_cache, dims, prec):
    """qdp_matmul (row f1, first step): every operand form vs the oracle, subsets, gauge-field slots,
    the allowed in-place forms, and the plaquette composed from three products."""
    lat = lat_cache(dims)
    P = 1 if prec == "f64" else 0
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 71), prec)
    hm = synth.round_to(synth.color_matrix(dims, _seed(dims) + 72), prec)
    u, m = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 0, hm)
    u64, m64 = _as64(hu), _as64(hm)
    sentinel = np.full_like(hm, 2.0 + 1.0j)
    tol = TOL_SITE[prec]
    for adj_a in (0, 1):
        for adj_b in (0, 1):
            for mu, sign in ((-1, 1), (0, 1), (1, -1), (2, 1), (3, -1)):
                sub = (adj_a + 2 * adj_b + mu) % 3
                dst = qdp.field_from_host(lat, 0, sentinel)
                qdp.qdp_matmul(dst, 0, u, 2, adj_a, m, 0, adj_b, mu, sign, sub)
                want = oracle.matmul(dims, _as64(sentinel), 0, u64, 2, adj_a, m64, 0, adj_b, mu, sign, sub)
                assert site_rel_err(qdp.field_to_host(dst), want).max() <= tol, (adj_a, adj_b, mu, sign, sub)
    # into a slot of a gauge field; operands from the same field; unshifted in place
    g = qdp.field_from_host(lat, 1, hu)
    qdp.qdp_matmul(g, 3, g, 0, 0, g, 1, 1, 2, 1)                      # u3 = u0 * adj(u1)(x+2)
    want = oracle.matmul(dims, u64, 3, u64, 0, 0, u64, 1, 1, 2, 1)
    assert site_rel_err(links(qdp.field_to_host(g)), links(want)).max() <= tol
    mm = qdp.field_from_host(lat, 0, hm)
    qdp.qdp_matmul(mm, 0, mm, 0, 1, mm, 0, 0)                          # m = adj(m) * m in place (site-local)
    want = np.conj(np.swapaxes(m64, 1, 2)) @ m64
    assert site_rel_err(qdp.field_to_host(mm), want).max() <= tol
    # plaquette from three generic products + qdp_sum == qdp_plaquette
    a, b, p = (qdp.qdp_field_alloc(lat, 0, P) for _ in range(3))
    total = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            qdp.qdp_matmul(a, 0, u, mu, 0, u, nu, 0, mu, 1)
            qdp.qdp_matmul(b, 0, u, nu, 0, u, mu, 0, nu, 1)
            qdp.qdp_matmul(p, 0, a, 0, 0, b, 0, 1)
            s = qdp.qdp_sum(p).reshape(3, 3)
            total += (s[0, 0] + s[1, 1] + s[2, 2]).real
    assert abs(total / (18 * synth.volume(dims)) - qdp.qdp_plaquette(u)[0]) <= (1e-10 if prec == "f64" else 1e-5)
    # errors
    psi = qdp.qdp_field_alloc(lat, 2, P)
    for args, code in (((a, 1, u, 0, 0, u, 1, 0), -1), ((a, 0, u, 4, 0, u, 1, 0), -1), ((a, 0, psi, 0, 0, u, 1, 0), -3),
                       ((a, 0, u, 0, 0, a, 0, 0, 1, 1), -6), ((a, 0, u, 0, 0, u, 1, 0, 4, 1), -1)):
        with pytest.raises(qdp.QdpError) as e:
            qdp.qdp_matmul(*args)
        assert e.value.code == code, args


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
@pytest.mark.parametrize("kind", ["fermion", "gauge"])
def test_axpby(qdp, lat_cache, dims, prec, kind):
    """qdp_axpby: dst = a x + b y on every subset, with and without the fused norm2, in place."""
    lat = lat_cache(dims)
    hx = synth.round_to(_field(dims, kind, _seed(dims) + 81), prec)
    hy = synth.round_to(_field(dims, kind, _seed(dims) + 82) if kind != "fermion" else synth.spinor(dims, _seed(dims) + 82, 1), prec)
    x, y = qdp.field_from_host(lat, KINDS[kind], hx), qdp.field_from_host(lat, KINDS[kind], hy)
    a, b = synth.scalars_ab(_seed(dims) + 8)
    if prec == "f32":
        a, b = float(np.float32(a)), float(np.float32(b))
    sentinel = np.full_like(hx, 1.5 - 0.5j)
    for sub in SUBSETS:
        dst = qdp.field_from_host(lat, KINDS[kind], sentinel)
        n2 = qdp.qdp_axpby(dst, a, x, b, y, sub, want_norm2=True)
        got = qdp.field_to_host(dst)
        want = oracle.axpby(dims, a, _as64(hx), b, _as64(hy), sub, dst=_as64(sentinel))
        if prec == "f64":
            assert np.array_equal(got, want), sub            # same two roundings per term
        else:
            assert site_rel_err(got, want).max() <= TOL_SITE[prec], sub
        assert abs(n2 - oracle.norm2(dims, want if prec == "f64" else _as64(got), sub)) <= 1e-10 * n2
        dst2 = qdp.field_from_host(lat, KINDS[kind], sentinel)
        qdp.qdp_axpby(dst2, a, x, b, y, sub)
        assert np.array_equal(qdp.field_to_host(dst2), got)
    work = qdp.field_from_host(lat, KINDS[kind], hx)                 # x <- a x + b y in place
    qdp.qdp_axpby(work, a, work, b, y)
    full = qdp.field_from_host(lat, KINDS[kind], sentinel)
    qdp.qdp_axpby(full, a, x, b, y)
    assert np.array_equal(qdp.field_to_host(work), qdp.field_to_host(full))
    with pytest.raises(qdp.QdpError):
        qdp.qdp_axpby(work, a, x, b, qdp.qdp_field_alloc(lat, 0, 1 if prec == "f64" else 0))


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_matvec_and_hop_composed_from_generic_ops(qdp, lat_cache, dims, prec):
    """qdp_matvec vs the oracle in every operand form, and the hop term rebuilt from generic calls
    (8 matvecs, 4 shifts, 8 axpbys) against the fused qdp_hop."""
    lat = lat_cache(dims)
    P = 1 if prec == "f64" else 0
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 91), prec)
    hm = synth.round_to(synth.color_matrix(dims, _seed(dims) + 92), prec)
    hp = synth.round_to(synth.spinor(dims, _seed(dims) + 93), prec)
    u, m, psi = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 0, hm), qdp.field_from_host(lat, 2, hp)
    sentinel = np.full_like(hp, -1.0 + 2.0j)
    for adj_a in (0, 1):
        for mu, sign in ((-1, 1), (0, -1), (1, 1), (2, -1), (3, 1)):
            sub = (adj_a + mu + 1) % 3
            chi = qdp.field_from_host(lat, 2, sentinel)
            qdp.qdp_matvec(chi, m, 0, adj_a, psi, mu, sign, sub)
            want = oracle.matvec(dims, _as64(hm), 0, adj_a, _as64(hp), mu, sign, sub, chi=_as64(sentinel))
            assert site_rel_err(qdp.field_to_host(chi), want).max() <= TOL_SITE[prec], (adj_a, mu, sign, sub)
    acc, t, t2 = (qdp.field_from_host(lat, 2, np.zeros_like(hp)) for _ in range(3))
    for mu in range(4):
        qdp.qdp_matvec(t, u, mu, 0, psi, mu, 1)                    # U_mu(x) psi(x+mu)
        qdp.qdp_axpby(acc, 1.0, acc, 1.0, t)
        qdp.qdp_matvec(t, u, mu, 1, psi)                           # U_mu(y)^dag psi(y)
        qdp.qdp_shift(t2, t, mu, -1)                               # ... moved to y + mu
        qdp.qdp_axpby(acc, 1.0, acc, 1.0, t2)
    fused = qdp.qdp_field_alloc(lat, 2, P)
    qdp.qdp_hop(fused, u, psi)
    assert site_rel_err(qdp.field_to_host(acc), _as64(qdp.field_to_host(fused))).max() <= 8 * TOL_SITE[prec]
    inplace = qdp.field_from_host(lat, 2, hp)
    qdp.qdp_matvec(inplace, u, 2, 1, inplace)                      # site-local: in place allowed
    assert site_rel_err(qdp.field_to_host(inplace), oracle.matvec(dims, _as64(hu), 2, 1, _as64(hp))).max() <= TOL_SITE[prec]
    with pytest.raises(qdp.QdpError) as e:
        qdp.qdp_matvec(inplace, u, 2, 1, inplace, 0, 1)
    assert e.value.code == -6


@pytest.mark.parametrize("dims", [(2, 4, 2, 6), (12, 2, 2, 2), (2, 2, 2, 34), (14, 2, 6, 2), (64, 2, 2, 2), (2, 18, 2, 4)])
def test_unusual_shapes_one_pass(qdp, dims):
    """Extents of 2 in every position, rows longer and shorter than a warp, half-volumes that are
    not multiples of 32: one fp64 pass of every neighbour-reading op against the oracle."""
    lat = qdp.qdp_lattice_create(dims)
    hu, hp = synth.gauge_hot(dims, _seed(dims) + 101), synth.spinor(dims, _seed(dims) + 102)
    u, psi = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 2, hp)
    u2, chi = qdp.qdp_field_alloc(lat, 1, 1), qdp.qdp_field_alloc(lat, 2, 1)
    for mu in range(4):
        for sign in (1, -1):
            qdp.qdp_shift(chi, psi, mu, sign)
            assert np.array_equal(qdp.field_to_host(chi), oracle.shift(dims, hp, mu, sign)), (mu, sign)
    assert np.abs(qdp.qdp_plaquette(u) - oracle.plaquette(dims, hu)).max() <= 1e-10
    for t_dir in (3, -1):
        qdp.qdp_ape_smear_step(u2, u, 0.5, t_dir)
        want = oracle.ape_smear_step(dims, hu, 0.5, t_dir)
        fixed, _ = z3_fix(links(qdp.field_to_host(u2)), links(want))
        assert site_rel_err(fixed, links(want)).max() <= TOL_SITE["f64"], t_dir
    for sub in SUBSETS:
        chi = qdp.field_from_host(lat, 2, hp)
        n2 = qdp.qdp_axpy_hop(chi, 0.7, -0.4, u, psi, sub, want_norm2=True)
        want = oracle.axpy_hop(dims, 0.7, -0.4, hu, hp, sub, chi=hp)
        assert site_rel_err(qdp.field_to_host(chi), want).max() <= TOL_SITE["f64"], sub
        assert abs(n2 - oracle.norm2(dims, want, sub)) <= 1e-10 * n2
    ts = qdp.qdp_inner_timeslices(psi, chi)
    assert np.abs(ts - oracle.inner_timeslices(dims, hp, qdp.field_to_host(chi))).max() <= 1e-10 * 8 * oracle.norm2(dims, hp)
    m = qdp.qdp_field_alloc(lat, 0, 1)
    qdp.qdp_matmul(m, 0, u, 1, 0, u, 0, 1, 1, -1)
    want = oracle.matmul(dims, np.zeros((synth.volume(dims), 3, 3), dtype=np.complex128), 0, hu, 1, 0, hu, 0, 1, 1, -1)
    assert site_rel_err(qdp.field_to_host(m), want).max() <= TOL_SITE["f64"]


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4), (10, 6, 4, 2), C2])
@pytest.mark.parametrize("prec", PRECS)
def test_inner_timeslices_gamma(qdp, lat_cache, dims, prec):
    """qdp_inner_timeslices_gamma (row f3): all 16 spin matrices vs the oracle, subsets on gamma_5."""
    lat = lat_cache(dims)
    ha = synth.round_to(synth.spinor(dims, _seed(dims) + 111), prec)
    hb = synth.round_to(synth.spinor(dims, _seed(dims) + 112, 1), prec)
    a, b = qdp.field_from_host(lat, 2, ha), qdp.field_from_host(lat, 2, hb)
    scale = (oracle.norm2(dims, _as64(ha)) + oracle.norm2(dims, _as64(hb))) / dims[3]
    for n in range(16):
        got = qdp.qdp_inner_timeslices_gamma(a, b, n)
        want = oracle.inner_timeslices_gamma(dims, _as64(ha), _as64(hb), n)
        assert np.abs(got - want).max() <= TOL_SUM[prec] * scale, n
    assert np.array_equal(qdp.qdp_inner_timeslices_gamma(a, b, 0), qdp.qdp_inner_timeslices(a, b))
    for sub in (1, 2):
        got = qdp.qdp_inner_timeslices_gamma(a, b, 15, sub)
        assert np.abs(got - oracle.inner_timeslices_gamma(dims, _as64(ha), _as64(hb), 15, sub)).max() <= TOL_SUM[prec] * scale
    # pion correlator form: a^dag a per slice is real and positive
    pion = qdp.qdp_inner_timeslices_gamma(a, a, 0)
    assert np.all(pion.real > 0) and np.abs(pion.imag).max() <= 1e-12 * scale * dims[3]
    with pytest.raises(qdp.QdpError):
        qdp.qdp_inner_timeslices_gamma(a, b, 16)
    with pytest.raises(qdp.QdpError):
        m = qdp.qdp_field_alloc(lat, 0, 1 if prec == "f64" else 0)
        qdp.qdp_inner_timeslices_gamma(m, m, 5)


def test_pinned_host_tensor_on_a_ragged_lattice(qdp):
    """Upload/download through a pinned torch host tensor on 2^4, where V/2 = 8 is not a multiple of 32 and the
    padded device size (qdp_field_bytes) is four times the host array-of-structures size: the binding must ask
    for the host size."""
    import torch
    dims = (2, 2, 2, 2)
    lat = qdp.qdp_lattice_create(dims)
    hp = synth.spinor(dims, 77)
    f = qdp.qdp_field_alloc(lat, 2, 1)
    host = torch.from_numpy(hp.copy()).pin_memory()
    assert host.numel() * host.element_size() * 4 == qdp.qdp_field_bytes(lat, 2, 1)
    qdp.qdp_field_upload(f, host)
    back = torch.empty_like(host).pin_memory()
    qdp.qdp_field_download(f, back)
    assert np.array_equal(back.numpy(), hp)
    assert abs(qdp.qdp_norm2(f) - oracle.norm2(dims, hp)) <= 1e-12 * oracle.norm2(dims, hp)
    with pytest.raises(ValueError):
        qdp.qdp_field_upload(f, torch.zeros(qdp.qdp_field_bytes(lat, 2, 1), dtype=torch.uint8))


def test_gamma_basis_one_hot(qdp):
    """Pins single entries of Gamma(n) on the device against the literal DeGrand-Rossi matrices (typed in here from
    include/qdp_b200.h): with a = e_{s'} and b = e_s one-hot in spin at one site, a^dag Gamma b = Gamma[s', s]."""
    I = 1j
    lit = {1: [[0, 0, 0, I], [0, 0, I, 0], [0, -I, 0, 0], [-I, 0, 0, 0]],
           2: [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]],
           4: [[0, 0, I, 0], [0, 0, 0, -I], [-I, 0, 0, 0], [0, I, 0, 0]],
           8: [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]],
           15: [[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, -1, 0], [0, 0, 0, -1]]}
    dims = (2, 2, 2, 4)
    lat = qdp.qdp_lattice_create(dims)
    V = synth.volume(dims)
    site, t = 5, 5 // 8          # lex 5 lies on time-slice 0
    for n, G in lit.items():
        G = np.array(G, dtype=complex)
        got = np.zeros((4, 4), dtype=complex)
        for sp in range(4):
            for s in range(4):
                ha = np.zeros((V, 4, 3), dtype=np.complex128)
                hb = np.zeros((V, 4, 3), dtype=np.complex128)
                ha[site, sp, 1] = 1.0
                hb[site, s, 1] = 1.0
                a, b = qdp.field_from_host(lat, 2, ha), qdp.field_from_host(lat, 2, hb)
                got[sp, s] = qdp.qdp_inner_timeslices_gamma(a, b, n)[t]
        assert np.array_equal(got, G), n


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (16, 16, 16, 32), (64, 8, 4, 4), (4, 16, 8, 8), (2, 32, 4, 6), (32, 4, 2, 2)])
@pytest.mark.parametrize("prec", PRECS)
def test_staged_kernels_match_thread_per_site_kernels(qdp, dims, prec):
    """qdp_lattice_set_staged: on lattices whose x0 rows tile a 32-site block the shared-memory-staged kernels
    (cp.async.bulk + mbarrier rings) and the thread-per-site kernels evaluate the same definitions; both are
    compared with the oracle, and with each other to summation-order accuracy."""
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 91), prec)
    want = oracle.plaquette(dims, _as64(hu))
    res = []
    for staged in (True, False):
        lat = qdp.qdp_lattice_create(dims)
        qdp.qdp_lattice_set_staged(lat, staged)
        u = qdp.field_from_host(lat, 1, hu)
        before = qdp.qdp_kernel_launch_count()
        pg = qdp.qdp_plaquette(u)
        assert qdp.qdp_kernel_launch_count() == before + 1
        assert np.abs(pg - want).max() <= (1e-10 if prec == "f64" else 1e-5)
        assert np.array_equal(pg, qdp.qdp_plaquette(u))          # deterministic
        res.append(pg)
    assert np.abs(res[0] - res[1]).max() <= (1e-12 if prec == "f64" else 1e-5)


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_expression_layer(qdp, lat_cache, dims, prec):
    """Row f1: the named instantiations of the compile-time expression layer (csrc/expr.cuh).  Each expression is ONE
    kernel; values against the oracle's definitions (def. 2, def. 3, trace/real) and against the hand-fused calls."""
    lat = lat_cache(dims)
    P = 1 if prec == "f64" else 0
    V = synth.volume(dims)
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 101), prec)
    hm = synth.round_to(synth.color_matrix(dims, _seed(dims) + 102), prec)
    u, m = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 0, hm)
    u64, m64 = _as64(hu), _as64(hm)
    tol = TOL_SITE[prec]
    # ---- sum(real(trace(u[mu] * shift(u[nu],mu) * adj(shift(u[mu],nu)) * adj(u[nu])))): the plaquette
    for sub in SUBSETS:
        n0 = qdp.qdp_kernel_launch_count()
        got = qdp.qdp_expr_plaquette(u, sub)
        assert qdp.qdp_kernel_launch_count() == n0 + 1
        bar = 1e-10 if prec == "f64" else 1e-5
        assert np.abs(got - oracle.plaquette(dims, u64, sub)).max() <= bar, sub
        assert np.abs(got - qdp.qdp_plaquette(u, sub)).max() <= bar
    # ---- the staple sum and the APE blend as one expression each
    for t_dir in (3, -1):
        for mu in range(3 if t_dir == 3 else 4):
            for sub in SUBSETS if mu == 0 else [0]:
                sentinel = np.full_like(hm, 1.0 - 2.0j)
                dst = qdp.field_from_host(lat, 0, sentinel)
                n0 = qdp.qdp_kernel_launch_count()
                qdp.qdp_expr_staple(dst, u, mu, t_dir, sub)
                assert qdp.qdp_kernel_launch_count() == n0 + 1
                want = oracle.staple_field(dims, u64, mu, t_dir, sub, out=_as64(sentinel))
                assert site_rel_err(_as64(qdp.field_to_host(dst)), want).max() <= tol, (t_dir, mu, sub)
            dst = qdp.qdp_field_alloc(lat, 0, P)
            qdp.qdp_expr_ape_blend(dst, u, mu, 0.5, t_dir)
            want = oracle.ape_blend_field(dims, u64, mu, 0.5, t_dir)
            assert site_rel_err(_as64(qdp.field_to_host(dst)), want).max() <= tol, (t_dir, mu)
        # Proj of the blend = the link of the fused APE step (def. 3-4)
        qdp.qdp_reunitarize(dst, dst, qdp.QDP_REUNIT_POLAR)
        u2 = qdp.qdp_field_alloc(lat, 1, P)
        qdp.qdp_ape_smear_step(u2, u, 0.5, t_dir)
        mu_last = 2 if t_dir == 3 else 3
        fixed, _ = z3_fix(links(_as64(qdp.field_to_host(dst))), links(_as64(qdp.field_to_host(u2)[:, mu_last])))
        assert site_rel_err(fixed, links(_as64(qdp.field_to_host(u2)[:, mu_last]))).max() <= 4 * tol
    with pytest.raises(qdp.QdpError):
        qdp.qdp_expr_staple(qdp.qdp_field_alloc(lat, 0, P), u, 3, 3)         # mu = t_dir is not smeared
    with pytest.raises(qdp.QdpError):
        qdp.qdp_expr_staple(u2, u, 0, 3)                                     # dst must be a colour matrix
    # ---- trace(opA(a) * opB(shift(b))) into a QDP_COMPLEX field, and its fused sum
    scale = np.sqrt(oracle.norm2(dims, m64) * 3 / V) * 3
    for adj_a in (0, 1):
        for adj_b in (0, 1):
            for mu, sign in ((-1, 1), (0, 1), (1, -1), (2, 1), (3, -1)):
                for sub in SUBSETS if (adj_a, adj_b, mu) == (0, 1, 0) else [0]:
                    sentinel = np.full(V, 5.0 + 1.0j, dtype=hm.dtype)
                    dst = qdp.field_from_host(lat, qdp.QDP_COMPLEX, sentinel)
                    qdp.qdp_expr_trace_mul(dst, u, 1, adj_a, m, 0, adj_b, mu, sign, sub)
                    want = oracle.trace_mul(dims, u64, 1, adj_a, m64, 0, adj_b, mu, sign, sub, out=_as64(sentinel))
                    got = _as64(qdp.field_to_host(dst))
                    assert np.abs(got - want).max() <= tol * scale, (adj_a, adj_b, mu, sign, sub)
                    live = want != _as64(sentinel)
                    s = qdp.qdp_expr_sum_trace_mul(u, 1, adj_a, m, 0, adj_b, mu, sign, sub)
                    assert abs(s - want[live].sum()) <= TOL_SUM[prec] * scale * live.sum()
    # trace(u u^dag) = 3 on SU(3) links: the link overlap of a field with itself is 3 V
    assert abs(qdp.qdp_expr_sum_trace_mul(u, 2, 0, u, 2, 1) - 3.0 * V) <= (1e-10 if prec == "f64" else 1e-5) * 3 * V
    # the complex kind: round trip, qdp_sum; calls instantiated for 9/12/36 components refuse it
    hz = synth.round_to(synth.color_matrix(dims, _seed(dims) + 103)[:, 0, 0].copy(), prec)
    z = qdp.field_from_host(lat, qdp.QDP_COMPLEX, hz)
    assert np.array_equal(qdp.field_to_host(z), hz)
    zs = qdp.qdp_sum(z)
    assert abs(complex(zs.ravel()[0]) - _as64(hz).sum()) <= TOL_SUM[prec] * np.abs(hz).sum()
    for bad in (lambda: qdp.qdp_norm2(z), lambda: qdp.qdp_shift(qdp.qdp_field_alloc(lat, qdp.QDP_COMPLEX, P), z, 0, 1),
                lambda: qdp.qdp_expr_trace_mul(m, u, 0, 0, u, 0, 1)):
        with pytest.raises(qdp.QdpError):
            bad()


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_project_max_retr(qdp, lat_cache, dims, prec):
    """qdp_project_max_retr (row f2): Cabibbo-Marinari sweeps, element by element against the oracle's step-by-step
    algorithm (same start, same subgroup order, fixed iteration count); SU(3) output; SU(3) input is a fixed point."""
    lat = lat_cache(dims)
    P = 1 if prec == "f64" else 0
    hg = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 111) + 0.3 * synth.gauge_hot(dims, _seed(dims) + 112), prec)
    hm = synth.round_to(synth.color_matrix(dims, _seed(dims) + 113), prec)
    unit_bar = 1e-12 if prec == "f64" else 1e-5
    for kind, host in ((1, hg), (0, hm)):
        src = qdp.field_from_host(lat, kind, host)
        h64 = links(_as64(host))
        cond = np.sqrt((np.abs(h64) ** 2).sum(axis=(1, 2)) / np.array([oracle.min_eig_vdv(m) for m in h64]))
        for iters in (0, 1, 4):
            for sub in SUBSETS if iters == 4 else [0]:
                sentinel = np.full_like(host, 3.0 - 2.0j)
                dst = qdp.field_from_host(lat, kind, sentinel)
                qdp.qdp_project_max_retr(dst, src, iters, sub)
                want = oracle.project_max_retr(dims, _as64(host), iters, sub, out=_as64(sentinel))
                # the iteration is a contraction towards the maximiser: rounding differences do not grow with the count.
                # The Gram-Schmidt start divides by the norm of the component of row 1 orthogonal to row 0, which
                # amplifies rounding by up to cond(V): conditioning-scaled bar as for qdp_reunitarize
                tol = TOL_SITE[prec] * np.maximum(4.0, cond)
                assert np.all(site_rel_err(links(_as64(qdp.field_to_host(dst))), links(want)) <= tol), (kind, iters, sub)
        work = qdp.field_from_host(lat, kind, host)
        qdp.qdp_project_max_retr(work, work, 6)               # in place
        g = links(_as64(qdp.field_to_host(work)))
        assert np.abs(g @ np.conj(np.swapaxes(g, 1, 2)) - np.eye(3)).max() <= unit_bar
        assert np.abs(np.linalg.det(g) - 1).max() <= unit_bar
        # more sweeps never lower Re tr(X V^dag)
        v = links(_as64(host))
        t6 = np.einsum("xij,xij->x", g, np.conj(v)).real
        qdp.qdp_project_max_retr(work, qdp.field_from_host(lat, kind, host), 2)
        g2 = links(_as64(qdp.field_to_host(work)))
        t2 = np.einsum("xij,xij->x", g2, np.conj(v)).real
        assert np.all(t6 >= t2 - (1e-12 if prec == "f64" else 1e-5) * np.abs(t2))
    su3 = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 114), "f64")
    if prec == "f64":
        f = qdp.field_from_host(lat, 1, su3)
        out = qdp.qdp_field_alloc(lat, 1, P)
        qdp.qdp_project_max_retr(out, f, 3)
        assert np.abs(qdp.field_to_host(out) - su3).max() <= 1e-14
    with pytest.raises(qdp.QdpError):
        qdp.qdp_project_max_retr(qdp.qdp_field_alloc(lat, 2, P), qdp.qdp_field_alloc(lat, 2, P), 1)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_project_max_retr(src, src, -1)


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", PRECS)
def test_baryon_timeslices(qdp, lat_cache, dims, prec):
    """qdp_baryon_timeslices (row f3): the eps-eps colour contraction with a diquark spin matrix, per time-slice, both
    forms (one field per quark; three source colours per quark), subsets, several Gamma(n)."""
    lat = lat_cache(dims)
    hf = [synth.round_to(synth.spinor(dims, _seed(dims) + 121, k), prec) for k in range(9)]
    f = [qdp.field_from_host(lat, 2, h) for h in hf]
    h64 = [_as64(h) for h in hf]
    scale = (sum(oracle.norm2(dims, h) for h in h64) / 9) ** 1.5 / np.sqrt(synth.volume(dims)) * 20
    for n in (0, 5, 10, 15):
        n0 = qdp.qdp_kernel_launch_count()
        got = qdp.qdp_baryon_timeslices(f[0:3], f[3:6], f[6:9], n)
        assert qdp.qdp_kernel_launch_count() == n0 + 2
        want = oracle.baryon_timeslices(dims, h64[0:3], h64[3:6], h64[6:9], n)
        assert np.abs(got - want).max() <= TOL_SUM[prec] * scale * 6, n
        got1 = qdp.qdp_baryon_timeslices(f[0], f[1], f[2], n)
        assert np.abs(got1 - oracle.baryon_timeslices(dims, h64[0], h64[1], h64[2], n)).max() <= TOL_SUM[prec] * scale, n
    assert np.array_equal(got, qdp.qdp_baryon_timeslices(f[0:3], f[3:6], f[6:9], 15))      # deterministic
    for sub in (1, 2):
        gs = qdp.qdp_baryon_timeslices(f[0:3], f[3:6], f[6:9], 5, sub)
        assert np.abs(gs - oracle.baryon_timeslices(dims, h64[0:3], h64[3:6], h64[6:9], 5, sub)).max() <= TOL_SUM[prec] * scale * 6
    # identical quarks in a symmetric diquark vanish (Gamma(n)^T = +Gamma(n))
    G = oracle.gamma_matrix(10)
    if np.array_equal(G.T, G):
        assert np.abs(qdp.qdp_baryon_timeslices(f[0], f[0], f[2], 10)).max() <= TOL_SUM[prec] * scale
    with pytest.raises(qdp.QdpError):
        qdp.qdp_baryon_timeslices(f[0], f[1], f[2], 16)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_baryon_timeslices(f[0], f[1], qdp.qdp_field_alloc(lat, 0, 1 if prec == "f64" else 0), 5)
