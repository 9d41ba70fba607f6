"""GPU-vs-oracle parity at BASELINE.json's full sizes (C3 24^3x64, C4 32^3x64, C5 48^3x96), in the
launch configuration bench.py times: sampled sites the oracle computes one by one
(`oracle.ape_site`, `oracle.hop_site`, `oracle.plaquette_site`), whole-lattice sums where the oracle
finishes in seconds, and properties that hold at any size (A17 even+odd = full bit-exactly, time
links untouched, unitarity and det = 1, fused norm2 = separate norm2, run-to-run identical sums).
Bars: BASELINE.json:north_star (per site 1e-12 fp64 / 2e-5 fp32; sums 1e-10 fp64)."""
import numpy as np
import pytest

import oracle
import synth
from parity import TOL_SITE, TOL_SUM, links, site_rel_err, z3_fix

pytestmark = pytest.mark.gpu

N_SAMPLE = 1500


def _sample_sites(dims, seed, n=N_SAMPLE):
    """Seeded sample of lex sites: uniform draws plus the corners and faces where the periodic
    wrap and the 32-site block boundaries of the device layout sit."""
    V = synth.volume(dims)
    rng = np.random.default_rng(seed)
    lex = set(int(v) for v in rng.integers(0, V, size=n))
    L0, L1, L2, L3 = dims
    for x3 in (0, L3 - 1):
        for x2 in (0, L2 - 1):
            for x1 in (0, 1, L1 - 1):
                for x0 in (0, 1, 31 % L0, L0 - 1):
                    lex.add(x0 + L0 * (x1 + L1 * (x2 + L2 * x3)))
    return np.array(sorted(lex), dtype=np.int64)


def _as64(a):
    return a.astype(np.complex128, copy=False)


def _prec_id(prec):
    return 1 if prec == "f64" else 0


def _check_step(qdp, dims, prec, seed, n_ape_steps=1, warm=False):
    """One pass of the ops bench.py times, checked against the oracle on sampled sites."""
    lat = qdp.qdp_lattice_create(dims)
    V = synth.volume(dims)
    hu = synth.round_to(synth.gauge_warm(dims, seed, 0.2) if warm else synth.gauge_hot(dims, seed), prec)
    hp = synth.round_to(synth.spinor(dims, seed), prec)
    a, b = synth.scalars_ab(seed)
    if prec == "f32":
        a, b = float(np.float32(a)), float(np.float32(b))
    u64, p64 = _as64(hu), _as64(hp)
    sites = _sample_sites(dims, seed)
    u, psi = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 2, hp)
    u2 = qdp.qdp_field_alloc(lat, 1, _prec_id(prec))
    chi = qdp.qdp_field_alloc(lat, 2, _prec_id(prec))

    # ---- plaquette: whole-lattice oracle sum, even + odd = all, run-to-run identical
    pg = qdp.qdp_plaquette(u)
    po = oracle.plaquette(dims, u64)
    bar = 1e-10 if prec == "f64" else 1e-6
    assert np.abs(pg - po).max() <= bar, (pg, po)
    assert np.array_equal(pg, qdp.qdp_plaquette(u))
    pe, pod = qdp.qdp_plaquette(u, 1), qdp.qdp_plaquette(u, 2)
    assert np.abs(0.5 * (pe + pod) - pg).max() <= bar

    # ---- one APE step (alpha = 0.5, spatial): sampled links, time links bit-exact, SU(3)
    qdp.qdp_ape_smear_step(u2, u, 0.5, 3)
    got_u = qdp.field_to_host(u2)
    assert np.array_equal(got_u[:, 3], hu[:, 3])
    for mu in range(3):
        want = np.stack([oracle.ape_site(dims, u64, int(s), mu, 0.5, 3) for s in sites])
        fixed, n_centre = z3_fix(_as64(got_u[sites, mu]), want)
        assert n_centre == 0
        assert site_rel_err(fixed, want).max() <= TOL_SITE[prec], mu
    g = _as64(got_u[sites, :3]).reshape(-1, 3, 3)
    unit_bar = 1e-12 if prec == "f64" else 1e-5
    assert np.abs(g @ np.conj(np.swapaxes(g, 1, 2)) - np.eye(3)).max() <= unit_bar
    assert np.abs(np.linalg.det(g) - 1).max() <= unit_bar

    # ---- further APE steps (ping-pong, A16): the plaquette triple is recorded after EVERY step and compared with the
    # oracle's plaquette of the downloaded device field of that step (whole-lattice sum, nothing chained); the spatial
    # plaquette rises, links stay in SU(3); the last step is also compared link by link with the oracle on the sampled
    # sites, restarted from the downloaded field of the step before it
    if n_ape_steps > 1:
        bufs = [u2, qdp.qdp_field_alloc(lat, 1, _prec_id(prec))]
        prev = qdp.qdp_plaquette(bufs[0])[1]
        triples = []
        field = _as64(got_u)                      # the device field after the first step, downloaded above
        for k in range(n_ape_steps - 1):
            before = field
            qdp.qdp_ape_smear_step(bufs[1], bufs[0], 0.5, 3)
            bufs.reverse()
            triple = qdp.qdp_plaquette(bufs[0])
            triples.append(triple)
            field = _as64(qdp.field_to_host(bufs[0]))
            assert np.abs(triple - oracle.plaquette(dims, field)).max() <= bar, ("plaquette after APE step", k + 2)
            assert triple[1] > prev
            prev = triple[1]
        assert len(triples) == n_ape_steps - 1 and np.all(np.isfinite(np.array(triples)))
        got_last = field
        for mu in range(3):
            want = np.stack([oracle.ape_site(dims, before, int(s), mu, 0.5, 3) for s in sites])
            fixed, n_centre = z3_fix(_as64(got_last[sites, mu]), want)
            assert n_centre == 0
            assert site_rel_err(fixed, want).max() <= TOL_SITE[prec], ("last APE step", mu)
        assert np.array_equal(got_last[:, 3], hu[:, 3])
        g = _as64(got_last[sites, :3]).reshape(-1, 3, 3)
        assert np.abs(g @ np.conj(np.swapaxes(g, 1, 2)) - np.eye(3)).max() <= unit_bar
        assert np.abs(np.linalg.det(g) - 1).max() <= unit_bar

    # ---- hop on EVEN then ODD (A17) == full hop bit-exactly; sampled sites vs the oracle
    qdp.qdp_hop(chi, u, psi, 1)
    qdp.qdp_hop(chi, u, psi, 2)
    eo = qdp.field_to_host(chi)
    chi_full = qdp.qdp_field_alloc(lat, 2, _prec_id(prec))
    qdp.qdp_hop(chi_full, u, psi, 0)
    full = qdp.field_to_host(chi_full)
    assert np.array_equal(eo, full)
    want = np.stack([oracle.hop_site(dims, u64, p64, int(s)) for s in sites])
    assert site_rel_err(_as64(full[sites]), want).max() <= TOL_SITE[prec]

    # ---- inner(psi, hop psi): whole-lattice oracle sum on the downloaded field; real (Hermitian)
    ip = qdp.qdp_inner(psi, chi_full)
    n2p = oracle.norm2(dims, p64)
    assert abs(ip - oracle.inner(dims, p64, _as64(full))) <= (1e-10 if prec == "f64" else 1e-6) * 8 * n2p
    assert abs(ip.imag) <= (1e-10 if prec == "f64" else 1e-5) * 8 * n2p

    # ---- chi = a psi + b hop(psi) with fused norm2; separate norm2; oracle norm2 of the output
    n2 = qdp.qdp_axpy_hop(chi, a, b, u, psi, 0, want_norm2=True)
    out = qdp.field_to_host(chi)
    want = a * p64[sites] + b * want
    assert site_rel_err(_as64(out[sites]), want).max() <= TOL_SITE[prec]
    sep = qdp.qdp_norm2(chi)
    assert abs(n2 - sep) <= 1e-12 * sep
    assert abs(sep - oracle.norm2(dims, _as64(out))) <= 1e-10 * sep
    assert sep == qdp.qdp_norm2(chi)
    ne, no_ = qdp.qdp_norm2(chi, 1), qdp.qdp_norm2(chi, 2)
    assert abs(ne + no_ - sep) <= 1e-12 * sep

    # ---- quark-smearing step (row f2): spatial hops only, sampled sites vs the oracle
    n2 = qdp.qdp_smear_hop(chi, a, b, u, psi, 3, 0, want_norm2=True)
    out = qdp.field_to_host(chi)
    want = a * p64[sites] + b * np.stack([oracle.hop_site_dirs(dims, u64, p64, int(s), 3) for s in sites])
    assert site_rel_err(_as64(out[sites]), want).max() <= TOL_SITE[prec]
    assert abs(n2 - oracle.norm2(dims, _as64(out))) <= 1e-10 * n2

    # ---- time-slice inner products (row f3): whole-lattice oracle on the downloaded fields
    ts = qdp.qdp_inner_timeslices(psi, chi)
    want_ts = oracle.inner_timeslices(dims, p64, _as64(out))
    assert np.abs(ts - want_ts).max() <= (1e-10 if prec == "f64" else 1e-6) * 8 * n2p
    assert abs(ts.sum() - qdp.qdp_inner(psi, chi)) <= 1e-12 * 8 * n2p

    # ---- shift: bit-exact on the whole lattice (one direction per axis, both signs on axis 3)
    sh = qdp.qdp_field_alloc(lat, 2, _prec_id(prec))
    for mu, sign in ((0, 1), (1, -1), (2, 1), (3, 1), (3, -1)):
        qdp.qdp_shift(sh, psi, mu, sign)
        assert np.array_equal(qdp.field_to_host(sh), oracle.shift(dims, hp, mu, sign)), (mu, sign)
    assert V == qdp.qdp_lattice_volume(lat)


def test_c4_bench_configuration_fp64(qdp):
    """BASELINE.json:configs[3] (the configuration bench.py times): plaquette, 20 APE steps,
    hop on red/black alternately, global sums."""
    _check_step(qdp, synth.CONFIGS["C4"], "f64", synth.BASE_SEED + 3, n_ape_steps=20)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_c3_sweep_and_normalised_iteration(qdp, prec):
    """BASELINE.json:configs[2]: chi = a psi + b hop(psi), norm2 after every step, 50 iterations
    (A14/A15: normalised, the 1/sqrt(n_k) folded into the scalars).  The field and the recorded n_k are
    compared with the oracle on the whole lattice at every step of the first spinor in fp64 and at a spread of
    steps otherwise (each time from the device field of the step before), the rest by the norm bound."""
    dims = synth.CONFIGS["C3"]
    seed = synth.BASE_SEED + 2
    _check_step(qdp, dims, prec, seed, warm=True)
    lat = qdp.qdp_lattice_create(dims)
    hu = synth.round_to(synth.gauge_hot(dims, seed), prec)
    a, b = synth.scalars_ab(seed)
    u = qdp.field_from_host(lat, 1, hu)
    u64 = _as64(hu)
    for ispinor in range(1, 5):          # reading A14: four independent spinor fields, the same (a, b)
        hp = synth.round_to(synth.spinor(dims, seed, ispinor), prec)
        bufs = [qdp.field_from_host(lat, 2, hp), qdp.qdp_field_alloc(lat, 2, _prec_id(prec))]
        # steps whose field and recorded n_k are compared with the oracle (about 1.2 s of oracle time each): the whole
        # 50-step sequence for the first spinor in fp64, a spread of it otherwise
        if ispinor == 1:
            checked = set(range(50)) if prec == "f64" else {0, 1, 2, 9, 19, 29, 39, 49}
        else:
            checked = {0, 49}
        scale = 1.0
        norms = []
        for k in range(50):
            ak, bk = a * scale, b * scale
            if prec == "f32":
                ak, bk = float(np.float32(ak)), float(np.float32(bk))
            n_k = qdp.qdp_axpy_hop(bufs[1], ak, bk, u, bufs[0], 0, want_norm2=True)
            bufs.reverse()
            norms.append(n_k)
            if k in checked:
                ref = oracle.axpy_hop(dims, ak, bk, u64, _as64(qdp.field_to_host(bufs[1])))   # from the device field of the step before: per-step error, no drift
                got = _as64(qdp.field_to_host(bufs[0]))
                assert site_rel_err(got, ref).max() <= TOL_SITE[prec], (ispinor, k)
                assert abs(n_k - oracle.norm2(dims, ref)) <= TOL_SUM[prec] * n_k, (ispinor, k)
            scale = 1.0 / np.sqrt(n_k)
        norms = np.array(norms)
        assert np.all(np.isfinite(norms)) and np.all(norms > 0)
        # after the first step psi has unit norm: n_k <= (|a| + 8 |b|)^2 (||hop|| <= 8)
        assert np.all(norms[1:] <= (abs(a) + 8 * abs(b)) ** 2 * (1 + 1e-6))
        for f in bufs:
            qdp.qdp_field_free(f)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_c5_full_sweep(qdp, prec):
    """BASELINE.json:configs[4]: 48^3x96, one sweep of plaquette, APE step, hop and norm2."""
    _check_step(qdp, synth.CONFIGS["C5"], prec, synth.BASE_SEED + 4)
