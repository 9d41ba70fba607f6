"""Pins for the oracle's plaquette (SURVEY.md 8(c) definition 2, readings A4, A5)."""
import numpy as np
import pytest

import oracle
import synth
from npref import coords, gauge_transform, parity, plaquette_np, sh

PLANES = [(0, 1), (0, 2), (1, 2), (0, 3), (1, 3), (2, 3)]


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4)])
def test_unit_field_is_exactly_one(dims):
    for sub in (oracle.ALL, oracle.EVEN, oracle.ODD):
        assert np.array_equal(oracle.plaquette(dims, synth.gauge_unit(dims), sub), [1.0, 1.0, 1.0])


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4)])
def test_gauge_invariance(dims):
    u = synth.gauge_hot(dims, 21)
    g = synth.su3_site_field(dims, 22)
    ug = gauge_transform(dims, u, g)
    for sub in (oracle.ALL, oracle.EVEN, oracle.ODD):
        assert np.abs(oracle.plaquette(dims, u, sub) - oracle.plaquette(dims, ug, sub)).max() < 1e-14


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
def test_abelian_closed_form(dims):
    """U_mu(x) = diag(e^{i phi}, e^{-i phi}, 1): Re tr P = 2 cos F + 1 with
    F = phi_mu(x) + phi_nu(x+mu) - phi_mu(x+nu) - phi_nu(x), from scalars only."""
    rng = np.random.default_rng(3)
    V = synth.volume(dims)
    phi = rng.uniform(-np.pi, np.pi, size=(V, 4))
    u = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    u[:, :, 0, 0] = np.exp(1j * phi)
    u[:, :, 1, 1] = np.exp(-1j * phi)
    u[:, :, 2, 2] = 1.0
    sp = tp = 0.0
    for (mu, nu) in PLANES:
        F = phi[:, mu] + sh(dims, phi[:, nu], mu) - sh(dims, phi[:, mu], nu) - phi[:, nu]
        val = (2 * np.cos(F) + 1).sum()
        if nu == 3:
            tp += val
        else:
            sp += val
    want = np.array([(sp + tp) / (18 * V), sp / (9 * V), tp / (9 * V)])
    assert np.abs(oracle.plaquette(dims, u) - want).max() < 1e-14
    # per-site values, per plane
    for lex in (0, 5, V - 1):
        got = oracle.plaquette_site(dims, u, lex)
        for k, (mu, nu) in enumerate(PLANES):
            F = phi[:, mu] + sh(dims, phi[:, nu], mu) - sh(dims, phi[:, mu], nu) - phi[:, nu]
            assert abs(got[k] - (2 * np.cos(F[lex]) + 1)) < 1e-14


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4)])
def test_brute_force_numpy(dims):
    u = synth.gauge_hot(dims, 31)
    V = synth.volume(dims)
    par = parity(dims)
    per_plane = np.stack([plaquette_np(dims, u, mu, nu) for (mu, nu) in PLANES], axis=1)
    for sub, sel in ((oracle.ALL, np.ones(V, bool)), (oracle.EVEN, par == 0), (oracle.ODD, par == 1)):
        n = sel.sum()
        sp, tp = per_plane[sel, :3].sum(), per_plane[sel, 3:].sum()
        want = np.array([(sp + tp) / (18 * n), sp / (9 * n), tp / (9 * n)])
        assert np.abs(oracle.plaquette(dims, u, sub) - want).max() < 1e-14
    for lex in range(0, V, 7):
        assert np.abs(oracle.plaquette_site(dims, u, lex) - per_plane[lex]).max() < 1e-14


def test_even_plus_odd_is_all_and_statistics():
    dims = (8, 8, 8, 8)
    V = synth.volume(dims)
    u = synth.gauge_hot(dims, 41)
    pa, pe, po = (oracle.plaquette(dims, u, s) for s in (oracle.ALL, oracle.EVEN, oracle.ODD))
    assert np.abs(pa - 0.5 * (pe + po)).max() < 1e-14
    # Haar links: plaquette 0 +- sqrt(0.5)/(3 sqrt(6V))  (SURVEY.md 8(c) pins)
    assert abs(pa[0]) < 5 * np.sqrt(0.5) / (3 * np.sqrt(6 * V))
    # warm eps=0.2 field: about c^4 = 0.806 (measured 0.804 on 8^4, Appendix D)
    pw = oracle.plaquette(dims, synth.gauge_warm(dims, 41, 0.2))
    assert abs(pw[0] - 0.805) < 0.01
