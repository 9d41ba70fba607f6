"""Pins for the oracle's staple sum, APE blend and SU(3) projection
(SURVEY.md 8(c) definitions 3-4, readings A6-A10)."""
import numpy as np
import pytest
import scipy.linalg

import oracle
import synth
from npref import dag, gauge_transform, parity, plaquette_np, sh, staple_np

EYE = np.eye(3)


def test_projection_matches_scipy_polar_and_newton():
    rng = np.random.default_rng(11)
    for _ in range(50):
        V = rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3))
        W = oracle.polar_unitary(V)
        Wsp, _ = scipy.linalg.polar(V)              # library routine (SVD based)
        assert np.abs(W - Wsp).max() < 1e-13
        X = V.copy()                                # Newton X <- (X + X^{-dag})/2
        for _ in range(60):
            X = 0.5 * (X + np.linalg.inv(dag(X)))
        assert np.abs(W - X).max() < 1e-12
        theta = np.angle(np.linalg.det(V))
        assert np.abs(oracle.proj_su3(V) - Wsp * np.exp(-1j * theta / 3)).max() < 1e-13


def test_projection_is_special_unitary_and_variational():
    rng = np.random.default_rng(12)
    for _ in range(50):
        V = EYE * 0.5 + 0.4 * (rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3)))
        U = oracle.proj_su3(V)
        assert np.abs(U @ dag(U) - EYE).max() < 1e-12
        assert abs(np.linalg.det(U) - 1) < 1e-12
        W = oracle.polar_unitary(V)
        sv = np.linalg.svd(V, compute_uv=False)
        assert abs(np.trace(W @ dag(V)).real - sv.sum()) < 1e-13     # maximises Re tr(X V^dag)
        X = synth.su3_site_field((2, 2, 2, 2), 99)[:4]
        assert all(np.trace(x @ dag(V)).real <= sv.sum() + 1e-13 for x in X)
        assert abs(oracle.min_eig_vdv(V) - sv.min() ** 2) < 1e-13


def test_projection_of_su3_is_identity_and_degenerate_cases():
    for U in synth.su3_site_field((2, 2, 2, 2), 5):
        assert np.abs(oracle.proj_su3(U) - U).max() < 2e-15
    # positive multiples of SU(3) (fully degenerate V^dag V) and diagonal input
    U = synth.su3_site_field((2, 2, 2, 2), 6)[0]
    assert np.abs(oracle.proj_su3(3.7 * U) - U).max() < 2e-15
    z = np.array([0.3 * np.exp(0.4j), 1.1 * np.exp(-1.0j), 2.0 * np.exp(2.2j)])
    theta = np.angle(np.prod(z))
    want = np.diag(z / np.abs(z) * np.exp(-1j * theta / 3))
    assert np.abs(oracle.proj_su3(np.diag(z)) - want).max() < 2e-15


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4)])
@pytest.mark.parametrize("t_dir", [3, -1])
def test_unit_field_is_a_fixed_point(dims, t_dir):
    u = synth.gauge_unit(dims)
    out = oracle.ape_smear_step(dims, u, 0.5, t_dir)
    assert np.array_equal(out, u)
    assert np.array_equal(oracle.plaquette(dims, out), [1.0, 1.0, 1.0])


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4)])
@pytest.mark.parametrize("t_dir", [3, -1])
def test_staples_brute_force_numpy(dims, t_dir):
    """On 2^4, x+nu == x-nu: upper and lower staple neighbours coincide (H5)."""
    u = synth.gauge_hot(dims, 51)
    V = synth.volume(dims)
    dirs = [0, 1, 2] if t_dir == 3 else [0, 1, 2, 3]
    for mu in dirs:
        S = staple_np(dims, u, mu, dirs)
        for lex in range(0, V, 5):
            got, n = oracle.staple_site(dims, u, lex, mu, t_dir)
            assert n == 2 * (len(dirs) - 1)
            assert np.abs(got - S[lex]).max() < 1e-13
            Vb = oracle.ape_blend_site(dims, u, lex, mu, 0.3, t_dir)
            assert np.abs(Vb - (0.7 * u[lex, mu] + 0.3 / n * S[lex])).max() < 1e-13


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
def test_alpha_zero_identity_unitarity_and_time_links(dims):
    u = synth.gauge_hot(dims, 61)
    same = oracle.ape_smear_step(dims, u, 0.0, 3)
    assert np.abs(same - u).max() < 1e-14
    out = oracle.ape_smear_step(dims, u, 0.5, 3)
    assert np.array_equal(out[:, 3], u[:, 3])                       # A7: bit-exact copy
    m = out.reshape(-1, 3, 3)
    assert np.abs(m @ dag(m) - EYE).max() < 1e-12                   # north_star: 1e-12
    assert np.abs(np.linalg.det(m) - 1).max() < 1e-12
    out4 = oracle.ape_smear_step(dims, u, 0.5, -1)
    assert np.abs(out4[:, 3] - u[:, 3]).max() > 0.1                 # 4D smears time links too


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
@pytest.mark.parametrize("t_dir", [3, -1])
def test_gauge_covariance(dims, t_dir):
    u = synth.gauge_hot(dims, 71)
    g = synth.su3_site_field(dims, 72)
    a = oracle.ape_smear_step(dims, gauge_transform(dims, u, g), 0.5, t_dir)
    b = gauge_transform(dims, oracle.ape_smear_step(dims, u, 0.5, t_dir), g)
    assert np.abs(a - b).max() < 1e-13
    assert np.abs(oracle.plaquette(dims, a) - oracle.plaquette(dims, b)).max() < 1e-14


def test_abelian_closed_form():
    """Diagonal links give diagonal V with entries z_k; Proj -> z_k/|z_k| e^{-i theta/3}."""
    dims = (4, 2, 6, 4)
    rng = np.random.default_rng(5)
    V = synth.volume(dims)
    ph = rng.uniform(-0.6, 0.6, size=(V, 4, 3))
    u = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    for k in range(3):
        u[:, :, k, k] = np.exp(1j * ph[:, :, k])
    out = oracle.ape_smear_step(dims, u, 0.5, 3)
    d = np.exp(1j * ph)                                              # [V,4,3] scalars
    for mu in range(3):
        st = np.zeros((V, 3), dtype=np.complex128)
        for nu in range(3):
            if nu == mu:
                continue
            st += d[:, nu] * sh(dims, d[:, mu], nu) * np.conj(sh(dims, d[:, nu], mu))
            low = np.conj(d[:, nu]) * d[:, mu] * sh(dims, d[:, nu], mu)
            st += sh(dims, low, nu, -1)
        z = 0.5 * d[:, mu] + 0.5 / 4 * st
        theta = np.angle(z.prod(axis=1))
        want = z / np.abs(z) * np.exp(-1j * theta / 3)[:, None]
        got = np.stack([out[:, mu, k, k] for k in range(3)], axis=1)
        assert np.abs(got - want).max() < 1e-14
        offd = out[:, mu].copy()
        for k in range(3):
            offd[:, k, k] = 0
        assert np.abs(offd).max() < 1e-15


def test_subset_writes_only_its_sites():
    dims = (4, 4, 4, 4)
    u = synth.gauge_hot(dims, 81)
    par = parity(dims)
    full = oracle.ape_smear_step(dims, u, 0.5, 3)
    sentinel = np.full_like(u, 9.0)
    ev = oracle.ape_smear_step(dims, u, 0.5, 3, oracle.EVEN, u_out=sentinel)
    assert np.array_equal(ev[par == 0], full[par == 0])
    assert np.array_equal(ev[par == 1], sentinel[par == 1])
    both = oracle.ape_smear_step(dims, u, 0.5, 3, oracle.ODD, u_out=ev)
    assert np.array_equal(both, full)


def test_plaquette_rises_under_smearing():
    dims = (8, 8, 8, 8)
    u = synth.gauge_warm(dims, 91, 0.2)
    p = [oracle.plaquette(dims, u)[1]]
    for _ in range(3):
        u = oracle.ape_smear_step(dims, u, 0.5, 3)
        p.append(oracle.plaquette(dims, u)[1])
    assert all(b > a for a, b in zip(p, p[1:])) and p[-1] > 0.95
