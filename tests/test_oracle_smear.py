"""Pins for the oracle's quark-smearing step (the SRC/SNK smearing stage of
PAPER.md:82, 106):  chi = a psi + b sum_{mu != t_dir} [U_mu(x) psi(x+mu) + U_mu(x-mu)^dag psi(x-mu)]."""
import numpy as np
import pytest

import oracle
import synth
from npref import coords, gauge_transform, parity, sh


def _hop_dirs_np(dims, u, psi, dirs):
    chi = np.zeros_like(psi)
    for mu in dirs:
        chi += np.einsum("xab,xsb->xsa", u[:, mu], sh(dims, psi, mu))
        back = np.einsum("xba,xsb->xsa", np.conj(u[:, mu]), psi)   # U^dag(y) psi(y) at y
        chi += sh(dims, back, mu, -1)
    return chi


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4)])
@pytest.mark.parametrize("t_dir", [3, -1])
def test_brute_force_numpy(dims, t_dir):
    u, psi = synth.gauge_hot(dims, 201), synth.spinor(dims, 202)
    a, b = 0.4, -1.3
    dirs = [mu for mu in range(4) if mu != t_dir]
    want = a * psi + b * _hop_dirs_np(dims, u, psi, dirs)
    assert np.abs(oracle.smear_hop(dims, a, b, u, psi, t_dir) - want).max() < 1e-13
    assert np.abs(oracle.hop_site_dirs(dims, u, psi, 5, t_dir) - _hop_dirs_np(dims, u, psi, dirs)[5]).max() < 1e-13


def test_all_directions_is_axpy_hop_bit_exactly():
    dims = (4, 2, 6, 4)
    u, psi = synth.gauge_hot(dims, 203), synth.spinor(dims, 204)
    for sub in (0, 1, 2):
        assert np.array_equal(oracle.smear_hop(dims, 0.3, 0.9, u, psi, -1, sub, chi=psi),
                              oracle.axpy_hop(dims, 0.3, 0.9, u, psi, sub, chi=psi))


def test_plane_wave_on_unit_field_closed_form():
    """chi = (a + b sum_{mu<3} 2 cos(2 pi k_mu / L_mu)) psi: the time component of k does not enter."""
    dims, k = (4, 8, 4, 6), np.array([1, 1, 0, 2])
    x = coords(dims)
    phase = np.exp(2j * np.pi * (x * k / np.array(dims)).sum(axis=1))
    v = np.arange(1, 13).reshape(4, 3) * (1 - 0.25j)
    psi = phase[:, None, None] * v[None]
    a, b = 0.7, 0.2
    lam = a + b * (2 * np.cos(2 * np.pi * k[:3] / np.array(dims)[:3])).sum()
    assert abs(lam - (0.7 + 0.2 * (0.0 + np.sqrt(2) + 2.0))) < 1e-15
    chi = oracle.smear_hop(dims, a, b, synth.gauge_unit(dims), psi, 3)
    assert np.abs(chi - lam * psi).max() < 1e-13


def test_time_slices_do_not_mix():
    """Spatial smearing never couples time-slices: a source on x3 = t0 stays on x3 = t0, exactly."""
    dims, t0 = (4, 4, 4, 6), 2
    u, psi = synth.gauge_hot(dims, 205), synth.spinor(dims, 206)
    on = coords(dims)[:, 3] == t0
    psi[~on] = 0
    chi = psi
    for _ in range(3):
        chi = oracle.smear_hop(dims, 1.0, 0.25, u, chi, 3)
    assert np.all(chi[~on] == 0)
    assert np.abs(chi[on]).min() > 0          # three steps reach every site of a 4^3 slice
    full = oracle.smear_hop(dims, 1.0, 0.25, u, psi, -1)
    assert np.abs(full[~on]).max() > 0        # whereas the four-direction hop does leave the slice


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
def test_gauge_covariance_hermiticity_and_bound(dims):
    u, psi, phi = synth.gauge_hot(dims, 211), synth.spinor(dims, 212), synth.spinor(dims, 213, 1)
    g = synth.su3_site_field(dims, 214)
    gpsi = np.einsum("xab,xsb->xsa", g, psi)
    lhs = oracle.smear_hop(dims, 0.5, 0.3, gauge_transform(dims, u, g), gpsi, 3)
    rhs = np.einsum("xab,xsb->xsa", g, oracle.smear_hop(dims, 0.5, 0.3, u, psi, 3))
    assert np.abs(lhs - rhs).max() < 1e-13
    h_psi, h_phi = oracle.smear_hop(dims, 0.0, 1.0, u, psi, 3), oracle.smear_hop(dims, 0.0, 1.0, u, phi, 3)
    ip1, ip2 = oracle.inner(dims, phi, h_psi), oracle.inner(dims, psi, h_phi)
    n2 = oracle.norm2(dims, psi)
    assert abs(ip1 - np.conj(ip2)) < 1e-12 * n2                   # Hermitian
    assert abs(oracle.inner(dims, psi, h_psi).imag) < 1e-12 * n2
    assert oracle.norm2(dims, h_psi) <= 36 * n2 * (1 + 1e-12)     # ||spatial hop|| <= 6


def test_subsets_and_parity_structure():
    dims = (4, 4, 2, 4)
    u, psi = synth.gauge_hot(dims, 221), synth.spinor(dims, 222)
    sentinel = synth.spinor(dims, 223, 1)
    full = oracle.smear_hop(dims, 0.2, 0.8, u, psi, 3)
    odd = parity(dims) == 1
    for sub, mask in ((1, ~odd), (2, odd)):
        out = oracle.smear_hop(dims, 0.2, 0.8, u, psi, 3, sub, chi=sentinel)
        assert np.array_equal(out[mask], full[mask]) and np.array_equal(out[~mask], sentinel[~mask])
    psi_e = psi.copy()
    psi_e[odd] = 0
    assert np.all(oracle.smear_hop(dims, 0.0, 1.0, u, psi_e, 3)[~odd] == 0)   # hops change parity
