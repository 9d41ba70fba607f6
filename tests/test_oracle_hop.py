"""Pins for the oracle's hop and axpy_hop (SURVEY.md 8(c) definitions 5-6, A11)."""
import numpy as np
import pytest

import oracle
import synth
from npref import coords, gauge_transform, hop_np, parity, sh


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4)])
def test_brute_force_numpy(dims):
    u, psi = synth.gauge_hot(dims, 101), synth.spinor(dims, 102)
    want = hop_np(dims, u, psi)
    assert np.abs(oracle.hop(dims, u, psi) - want).max() < 1e-13
    assert np.abs(oracle.hop_site(dims, u, psi, 3) - want[3]).max() < 1e-13


def test_plane_wave_on_unit_field():
    """chi = (sum_mu 2 cos(2 pi k_mu / L_mu)) psi; L=(4,4,4,8), k=(1,0,0,1): 5.41421356..."""
    dims, k = (4, 4, 4, 8), np.array([1, 0, 0, 1])
    x = coords(dims)
    phase = np.exp(2j * np.pi * (x * k / np.array(dims)).sum(axis=1))
    v = np.arange(1, 13).reshape(4, 3) * (1 + 0.5j)
    psi = phase[:, None, None] * v[None]
    chi = oracle.hop(dims, synth.gauge_unit(dims), psi)
    lam = (2 * np.cos(2 * np.pi * k / np.array(dims))).sum()
    assert abs(lam - (4 + np.sqrt(2))) < 1e-15
    assert np.abs(chi - lam * psi).max() < 1e-13
    chi0 = oracle.hop(dims, synth.gauge_unit(dims), np.ones_like(psi))
    assert np.array_equal(chi0, 8 * np.ones_like(psi))              # k = 0


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
def test_gauge_covariance_and_hermiticity(dims):
    u, psi, phi = synth.gauge_hot(dims, 111), synth.spinor(dims, 112), synth.spinor(dims, 113, 1)
    g = synth.su3_site_field(dims, 114)
    gpsi = np.einsum("xab,xsb->xsa", g, psi)
    lhs = oracle.hop(dims, gauge_transform(dims, u, g), gpsi)
    rhs = np.einsum("xab,xsb->xsa", g, oracle.hop(dims, u, psi))
    assert np.abs(lhs - rhs).max() < 1e-13
    assert abs(oracle.norm2(dims, lhs) / oracle.norm2(dims, rhs) - 1) < 1e-14
    hp, hph = oracle.hop(dims, u, psi), oracle.hop(dims, u, phi)
    ip = oracle.inner(dims, psi, hp)
    n2 = oracle.norm2(dims, psi)
    assert abs(ip.imag) < 1e-13 * 8 * n2 and abs(ip) <= 8 * n2
    assert abs(oracle.inner(dims, phi, hp) - np.conj(oracle.inner(dims, psi, hph))) < 1e-12 * 8 * n2


def test_parity_structure_and_subsets():
    dims = (4, 2, 6, 4)
    u, psi = synth.gauge_hot(dims, 121), synth.spinor(dims, 122)
    par = parity(dims)
    pe = psi.copy()
    pe[par == 1] = 0
    chi = oracle.hop(dims, u, pe)
    assert np.array_equal(chi[par == 0], np.zeros_like(chi[par == 0]))
    full = oracle.hop(dims, u, psi)
    sentinel = np.full_like(psi, 5.0 - 2.0j)
    ev = oracle.hop(dims, u, psi, oracle.EVEN, chi=sentinel)
    assert np.array_equal(ev[par == 0], full[par == 0])
    assert np.array_equal(ev[par == 1], sentinel[par == 1])
    assert np.array_equal(oracle.hop(dims, u, psi, oracle.ODD, chi=ev), full)     # A17


def test_haar_links_norm_ratio():
    dims = (8, 8, 8, 8)
    u, psi = synth.gauge_hot(dims, 131), synth.spinor(dims, 132)
    r = oracle.norm2(dims, oracle.hop(dims, u, psi)) / oracle.norm2(dims, psi)
    assert 7.8 < r < 8.2


def test_axpy_hop():
    dims = (4, 4, 4, 4)
    u, psi, phi = synth.gauge_hot(dims, 141), synth.spinor(dims, 142), synth.spinor(dims, 143, 1)
    a, b = synth.scalars_ab(144)
    assert np.array_equal(oracle.axpy_hop(dims, a, 0.0, u, psi), a * psi)
    assert np.array_equal(oracle.axpy_hop(dims, 0.0, 1.0, u, psi), oracle.hop(dims, u, psi))
    want = a * psi + b * hop_np(dims, u, psi)
    assert np.abs(oracle.axpy_hop(dims, a, b, u, psi) - want).max() < 1e-13
    lin = oracle.axpy_hop(dims, a, b, u, psi + 2 * phi)
    assert np.abs(lin - (oracle.axpy_hop(dims, a, b, u, psi)
                         + 2 * oracle.axpy_hop(dims, a, b, u, phi))).max() < 1e-12
