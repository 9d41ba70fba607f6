"""Pins for the oracle's baryon building block: eps_{abc} eps_{a'b'c'} colour contraction of
three quark fields with a diquark spin matrix, per time-slice."""
import itertools

import numpy as np
import pytest

import oracle
import synth
from npref import parity, view4

EPS = np.zeros((3, 3, 3))
for (a, b, c), sgn in (((0, 1, 2), 1), ((1, 2, 0), 1), ((2, 0, 1), 1), ((0, 2, 1), -1), ((2, 1, 0), -1), ((1, 0, 2), -1)):
    EPS[a, b, c] = sgn


def _brute(dims, q1, q2, q3, n):
    """numpy einsum with the explicit Levi-Civita tensor; q*: lists of 1 or 3 fields [V,4,3]."""
    G = oracle.gamma_matrix(n)
    site = 0
    if len(q1) == 1:
        site = np.einsum("abc,xia,ij,xjb,xgc->xg", EPS, q1[0], G, q2[0], q3[0])
    else:
        Q1, Q2, Q3 = np.stack(q1), np.stack(q2), np.stack(q3)            # [source colour, V, spin, colour]
        site = np.einsum("ABC,abc,Axia,ij,Bxjb,Cxgc->xg", EPS, EPS, Q1, G, Q2, Q3)
    return view4(dims, site).reshape(dims[3], -1, 4).sum(axis=1)


@pytest.mark.parametrize("dims", [(2, 2, 2, 4), (4, 2, 6, 4)])
def test_brute_force_numpy(dims):
    f = [synth.spinor(dims, 1001, k) for k in range(9)]
    scale = sum(oracle.norm2(dims, x) for x in f) ** 1.5
    for n in (0, 5, 10, 15, 7):
        got = oracle.baryon_timeslices(dims, f[0], f[1], f[2], n)
        assert np.abs(got - _brute(dims, [f[0]], [f[1]], [f[2]], n)).max() < 1e-13 * scale
        got = oracle.baryon_timeslices(dims, f[0:3], f[3:6], f[6:9], n)
        assert np.abs(got - _brute(dims, f[0:3], f[3:6], f[6:9], n)).max() < 1e-13 * scale


def test_one_hot_closed_form():
    """q1 = e_(al,0), q2 = e_(be,1), q3 = e_(g,2) at one site: out[t][g] = Gamma_{al be} eps_{012} = Gamma_{al be};
    exchanging the colours of q1 and q2 flips the sign."""
    dims = (2, 2, 2, 4)
    V = synth.volume(dims)
    site, t = 11, 11 // 8
    for n in (5, 10, 15):
        G = oracle.gamma_matrix(n)
        for al, be, g in itertools.product(range(4), range(4), (0, 3)):
            q1, q2, q3 = (np.zeros((V, 4, 3), dtype=np.complex128) for _ in range(3))
            q1[site, al, 0], q2[site, be, 1], q3[site, g, 2] = 1, 1, 1
            out = oracle.baryon_timeslices(dims, q1, q2, q3, n)
            want = np.zeros((dims[3], 4), dtype=complex)
            want[t, g] = G[al, be]
            assert np.array_equal(out, want)
            q1[site, al, 0], q1[site, al, 1], q2[site, be, 1], q2[site, be, 0] = 0, 1, 0, 1
            assert np.array_equal(oracle.baryon_timeslices(dims, q1, q2, q3, n), -want)


def test_colour_singlet_invariance_and_diquark_symmetry():
    dims = (4, 2, 2, 4)
    f = [synth.spinor(dims, 1002, k) for k in range(9)]
    scale = sum(oracle.norm2(dims, x) for x in f) ** 1.5
    g = synth.su3_site_field(dims, 1003)                       # one SU(3) matrix per site
    rot = lambda q: np.einsum("xab,xsb->xsa", g, q)
    for n in (5, 10):
        base = oracle.baryon_timeslices(dims, f[0], f[1], f[2], n)
        # a site-local SU(3) rotation of all three quarks leaves eps_{abc} q q q invariant (det g = 1): gauge invariance
        assert np.abs(oracle.baryon_timeslices(dims, rot(f[0]), rot(f[1]), rot(f[2]), n) - base).max() < 1e-12 * scale
        # a U(3) phase multiplies it by det = e^{3 i phi}
        ph = np.exp(0.3j)
        assert np.abs(oracle.baryon_timeslices(dims, ph * f[0], ph * f[1], ph * f[2], n) - ph ** 3 * base).max() < 1e-12 * scale
        # exchanging the two diquark quarks: eps_{abc} q1_a G q2_b = -eps_{abc} q2_a G^T q1_b; Gamma(n)^T = +-Gamma(n)
        G = oracle.gamma_matrix(n)
        sign = 1.0 if np.array_equal(G.T, G) else -1.0
        assert np.array_equal(G.T, sign * G)
        swapped = oracle.baryon_timeslices(dims, f[1], f[0], f[2], n)
        assert np.abs(swapped + sign * base).max() < 1e-12 * scale
        if sign > 0:       # identical quarks in a symmetric diquark vanish
            assert np.abs(oracle.baryon_timeslices(dims, f[0], f[0], f[2], n)).max() < 1e-12 * scale
    # the source contraction is the signed sum over the six source-colour permutations of the single-triple form
    n = 5
    full = oracle.baryon_timeslices(dims, f[0:3], f[3:6], f[6:9], n)
    acc = 0
    for (a, b, c) in itertools.permutations(range(3)):
        acc = acc + EPS[a, b, c] * oracle.baryon_timeslices(dims, f[a], f[3 + b], f[6 + c], n)
    assert np.abs(full - acc).max() < 1e-12 * scale
    # ... and is invariant under an SU(3) rotation of the source colour index
    h = synth.gauge_hot((2, 2, 2, 2), 1004)[0, 0]
    mix = lambda fs: [sum(h[a, b] * fs[b] for b in range(3)) for a in range(3)]
    assert np.abs(oracle.baryon_timeslices(dims, mix(f[0:3]), mix(f[3:6]), mix(f[6:9]), n) - full).max() < 1e-12 * scale
    # subsets: even + odd = all
    e = oracle.baryon_timeslices(dims, f[0], f[1], f[2], n, oracle.EVEN)
    o = oracle.baryon_timeslices(dims, f[0], f[1], f[2], n, oracle.ODD)
    assert np.abs(e + o - oracle.baryon_timeslices(dims, f[0], f[1], f[2], n)).max() < 1e-12 * scale
