"""Pins for the oracle's global sums (SURVEY.md 8(c) definition 6, A12).
math.fsum is an exactly rounded sum: the compensated oracle must agree to ~1 ulp."""
import math

import numpy as np

import oracle
import synth
from npref import parity


def test_against_exact_summation():
    dims = (4, 2, 6, 4)
    a, b = synth.spinor(dims, 201), synth.spinor(dims, 202, 1)
    par = parity(dims)
    for sub, sel in ((0, par >= 0), (1, par == 0), (2, par == 1)):
        fa, fb = a[sel].ravel(), b[sel].ravel()
        n2 = math.fsum((fa.real ** 2).tolist() + (fa.imag ** 2).tolist())
        assert abs(oracle.norm2(dims, a, sub) - n2) <= 2e-16 * n2
        prod = np.conj(fa) * fb
        ip = complex(math.fsum(prod.real.tolist()), math.fsum(prod.imag.tolist()))
        assert abs(oracle.inner(dims, a, b, sub) - ip) <= 1e-13
        s = oracle.sum_field(dims, a, sub)
        want = np.array([complex(math.fsum(a[sel][:, i, j].real.tolist()),
                                 math.fsum(a[sel][:, i, j].imag.tolist()))
                         for i in range(4) for j in range(3)])
        assert np.abs(s - want).max() < 1e-13


def test_identities():
    dims = (4, 4, 4, 4)
    V = synth.volume(dims)
    a, b = synth.spinor(dims, 211), synth.spinor(dims, 212, 1)
    assert abs(oracle.inner(dims, a, a).real - oracle.norm2(dims, a)) < 1e-10
    assert abs(oracle.inner(dims, a, a).imag) < 1e-12
    assert abs(oracle.inner(dims, 1j * a, b) + 1j * oracle.inner(dims, a, b)) < 1e-12   # conj on FIRST
    assert abs(oracle.inner(dims, a, b)) ** 2 <= oracle.norm2(dims, a) * oracle.norm2(dims, b)
    assert abs(oracle.norm2(dims, a, 1) + oracle.norm2(dims, a, 2) - oracle.norm2(dims, a)) < 1e-10
    c = np.full((V, 4, 3), 0.5 - 0.25j)
    assert oracle.norm2(dims, c) == (0.25 + 0.0625) * 12 * V
    assert np.array_equal(oracle.sum_field(dims, c), np.full(12, (0.5 - 0.25j) * V))
    m = synth.color_matrix(dims, 213)
    assert abs(oracle.norm2(dims, m) - (np.abs(m) ** 2).sum()) < 1e-9
