"""Pins for the oracle's time-slice sums (HAD stage)."""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import synth
from npref import coords, parity, view4


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4), (4, 4, 2, 8)])
@pytest.mark.parametrize("kind", ["spinor", "matrix"])
def test_brute_force_numpy_and_total(dims, kind):
    gen = synth.spinor if kind == "spinor" else synth.color_matrix
    a, b = gen(dims, 301), gen(dims, 302)
    got = oracle.inner_timeslices(dims, a, b)
    prod = view4(dims, np.conj(a) * b)                                   # [L3, L2, L1, L0, ...]
    want = prod.reshape(dims[3], -1).sum(axis=1)
    assert got.shape == (dims[3],)
    assert np.abs(got - want).max() < 1e-12 * np.abs(want).max()
    assert abs(got.sum() - oracle.inner(dims, a, b)) < 1e-12 * abs(oracle.norm2(dims, a))
    n = oracle.inner_timeslices(dims, a, a)                              # pion-correlator form
    assert np.all(n.real > 0) and np.abs(n.imag).max() == 0
    assert abs(n.real.sum() - oracle.norm2(dims, a)) < 1e-12 * n.real.sum()
    assert np.abs(oracle.inner_timeslices(dims, b, a) - np.conj(got)).max() < 1e-13 * np.abs(want).max()


def test_exact_rational_sum_on_integer_fields():
    """Small-integer inputs: every product and partial sum is exact, so the result must equal the
    rational sum exactly."""
    dims = (4, 2, 2, 4)
    rng = np.random.default_rng(7)
    V = synth.volume(dims)
    a = (rng.integers(-8, 9, (V, 4, 3)) + 1j * rng.integers(-8, 9, (V, 4, 3))).astype(np.complex128)
    b = (rng.integers(-8, 9, (V, 4, 3)) + 1j * rng.integers(-8, 9, (V, 4, 3))).astype(np.complex128)
    got = oracle.inner_timeslices(dims, a, b)
    x3 = coords(dims)[:, 3]
    for t in range(dims[3]):
        re = sum(Fraction(int(v)) for v in (np.conj(a[x3 == t]) * b[x3 == t]).real.ravel())
        im = sum(Fraction(int(v)) for v in (np.conj(a[x3 == t]) * b[x3 == t]).imag.ravel())
        assert got[t].real == float(re) and got[t].imag == float(im)


def test_single_slice_support_subsets_and_constant_field():
    dims, t0 = (4, 4, 2, 6), 4
    a, b = synth.spinor(dims, 303), synth.spinor(dims, 304)
    x3, odd = coords(dims)[:, 3], parity(dims) == 1
    a0 = a.copy()
    a0[x3 != t0] = 0
    got = oracle.inner_timeslices(dims, a0, b)
    assert np.all(got[np.arange(dims[3]) != t0] == 0) and got[t0] != 0
    e, o, full = (oracle.inner_timeslices(dims, a, b, s) for s in (1, 2, 0))
    assert np.abs(e + o - full).max() < 1e-12 * np.abs(full).max()
    b_e = b.copy()
    b_e[odd] = 0
    assert np.abs(oracle.inner_timeslices(dims, a, b_e) - e).max() < 1e-12 * np.abs(full).max()
    ones = np.full_like(a, 2.0 - 1.0j)                                    # |c|^2 * 12 * spatial volume
    assert np.array_equal(oracle.inner_timeslices(dims, ones, ones), np.full(dims[3], 5.0 * 12 * 32 + 0j))
