"""Pins for the oracle's geometry and shift (SURVEY.md 8(c) definition 1, readings A1-A4).

Closed forms: a field filled with its own coordinates must come back as
(x +- mu_hat) mod L; tables must equal np.roll of the site numbering; masks
must equal the coordinate sum; anisotropic dims catch axis mix-ups.
"""
import numpy as np
import pytest

import oracle
import synth
from npref import coords, parity, sh

DIMS = [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4), (6, 4, 2, 8)]


@pytest.mark.parametrize("dims", DIMS)
def test_neighbor_table_closed_form(dims):
    x = coords(dims)
    L = np.array(dims)
    strides = np.array([1, dims[0], dims[0] * dims[1], dims[0] * dims[1] * dims[2]])
    for mu in range(4):
        for sign in (+1, -1):
            y = x.copy()
            y[:, mu] = (y[:, mu] + sign) % L[mu]
            want = (y * strides).sum(axis=1).astype(np.int32)
            got = oracle.neighbor_table(dims, mu, sign)
            assert np.array_equal(got, want)
            # and as a roll of the numbering
            V = len(x)
            assert np.array_equal(got, sh(dims, np.arange(V, dtype=np.int32), mu, sign))


@pytest.mark.parametrize("dims", DIMS)
def test_parity_mask(dims):
    m = oracle.parity_mask(dims)
    assert np.array_equal(m, parity(dims).astype(np.uint8))
    assert m.sum() * 2 == len(m)            # two-colourable: all L even (A2)


@pytest.mark.parametrize("dims", DIMS)
def test_shift_of_coordinate_field(dims):
    x = coords(dims).astype(np.float64)
    L = np.array(dims)
    for mu in range(4):
        for sign in (+1, -1):
            got = oracle.shift(dims, x, mu, sign)
            want = x.copy()
            want[:, mu] = (want[:, mu] + sign) % L[mu]
            assert np.array_equal(got, want)


@pytest.mark.parametrize("dims", DIMS)
def test_shift_round_trip_and_subsets(dims):
    f = synth.spinor(dims, 5)
    par = parity(dims)
    for mu in range(4):
        fwd = oracle.shift(dims, f, mu, +1)
        assert np.array_equal(oracle.shift(dims, fwd, mu, -1), f)
        if dims[mu] == 2:
            assert np.array_equal(fwd, oracle.shift(dims, f, mu, -1))
        # subset writes only its sites; even U odd = full, bit-exact
        sentinel = np.full_like(f, 7.0 + 3.0j)
        ev = oracle.shift(dims, f, mu, +1, oracle.EVEN, dst=sentinel)
        assert np.array_equal(ev[par == 0], fwd[par == 0])
        assert np.array_equal(ev[par == 1], sentinel[par == 1])
        both = oracle.shift(dims, f, mu, +1, oracle.ODD, dst=ev)
        assert np.array_equal(both, fwd)


def test_shift_is_bit_exact_for_fp32_records():
    dims = (4, 2, 6, 4)
    f = synth.round_to(synth.color_matrix(dims, 9), "f32")
    got = oracle.shift(dims, f, 2, -1)
    assert got.dtype == np.complex64
    assert np.array_equal(got, sh(dims, f, 2, -1))
