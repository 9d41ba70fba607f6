"""Pins for the oracle's axpby (dst = a x + b y; the residual / solution-reconstruction expressions
of PAPER.md:96)."""
import numpy as np

import oracle
import synth
from npref import parity


def test_numpy_definition_subsets_and_kinds():
    dims = (4, 2, 6, 4)
    odd = parity(dims) == 1
    for gen in (synth.spinor, synth.color_matrix, synth.gauge_hot):
        x, y = gen(dims, 601), gen(dims, 602)
        a, b = 0.37, -1.25
        want = a * x + b * y                      # same two roundings per term
        assert np.array_equal(oracle.axpby(dims, a, x, b, y), want)
        sentinel = np.full_like(x, 9.0)
        e = oracle.axpby(dims, a, x, b, y, 1, dst=sentinel)
        assert np.array_equal(e[~odd], want[~odd]) and np.all(e[odd] == 9.0)


def test_algebra():
    dims = (2, 2, 2, 4)
    x, y = synth.spinor(dims, 603), synth.spinor(dims, 604, 1)
    assert np.array_equal(oracle.axpby(dims, 1.0, x, 0.0, y), x)
    assert np.array_equal(oracle.axpby(dims, 0.0, x, 1.0, y), y)
    assert np.array_equal(oracle.axpby(dims, 2.0, x, -2.0, x), np.zeros_like(x))
    r = oracle.axpby(dims, 1.0, y, -0.5, x)                       # residual form r = y - alpha x
    back = oracle.axpby(dims, 1.0, r, 0.5, x)
    assert np.abs(back - y).max() < 1e-15
    n = oracle.norm2(dims, oracle.axpby(dims, 3.0, x, 4.0, x))
    assert abs(n - 49.0 * oracle.norm2(dims, x)) < 1e-12 * n
