"""The seeded generators give the distributions BASELINE.json:configs names (A20)."""
import numpy as np

import synth
from npref import dag


def test_hot_links_are_su3_and_haar_like():
    u = synth.gauge_hot((8, 8, 8, 8), 7).reshape(-1, 3, 3)
    eye = np.eye(3)
    assert np.abs(u @ dag(u) - eye).max() < 1e-12   # Gram-Schmidt conditioning
    assert np.abs(np.linalg.det(u) - 1).max() < 1e-12
    tr = np.trace(u, axis1=1, axis2=2)
    n = len(tr)
    assert abs(tr.mean()) < 5 / np.sqrt(n)
    assert abs((np.abs(tr) ** 2).mean() - 1.0) < 0.03


def test_warm_links():
    u = synth.gauge_warm((8, 8, 8, 8), 7, 0.2).reshape(-1, 3, 3)
    assert np.abs(u @ dag(u) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(u) - 1).max() < 1e-12
    c = np.trace(u, axis1=1, axis2=2).real.mean() / 3
    assert abs(c - 0.9475) < 0.003


def test_spinor_moments_and_determinism():
    a = synth.spinor((4, 4, 4, 4), 3)
    b = synth.spinor((4, 4, 4, 4), 3)
    c = synth.spinor((4, 4, 4, 4), 4)
    assert np.array_equal(a, b) and not np.array_equal(a, c)
    big = synth.spinor((8, 8, 8, 8), 1)
    assert abs(big.real.mean()) < 0.02 and abs(big.real.var() - 1) < 0.03
    assert abs(big.imag.var() - 1) < 0.03
    # prefix property: values depend on the counter only, not on the volume
    small = synth.spinor((4, 4, 4, 4), 1)
    assert np.array_equal(big[: small.shape[0]], small)


def test_scalars_in_range():
    a, b = synth.scalars_ab(synth.BASE_SEED + 2)
    assert -1 < a < 1 and -1 < b < 1 and a != b
