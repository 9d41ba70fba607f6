"""Pins for the oracle's spin matrices and the gamma-inserted time-slice contraction (row f3)."""
import numpy as np
import pytest

import oracle
import synth
from npref import view4


# The four Euclidean gamma matrices of the DeGrand-Rossi basis (QDP++'s convention), typed in as numbers from the
# statement of the convention in include/qdp_b200.h (qdp_inner_timeslices_gamma); rows = s', columns = s.
# The Clifford/Hermiticity pins below hold in every Hermitian representation; this one fixes the basis itself
# (a sign flip of one matrix or a swap of two fails it).
I = 1j
DEGRAND_ROSSI = {
    0: [[0, 0, 0, I], [0, 0, I, 0], [0, -I, 0, 0], [-I, 0, 0, 0]],
    1: [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]],
    2: [[0, 0, I, 0], [0, 0, 0, -I], [-I, 0, 0, 0], [0, I, 0, 0]],
    3: [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]],
}
# gamma_5 = g0 g1 g2 g3 in this basis is diagonal (chiral basis): multiplied out by hand
GAMMA5_DIAG = [1, 1, -1, -1]


def test_basis_is_the_literal_degrand_rossi_matrices():
    for mu in range(4):
        assert np.array_equal(oracle.gamma_matrix(1 << mu), np.array(DEGRAND_ROSSI[mu], dtype=complex)), mu
    assert np.array_equal(oracle.gamma_matrix(15), np.diag(GAMMA5_DIAG).astype(complex))
    # a composite one: g0 g1 = diag(-i, i, -i, i)
    g01 = np.array(DEGRAND_ROSSI[0], dtype=complex) @ np.array(DEGRAND_ROSSI[1], dtype=complex)
    assert np.array_equal(oracle.gamma_matrix(3), g01)


def test_clifford_algebra_hermiticity_and_gamma5():
    g = [oracle.gamma_matrix(1 << mu) for mu in range(4)]
    eye = np.eye(4)
    for mu in range(4):
        assert np.array_equal(g[mu], np.conj(g[mu].T))                       # Hermitian
        for nu in range(4):
            assert np.array_equal(g[mu] @ g[nu] + g[nu] @ g[mu], 2 * eye * (mu == nu))
    g5 = oracle.gamma_matrix(15)
    assert np.array_equal(g5, g[0] @ g[1] @ g[2] @ g[3])
    assert np.array_equal(g5 @ g5, eye) and np.trace(g5) == 0 and np.array_equal(g5, np.conj(g5.T))
    for mu in range(4):
        assert np.array_equal(g5 @ g[mu] + g[mu] @ g5, np.zeros((4, 4)))
    assert np.array_equal(oracle.gamma_matrix(0), eye)
    # every Gamma(n) is a signed/phased permutation (one entry of modulus 1 per row and column): the
    # 16 of them are linearly independent (a basis of the 4x4 matrices)
    basis = np.stack([oracle.gamma_matrix(n).ravel() for n in range(16)])
    assert np.linalg.matrix_rank(basis) == 16
    for n in range(16):
        G = oracle.gamma_matrix(n)
        assert np.array_equal((np.abs(G) == 1).sum(axis=0), np.ones(4)) and np.abs(G).sum() == 4
        assert n == sum(((n >> mu) & 1) << mu for mu in range(4))
        want = eye.astype(complex)
        for mu in range(4):
            if (n >> mu) & 1:
                want = want @ g[mu]
        assert np.array_equal(G, want)


@pytest.mark.parametrize("dims", [(2, 2, 2, 4), (4, 2, 6, 4)])
def test_contraction_brute_force_and_identities(dims):
    a, b = synth.spinor(dims, 701), synth.spinor(dims, 702, 1)
    scale = oracle.norm2(dims, a) + oracle.norm2(dims, b)
    for n in (0, 1, 6, 8, 15, 11):
        G = oracle.gamma_matrix(n)
        gb = np.einsum("ts,xsc->xtc", G, b)
        want = view4(dims, np.conj(a) * gb).reshape(dims[3], -1).sum(axis=1)
        got = oracle.inner_timeslices_gamma(dims, a, b, n)
        assert np.abs(got - want).max() < 1e-13 * scale
        # <a, G b> = conj(<b, G^dag a>), G^dag = +-G
        sign = 1.0 if np.array_equal(G, np.conj(G.T)) else -1.0
        assert np.array_equal(np.conj(G.T), sign * G)
        back = oracle.inner_timeslices_gamma(dims, b, a, n)
        assert np.abs(got - sign * np.conj(back)).max() < 1e-13 * scale
    assert np.abs(oracle.inner_timeslices_gamma(dims, a, b, 0) - oracle.inner_timeslices(dims, a, b)).max() < 1e-13 * scale
    e, o = oracle.inner_timeslices_gamma(dims, a, b, 15, 1), oracle.inner_timeslices_gamma(dims, a, b, 15, 2)
    assert np.abs(e + o - oracle.inner_timeslices_gamma(dims, a, b, 15)).max() < 1e-13 * scale
