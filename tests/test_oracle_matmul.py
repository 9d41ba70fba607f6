"""Pins for the oracle's binary colour-matrix expression (first step):
dst(x) = opA(A(x)) * opB(B(x + sign*mu))."""
import numpy as np
import pytest

import oracle
import synth
from npref import dag, parity, plaquette_np, sh


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4)])
def test_brute_force_numpy_all_operand_forms(dims):
    u, m = synth.gauge_hot(dims, 501), synth.color_matrix(dims, 502)
    zero = np.zeros_like(m)
    for adj_a in (0, 1):
        for adj_b in (0, 1):
            for mu, sign in ((-1, 1), (0, 1), (1, -1), (3, 1), (2, -1)):
                A = dag(u[:, 1]) if adj_a else u[:, 1]
                B = m if mu < 0 else sh(dims, m, mu, sign)
                B = dag(B) if adj_b else B
                got = oracle.matmul(dims, zero, 0, u, 1, adj_a, m, 0, adj_b, mu, sign)
                assert np.abs(got - A @ B).max() < 1e-13, (adj_a, adj_b, mu, sign)


def test_plaquette_composed_from_products_equals_the_fused_definition():
    """P_{mu nu}(x) = [U_mu(x) U_nu(x+mu)] [U_nu(x) U_mu(x+nu)]^dag built from three generic
    products reproduces def. 2 (and its numpy form) plane by plane."""
    dims = (4, 2, 6, 4)
    u = synth.gauge_hot(dims, 503)
    V = synth.volume(dims)
    z = np.zeros((V, 3, 3), dtype=np.complex128)
    total = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a = oracle.matmul(dims, z, 0, u, mu, 0, u, nu, 0, mu, +1)        # U_mu(x) U_nu(x+mu)
            b = oracle.matmul(dims, z, 0, u, nu, 0, u, mu, 0, nu, +1)        # U_nu(x) U_mu(x+nu)
            p = oracle.matmul(dims, z, 0, a, 0, 0, b, 0, 1)                  # a b^dag
            tr = np.trace(p, axis1=1, axis2=2).real
            assert np.abs(tr - plaquette_np(dims, u, mu, nu)).max() < 1e-13
            total += tr.sum()
    assert abs(total / (18 * V) - oracle.plaquette(dims, u)[0]) < 1e-13


def test_unitarity_adjoint_rule_subsets_and_gauge_slots():
    dims = (4, 4, 2, 4)
    u, m, n = synth.gauge_hot(dims, 504), synth.color_matrix(dims, 505), synth.color_matrix(dims, 506)
    V = synth.volume(dims)
    z = np.zeros((V, 3, 3), dtype=np.complex128)
    one = oracle.matmul(dims, z, 0, u, 2, 0, u, 2, 1)                        # U U^dag = 1
    assert np.abs(one - np.eye(3)).max() < 1e-14
    ab = oracle.matmul(dims, z, 0, m, 0, 0, n, 0, 0, 1, 1)
    ba = oracle.matmul(dims, z, 0, sh(dims, n, 1, 1), 0, 1, m, 0, 1)         # (A B)^dag = B^dag A^dag
    assert np.abs(dag(ab) - ba).max() < 1e-13
    odd = parity(dims) == 1
    sentinel = np.full_like(u, 5.0)
    out = oracle.matmul(dims, sentinel, 3, m, 0, 0, n, 0, 0, -1, 1, 2)       # into link 3 of a gauge field, odd sites
    assert np.all(out[:, :3] == 5.0) and np.all(out[~odd, 3] == 5.0)
    assert np.abs(out[odd, 3] - (m @ n)[odd]).max() < 1e-13


def test_matvec_brute_force_and_hop_composed_from_it():
    """matvec against numpy einsum for every operand form, and the hop term (def. 5) rebuilt from
    eight matvecs: chi = sum_mu [U_mu(x) psi(x+mu) + shift(adj(U_mu) psi, -mu)]."""
    dims = (4, 2, 6, 4)
    u, m, psi = synth.gauge_hot(dims, 511), synth.color_matrix(dims, 512), synth.spinor(dims, 513)
    for adj_a in (0, 1):
        for mu, sign in ((-1, 1), (0, 1), (2, -1), (3, 1)):
            A = dag(m) if adj_a else m
            p = psi if mu < 0 else sh(dims, psi, mu, sign)
            want = np.einsum("xab,xsb->xsa", A, p)
            assert np.abs(oracle.matvec(dims, m, 0, adj_a, psi, mu, sign) - want).max() < 1e-13
    chi = np.zeros_like(psi)
    for mu in range(4):
        chi += oracle.matvec(dims, u, mu, 0, psi, mu, +1)
        back = oracle.matvec(dims, u, mu, 1, psi)                       # U_mu(y)^dag psi(y) at y
        chi += oracle.shift(dims, back, mu, -1)
    assert np.abs(chi - oracle.hop(dims, u, psi)).max() < 1e-13
    odd = parity(dims) == 1
    sentinel = np.full_like(psi, 4.0)
    out = oracle.matvec(dims, u, 1, 0, psi, 1, 1, 1, chi=sentinel)
    assert np.all(out[odd] == 4.0) and np.abs(out[~odd] - np.einsum("xab,xsb->xsa", u[:, 1], sh(dims, psi, 1, 1))[~odd]).max() < 1e-13
