"""Pins for the oracle's reunitarisation (alternative projections)."""
import numpy as np
import pytest

import oracle
import synth
from npref import dag, parity


def _general(n, seed):
    """n general complex 3x3 matrices: SU(3) links perturbed by 30 % noise."""
    dims = (2, 2, 2, max(2, 2 * ((n + 15) // 16)))
    u = synth.gauge_hot(dims, seed).reshape(-1, 3, 3)[:n]
    noise = synth.color_matrix(dims, seed + 1).reshape(-1, 3, 3)[:n]
    return u + 0.3 * noise


def test_gram_schmidt_is_special_unitary_and_matches_qr():
    for k, V in enumerate(_general(40, 401)):
        G = oracle.gram_schmidt_su3(V)
        assert np.abs(G @ dag(G) - np.eye(3)).max() < 1e-14
        assert abs(np.linalg.det(G) - 1) < 1e-14
        # library pin: rows 0, 1 are the Q factor of a QR decomposition of V^T (columns = rows of V)
        # with the diagonal of R made positive; row 2 is then fixed by det = 1
        Q, R = np.linalg.qr(V.T)
        Q = Q * (np.conj(np.diag(R)) / np.abs(np.diag(R)))[None, :]
        assert np.abs(G[0] - Q[:, 0]).max() < 1e-13 and np.abs(G[1] - Q[:, 1]).max() < 1e-13
        assert np.abs(G[2] - np.conj(np.cross(G[0], G[1]))).max() < 1e-15
        # row 0 keeps its direction, row 1 stays in span(row0, row1)
        assert np.abs(G[0] - V[0] / np.linalg.norm(V[0])).max() < 1e-15
        assert abs(np.vdot(G[2], V[0])) < 1e-13 and abs(np.vdot(G[2], V[1])) < 1e-13


def test_both_methods_fix_su3_and_are_idempotent():
    dims = (2, 2, 2, 2)
    u = synth.gauge_hot(dims, 402)
    for method in (oracle.POLAR, oracle.GRAM_SCHMIDT):
        assert np.abs(oracle.reunitarize(dims, u, method) - u).max() < 1e-14
        v = u + 0.2 * synth.gauge_hot(dims, 403)
        once = oracle.reunitarize(dims, v, method)
        assert np.abs(oracle.reunitarize(dims, once, method) - once).max() < 1e-14
        g = once.reshape(-1, 3, 3)
        assert np.abs(g @ dag(g) - np.eye(3)).max() < 1e-13 and np.abs(np.linalg.det(g) - 1).max() < 1e-13


def test_polar_is_closer_than_gram_schmidt_and_covariant():
    """The polar factor maximises Re tr(X V^dag) over unitary X (so it beats Gram-Schmidt before the
    phase is removed), and Proj(g V h^dag) = g Proj(V) h^dag while Gram-Schmidt is not covariant."""
    V = _general(30, 404)
    g, h = synth.su3_site_field((2, 2, 2, 4), 405)[:30], synth.su3_site_field((2, 2, 2, 4), 406)[:30]
    worst_gs = 0.0
    for k in range(30):
        W, G = oracle.polar_unitary(V[k]), oracle.gram_schmidt_su3(V[k])
        assert np.trace(W @ dag(V[k])).real >= np.trace(G @ dag(V[k])).real - 1e-13
        lhs = oracle.proj_su3(g[k] @ V[k] @ dag(h[k]))
        assert np.abs(lhs - g[k] @ oracle.proj_su3(V[k]) @ dag(h[k])).max() < 1e-13
        worst_gs = max(worst_gs, np.abs(oracle.gram_schmidt_su3(g[k] @ V[k] @ dag(h[k])) - g[k] @ G @ dag(h[k])).max())
    assert worst_gs > 1e-3          # Gram-Schmidt is not covariant (reading A8)


def test_diagonal_closed_forms_and_fields():
    z = np.array([1.5 * np.exp(0.3j), 0.5 * np.exp(-1.1j), 2.0 * np.exp(0.4j)])
    G = oracle.gram_schmidt_su3(np.diag(z))
    want = np.diag([z[0] / abs(z[0]), z[1] / abs(z[1]), np.conj(z[0] * z[1]) / abs(z[0] * z[1])])
    assert np.abs(G - want).max() < 1e-15
    dims = (4, 2, 2, 2)
    u = synth.gauge_hot(dims, 407) + 0.1 * synth.gauge_hot(dims, 408)
    m = synth.color_matrix(dims, 409)
    odd = parity(dims) == 1
    for f in (u, m):
        sentinel = np.full_like(f, 7.0)
        full = oracle.reunitarize(dims, f, oracle.GRAM_SCHMIDT)
        assert np.abs(full.reshape(-1, 3, 3)[5] - oracle.gram_schmidt_su3(f.reshape(-1, 3, 3)[5])).max() == 0
        e = oracle.reunitarize(dims, f, oracle.GRAM_SCHMIDT, 1, out=sentinel)
        assert np.array_equal(e[~odd], full[~odd]) and np.all(e[odd] == 7.0)
        p = oracle.reunitarize(dims, f, oracle.POLAR)
        assert np.abs(p.reshape(-1, 3, 3)[3] - oracle.proj_su3(f.reshape(-1, 3, 3)[3])).max() == 0
