"""Pins for the oracle's iterative max-Re-tr (Cabibbo-Marinari) projection, SURVEY.md 8(f) row f2."""
import numpy as np
import pytest

import oracle
import synth
from npref import parity


def _su3(seed, n):
    return synth.gauge_hot((2, 2, 2, 2), seed).reshape(-1, 3, 3)[:n]


def test_every_subgroup_update_keeps_su3_and_never_decreases_re_tr():
    Vs = synth.color_matrix((4, 2, 2, 2), 901)[:24]
    for V in Vs:
        X, tr = oracle.max_retr_su3(V, 8, with_trace=True)
        assert np.all(np.diff(tr) >= -1e-14 * np.abs(tr).max())          # monotone, update by update
        assert np.abs(X @ np.conj(X.T) - np.eye(3)).max() < 1e-14 and abs(np.linalg.det(X) - 1) < 1e-14
        # iters = 0 is the starting point: Gram-Schmidt of V
        assert np.array_equal(oracle.max_retr_su3(V, 0), oracle.gram_schmidt_su3(V))
        assert abs(tr[-1] - np.trace(X @ np.conj(V.T)).real) < 1e-13


def test_su3_input_is_a_fixed_point_and_the_maximum_is_three():
    for U in _su3(902, 16):
        X, tr = oracle.max_retr_su3(U, 3, with_trace=True)
        assert np.abs(X - U).max() < 1e-14
        assert np.abs(tr - 3.0).max() < 1e-14


def test_converges_to_the_known_maximiser():
    """V = U H with U in SU(3) and H Hermitian positive definite has polar factor U, the maximiser of Re tr(X V^dag)
    over all unitary X (value tr H); it lies in SU(3), so the sweeps must converge to it."""
    rng_mats = synth.color_matrix((2, 2, 2, 2), 903)[:8]
    for U, A in zip(_su3(904, 8), rng_mats):
        H = A @ np.conj(A.T) + 0.5 * np.eye(3)
        V = U @ H
        X, tr = oracle.max_retr_su3(V, 200, with_trace=True)
        assert abs(tr[-1] - np.trace(H).real) < 1e-9 * np.trace(H).real
        assert np.abs(X - U).max() < 1e-5            # quadratic objective: error in X ~ sqrt(error in the trace)
        assert np.abs(oracle.polar_unitary(V) - U).max() < 1e-12


def test_result_beats_other_su3_candidates():
    """Variational: after many sweeps Re tr(X V^dag) >= Re tr(Y V^dag) for Y = Gram-Schmidt(V), Proj(V) and random SU(3) Y."""
    Vs = synth.color_matrix((2, 2, 2, 2), 905)[:8]
    cands = _su3(906, 32)
    for V in Vs:
        X = oracle.max_retr_su3(V, 100)
        best = np.trace(X @ np.conj(V.T)).real
        for Y in [oracle.gram_schmidt_su3(V), oracle.proj_su3(V)] + list(cands):
            assert np.trace(Y @ np.conj(V.T)).real <= best + 1e-9 * abs(best)


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4)])
def test_whole_field_form_and_subsets(dims):
    u = synth.gauge_hot(dims, 907) + 0.3 * synth.gauge_hot(dims, 908)
    out = oracle.project_max_retr(dims, u, 4)
    for lex, mu in ((0, 0), (3, 2), (synth.volume(dims) - 1, 3)):
        assert np.array_equal(out[lex, mu], oracle.max_retr_su3(u[lex, mu], 4))
    par = parity(dims)
    sentinel = np.full_like(u, 1.0 + 1.0j)
    odd = oracle.project_max_retr(dims, u, 4, oracle.ODD, out=sentinel)
    assert np.array_equal(odd[par == 0], sentinel[par == 0]) and np.array_equal(odd[par == 1], out[par == 1])
