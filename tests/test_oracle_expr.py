"""Pins for the oracle side of the expression layer: `trace` / `real` of a product with
adjoints and shifted leaves, and the whole-field staple sum and APE blend (def. 3) that the expression kernels of
csrc/expr.cuh are compared with."""
import numpy as np
import pytest

import oracle
import synth
from npref import dag, parity, plaquette_np, sh, staple_np


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4)])
def test_trace_mul_brute_force_numpy_all_operand_forms(dims):
    u, m = synth.gauge_hot(dims, 801), synth.color_matrix(dims, 802)
    for adj_a in (0, 1):
        for adj_b in (0, 1):
            for mu, sign in ((-1, 1), (0, 1), (1, -1), (3, 1), (2, -1)):
                A = dag(u[:, 2]) if adj_a else u[:, 2]
                B = m if mu < 0 else sh(dims, m, mu, sign)
                B = dag(B) if adj_b else B
                want = np.einsum("xij,xji->x", A, B)
                got = oracle.trace_mul(dims, u, 2, adj_a, m, 0, adj_b, mu, sign)
                assert np.abs(got - want).max() < 1e-13, (adj_a, adj_b, mu, sign)


def test_trace_identities_and_closed_forms():
    dims = (4, 2, 6, 4)
    V = synth.volume(dims)
    a, b = synth.color_matrix(dims, 803), synth.color_matrix(dims, 804, 41)
    # cyclicity tr(AB) = tr(BA); tr(A A^dag) = |A|_F^2 is real and positive; tr(A^dag B) = conj tr(B^dag A)
    assert np.abs(oracle.trace_mul(dims, a, 0, 0, b, 0, 0) - oracle.trace_mul(dims, b, 0, 0, a, 0, 0)).max() < 1e-13
    n2 = oracle.trace_mul(dims, a, 0, 0, a, 0, 1)
    assert np.abs(n2.imag).max() == 0.0
    assert np.abs(n2.real - (np.abs(a) ** 2).sum(axis=(1, 2))).max() < 1e-13
    assert abs(n2.real.sum() - oracle.norm2(dims, a)) < 1e-10 * oracle.norm2(dims, a)
    t1, t2 = oracle.trace_mul(dims, a, 0, 1, b, 0, 0), oracle.trace_mul(dims, b, 0, 1, a, 0, 0)
    assert np.abs(t1 - np.conj(t2)).max() < 1e-13
    # SU(3) links: tr(U U^dag) = 3 exactly up to rounding; the unit field gives 3 for every form
    u = synth.gauge_hot(dims, 805)
    assert np.abs(oracle.trace_mul(dims, u, 1, 0, u, 1, 1) - 3.0).max() < 1e-14
    one = np.zeros((V, 3, 3), dtype=np.complex128)
    one[:] = np.eye(3)
    assert np.array_equal(oracle.trace_mul(dims, one, 0, 1, one, 0, 0, 2, -1), np.full(V, 3.0 + 0j))
    # subsets: only subset sites are written
    par = parity(dims)
    sentinel = np.full(V, 7.0 - 1.0j)
    got = oracle.trace_mul(dims, a, 0, 0, b, 0, 1, 1, 1, oracle.ODD, out=sentinel)
    assert np.array_equal(got[par == 0], sentinel[par == 0]) and not np.any(got[par == 1] == sentinel[par == 1])


def test_plaquette_is_the_sum_of_real_traces_of_composed_products():
    """sum_x real(trace(u[mu] * shift(u[nu], mu) * adj(shift(u[mu], nu)) * adj(u[nu]))) = def. 2: the expression the
    device layer evaluates in one kernel, composed here from matmul + trace_mul + real."""
    dims = (4, 2, 6, 4)
    u = synth.gauge_hot(dims, 806)
    V = synth.volume(dims)
    z = np.zeros((V, 3, 3), dtype=np.complex128)
    tot = np.zeros(3)
    for mu in range(4):
        for nu in range(mu + 1, 4):
            ab = oracle.matmul(dims, z, 0, u, mu, 0, u, nu, 0, mu, +1)          # u[mu] * shift(u[nu], mu)
            abc = oracle.matmul(dims, z, 0, ab, 0, 0, u, mu, 1, nu, +1)         # ... * adj(shift(u[mu], nu))
            retr = oracle.trace_mul(dims, abc, 0, 0, u, nu, 1).real             # real(trace(... * adj(u[nu])))
            assert np.abs(retr - plaquette_np(dims, u, mu, nu)).max() < 1e-13
            tot[0] += retr.sum()
            tot[1 if nu < 3 else 2] += retr.sum()
    want = oracle.plaquette(dims, u)
    assert abs(tot[0] / (18 * V) - want[0]) < 1e-13 and abs(tot[1] / (9 * V) - want[1]) < 1e-13
    assert abs(tot[2] / (9 * V) - want[2]) < 1e-13


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4)])
@pytest.mark.parametrize("t_dir", [3, -1])
def test_staple_and_blend_fields(dims, t_dir):
    u = synth.gauge_hot(dims, 807)
    dirs = [0, 1, 2] if t_dir == 3 else [0, 1, 2, 3]
    par = parity(dims)
    for mu in dirs:
        S = oracle.staple_field(dims, u, mu, t_dir)
        assert np.abs(S - staple_np(dims, u, mu, dirs)).max() < 1e-13          # numpy brute force (np.roll shifts)
        for lex in (0, 5, synth.volume(dims) - 1):
            assert np.array_equal(S[lex], oracle.staple_site(dims, u, lex, mu, t_dir)[0])
        n = 2 * (len(dirs) - 1)
        Vb = oracle.ape_blend_field(dims, u, mu, 0.35, t_dir)
        assert np.abs(Vb - (0.65 * u[:, mu] + 0.35 / n * S)).max() < 1e-14
        assert np.array_equal(oracle.ape_blend_field(dims, u, mu, 0.0, t_dir), u[:, mu])     # alpha = 0: the link itself
        # the APE step is Proj of the blend (def. 3-4)
        lex = 3
        assert np.abs(oracle.proj_su3(Vb[lex]) - oracle.ape_site(dims, u, lex, mu, 0.35, t_dir)).max() < 1e-14
        sentinel = np.full_like(S, 2.0 + 3.0j)
        Se = oracle.staple_field(dims, u, mu, t_dir, oracle.EVEN, out=sentinel)
        assert np.array_equal(Se[par == 1], sentinel[par == 1]) and np.array_equal(Se[par == 0], S[par == 0])
    # unit field: every staple is 1, S = n 1, the blend is 1
    one = np.zeros_like(u)
    one[:] = np.eye(3)
    assert np.array_equal(oracle.staple_field(dims, one, 0, t_dir), np.broadcast_to((2 * (len(dirs) - 1)) * np.eye(3), (synth.volume(dims), 3, 3)))
    assert np.abs(oracle.ape_blend_field(dims, one, 1, 0.5, t_dir) - np.eye(3)).max() < 1e-15
