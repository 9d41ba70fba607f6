"""Run-time expressions on the GPU (qdp_expr_jit_*, second step) against the oracle's
evaluator (oracle/expr_eval.py), element by element, through the C ABI."""
import numpy as np
import pytest

import oracle
import synth
from oracle import expr_eval as ee
from parity import TOL_SITE, TOL_SUM, site_rel_err

pytestmark = pytest.mark.gpu

SMALL = [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4), (6, 4, 2, 8), (10, 6, 4, 2)]
C2 = synth.CONFIGS["C2"]
PLAQ01 = "real(trace(f0[0] * shift(f0[1], +0) * adj(shift(f0[0], +1)) * adj(f0[1])))"
# (expression, scalars): f0 = gauge field, f1 = colour-matrix field
ASSIGN = [
    ("f0[2] * shift(f1, +1)", ()),
    ("adj(f0[1]) * f1 + s0 * f0[3]", (0.7,)),
    ("shift(adj(f0[1]) * f0[0] * shift(f0[1], +0), -1)", ()),                    # a lower staple: nested shifts
    ("f0[1] * shift(f0[0], +1) * adj(shift(f0[1], +0)) + shift(adj(f0[2]) * f0[0] * shift(f0[2], +0), -2)", ()),
    ("(f1 + adj(f1)) * s1", (0.0, -1.5)),
    ("trace(f0[0] * adj(shift(f1, -3)))", ()),                                   # complex-valued
    ("s0 * trace(f1) * trace(adj(f0[2])) + trace(f1 * f1)", (0.3,)),
    ("trace(s0 * f1)", (0.7,)),                                                  # a real scalar directly under the trace
    ("trace((s0 * f1) * f0[2]) + trace(f0[1] * s1)", (1.3, -0.6)),
    ("f0[1] - f1 * 0.5", ()),                                                    # '-', literals, unary minus
    ("-f1 * f0[2] - (f1 - adj(f1)) * s0 - - shift(f0[3], -1)", (0.25,)),
    ("trace(f1 - adj(f1)) * -1.5e-1 - trace(f0[0])", ()),
]
SUMS = [
    (PLAQ01, ()),
    ("trace(f0[3] * shift(f1, -2)) * s0", (2.0,)),
    ("imag(trace(f1)) * real(trace(f0[0]))", ()),
    ("real(trace(adj(f1) * f1))", ()),
    ("real(trace(f1 * s0)) + real(trace(s1 * f0[2]))", (-0.4, 1.1)),
    ("3 - real(trace(f0[0] * shift(f0[1], +0) * adj(shift(f0[0], +1)) * adj(f0[1])))", ()),   # 3 - Re tr (plaquette): the Wilson action density
    ("-imag(trace(f1)) - 0.125 * real(trace(f0[2] - f1))", ()),
]


def _seed(dims):
    return synth.BASE_SEED + 7 * sum(dims)


def _setup(qdp, dims, prec):
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 201), prec)
    hm = synth.round_to(synth.color_matrix(dims, _seed(dims) + 202), prec)
    lat = qdp.qdp_lattice_create(dims)
    return lat, hu, hm, qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 0, hm)


def _scalars(sc, prec):
    return tuple(float(np.float32(x)) for x in sc) if prec == "f32" else tuple(sc)   # the kernel casts scalars to the field precision


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_jit_assign_matches_oracle(qdp, dims, prec):
    lat, hu, hm, u, m = _setup(qdp, dims, prec)
    P = 1 if prec == "f64" else 0
    V = synth.volume(dims)
    mask = oracle.parity_mask(dims)
    cdt = np.complex128 if P else np.complex64
    for text, sc in ASSIGN:
        want, kind = ee.evaluate(dims, text, [hu.astype(np.complex128), hm.astype(np.complex128)], _scalars(sc, prec))
        for subset in (0, 1, 2):
            sel = np.ones(V, bool) if subset == 0 else (mask == (subset - 1))
            if kind == ee.MAT:
                sentinel = np.full((V, 3, 3), 5.0 - 2.0j, cdt)
                dst = qdp.field_from_host(lat, 0, sentinel)
            else:
                sentinel = np.full((V,), 5.0 - 2.0j, cdt)
                dst = qdp.field_from_host(lat, 3, sentinel)
            before = qdp.qdp_kernel_launch_count()
            qdp.qdp_expr_jit_assign(dst, 0, text, [u, m], sc, subset)
            assert qdp.qdp_kernel_launch_count() == before + 1                  # one kernel per expression
            got = qdp.field_to_host(dst)
            assert np.array_equal(got[~sel], sentinel[~sel]), text              # other sites untouched
            scale = np.sqrt((np.abs(want.reshape(V, -1)) ** 2).sum(axis=1)).max()
            err = np.abs(got.reshape(V, -1)[sel] - want.reshape(V, -1)[sel]).max()
            # per-site bar of the north star, relative to the largest site value (a complex-valued trace can cancel to ~0
            # at single sites; its terms are O(scale))
            assert err <= TOL_SITE[prec] * max(scale, 1.0), (text, subset, err)


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_jit_sum_matches_oracle(qdp, dims, prec):
    lat, hu, hm, u, m = _setup(qdp, dims, prec)
    V = synth.volume(dims)
    mask = oracle.parity_mask(dims)
    for text, sc in SUMS:
        v, _ = ee.evaluate(dims, text, [hu.astype(np.complex128), hm.astype(np.complex128)], _scalars(sc, prec))
        for subset in (0, 1, 2):
            sel = np.ones(V, bool) if subset == 0 else (mask == (subset - 1))
            want = ee.total(dims, text, [hu.astype(np.complex128), hm.astype(np.complex128)], _scalars(sc, prec), sel)
            got = qdp.qdp_expr_jit_sum(text, [u, m], sc, subset)
            assert abs(got - want) <= TOL_SUM[prec] * np.abs(v[sel]).sum(), (text, subset, got, want)
            assert got == qdp.qdp_expr_jit_sum(text, [u, m], sc, subset)        # deterministic


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_jit_equals_build_time_instantiations(qdp, prec):
    """The same expression through NVRTC and through nvcc (qdp_expr_plaquette, qdp_expr_staple): same node types, same
    arithmetic per site."""
    dims = (4, 2, 6, 4)
    lat, hu, hm, u, m = _setup(qdp, dims, prec)
    V = synth.volume(dims)
    plane = "real(trace(f0[{a}] * shift(f0[{b}], +{a}) * adj(shift(f0[{a}], +{b})) * adj(f0[{b}])))"
    planes = lambda pairs: " + ".join(plane.format(a=a, b=b) for a, b in pairs)
    sp = qdp.qdp_expr_jit_sum(planes([(0, 1), (0, 2), (1, 2)]), [u]).real / (9 * V)
    tp = qdp.qdp_expr_jit_sum(planes([(0, 3), (1, 3), (2, 3)]), [u]).real / (9 * V)
    ref = qdp.qdp_expr_plaquette(u)
    tol = 1e-12 if prec == "f64" else 1e-5
    assert abs(sp - ref[1]) <= tol and abs(tp - ref[2]) <= tol
    staple = ("(f0[1] * shift(f0[0], +1) * adj(shift(f0[1], +0)) + shift(adj(f0[1]) * f0[0] * shift(f0[1], +0), -1)) + "
              "(f0[2] * shift(f0[0], +2) * adj(shift(f0[2], +0)) + shift(adj(f0[2]) * f0[0] * shift(f0[2], +0), -2))")
    a, b = qdp.qdp_field_alloc(lat, 0, u.prec), qdp.qdp_field_alloc(lat, 0, u.prec)
    qdp.qdp_expr_jit_assign(a, 0, staple, [u])
    qdp.qdp_expr_staple(b, u, 0, 3)
    assert np.array_equal(qdp.field_to_host(a), qdp.field_to_host(b))


def test_jit_cache_errors_and_aliasing(qdp):
    dims = (4, 4, 4, 4)
    lat, hu, hm, u, m = _setup(qdp, dims, "f64")
    text = "f1 * adj(f0[2]) * s0"
    dst = qdp.qdp_field_alloc(lat, 0, 1)
    qdp.qdp_expr_jit_assign(dst, 0, text, [u, m], (1.0,))
    n = qdp.qdp_expr_jit_compilations()
    for _ in range(3):
        qdp.qdp_expr_jit_assign(dst, 0, " f1*adj( f0[2] ) * s0 ", [u, m], (2.0,))      # same tree: cached kernel
    assert qdp.qdp_expr_jit_compilations() == n
    want, _ = ee.evaluate(dims, text, [hu, hm], (2.0,))
    assert site_rel_err(qdp.field_to_host(dst), want).max() <= 1e-12
    # site-local expressions may overwrite an operand; a gauge slot can be the destination
    qdp.qdp_expr_jit_assign(m, 0, "f1 * adj(f0[2]) * s0", [u, m], (2.0,))
    assert site_rel_err(qdp.field_to_host(m), want).max() <= 1e-12
    qdp.qdp_expr_jit_assign(u, 3, "f0[0] * f0[1]", [u])
    w2, _ = ee.evaluate(dims, "f0[0] * f0[1]", [hu])
    got = qdp.field_to_host(u)
    assert site_rel_err(got[:, 3], w2).max() <= 1e-12 and np.array_equal(got[:, :3], hu[:, :3])
    with pytest.raises(qdp.QdpError):      # neighbour reads of the destination
        qdp.qdp_expr_jit_assign(m, 0, "shift(f1, +0) * f0[1]", [u, m])
    with pytest.raises(qdp.QdpError):      # kind of the destination
        qdp.qdp_expr_jit_assign(dst, 0, "trace(f1)", [u, m])
    with pytest.raises(qdp.QdpError):      # syntax
        qdp.qdp_expr_jit_assign(dst, 0, "f1 * ", [u, m])
    with pytest.raises(qdp.QdpError):      # a matrix cannot be summed
        qdp.qdp_expr_jit_sum("f1", [u, m])
    psi = qdp.field_from_host(lat, 2, synth.spinor(dims, 3))
    with pytest.raises(qdp.QdpError):      # fermions are not matrix operands
        qdp.qdp_expr_jit_assign(dst, 0, "f0", [psi])


HOP = " + ".join(f"f0[{m}] * shift(f1, +{m}) + shift(adj(f0[{m}]) * f1, -{m})" for m in range(4))


@pytest.mark.parametrize("dims", SMALL + [C2])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_jit_spinor_expressions(qdp, dims, prec):
    """Fermion leaves: the hopping term (def. 5) and a psi + b hop(psi) (def. 6) written as text, their fused norm2 and
    innerProduct, against the oracle's evaluator and against the hand-fused kernels."""
    hu = synth.round_to(synth.gauge_hot(dims, _seed(dims) + 211), prec)
    hp = synth.round_to(synth.spinor(dims, _seed(dims) + 212), prec)
    lat = qdp.qdp_lattice_create(dims)
    u, psi = qdp.field_from_host(lat, 1, hu), qdp.field_from_host(lat, 2, hp)
    V = synth.volume(dims)
    mask = oracle.parity_mask(dims)
    h64 = [hu.astype(np.complex128), hp.astype(np.complex128)]
    sc = _scalars((0.3, -0.7), prec)
    axpy = f"s0 * f1 + s1 * ({HOP})"
    want_hop, kind = ee.evaluate(dims, HOP, h64)
    assert kind == ee.SPINOR
    want_axpy, _ = ee.evaluate(dims, axpy, h64, sc)
    resid = f"f1 - s0 * ({HOP}) - 0.5 * -f1"          # the residual form b - A x of PAPER.md:96, with '-' and a literal
    want_resid, _ = ee.evaluate(dims, resid, h64, _scalars((0.3,), prec))
    sentinel = np.full((V, 4, 3), 3.0 + 1.0j, hp.dtype)
    for subset in (0, 1, 2):
        sel = np.ones(V, bool) if subset == 0 else (mask == (subset - 1))
        for text, want, s in ((HOP, want_hop, ()), (axpy, want_axpy, (0.3, -0.7)), (resid, want_resid, (0.3,))):
            chi = qdp.field_from_host(lat, 2, sentinel)
            qdp.qdp_expr_jit_assign(chi, 0, text, [u, psi], s, subset)
            got = qdp.field_to_host(chi)
            assert np.array_equal(got[~sel], sentinel[~sel])
            assert site_rel_err(got[sel], want[sel]).max() <= TOL_SITE[prec], (text[:30], subset)
        n2 = qdp.qdp_expr_jit_sum(f"norm2({HOP})", [u, psi], (), subset)
        w = ee.total(dims, f"norm2({HOP})", h64, (), sel)
        assert abs(n2 - w) <= TOL_SUM[prec] * abs(w) and n2.imag == 0.0
        ip = qdp.qdp_expr_jit_sum(f"inner(f1, {HOP})", [u, psi], (), subset)
        wi = ee.total(dims, f"inner(f1, {HOP})", h64, (), sel)
        assert abs(ip - wi) <= TOL_SUM[prec] * 8 * float((np.abs(h64[1][sel]) ** 2).sum())
    # the hand-fused kernel evaluates the same definition
    a, b = qdp.qdp_field_alloc(lat, 2, u.prec), qdp.qdp_field_alloc(lat, 2, u.prec)
    qdp.qdp_expr_jit_assign(a, 0, HOP, [u, psi])
    qdp.qdp_hop(b, u, psi)
    assert site_rel_err(qdp.field_to_host(a), qdp.field_to_host(b)).max() <= (1e-13 if prec == "f64" else 1e-5)
    # destination kinds
    m = qdp.qdp_field_alloc(lat, 0, u.prec)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_expr_jit_assign(m, 0, HOP, [u, psi])
    with pytest.raises(qdp.QdpError):
        qdp.qdp_expr_jit_sum(HOP, [u, psi])
