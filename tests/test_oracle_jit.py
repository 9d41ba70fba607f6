"""Pins of the oracle's run-time expression evaluator (oracle/expr_eval.py, second step), and the
host half of the library's front end (parser, kind check, NVRTC compilation) which needs no GPU."""
import numpy as np
import pytest

import oracle
import synth
from oracle import expr_eval as ee

DIMS = [(4, 4, 4, 4), (4, 2, 6, 4)]
PLAQ = "real(trace(f0[{m}] * shift(f0[{n}], +{m}) * adj(shift(f0[{m}], +{n})) * adj(f0[{n}])))"
UPPER = "f0[{n}] * shift(f0[{m}], +{n}) * adj(shift(f0[{n}], +{m}))"
LOWER = "shift(adj(f0[{n}]) * f0[{m}] * shift(f0[{n}], +{m}), -{n})"


def test_parser_precedence_and_associativity():
    assert ee.parse("f0 + f1 * f2") == ("+", ("f", 0, None), ("*", ("f", 1, None), ("f", 2, None)))
    assert ee.parse("f0 * f1 * f2") == ("*", ("*", ("f", 0, None), ("f", 1, None)), ("f", 2, None))
    assert ee.parse("(f0 + f1) * s2") == ("*", ("+", ("f", 0, None), ("f", 1, None)), ("s", 2))
    assert ee.parse("inner(f2, f0[1] * f2)") == ("inner", ("f", 2, None), ("*", ("f", 0, 1), ("f", 2, None)))
    assert ee.parse("shift(adj(f0[3]), -2)") == ("shift", ("adj", ("f", 0, 3)), 2, -1)
    for bad in ("f0 +", "f0 * * f1", "shift(f0, 2)", "trace f0", "f0[", "g0", "f0 f1", "(f0"):
        with pytest.raises(ee.ExprError):
            ee.parse(bad)


def test_kinds():
    slots = [4, 1]
    assert ee.kind_of(ee.parse("f0[1] * f1"), slots) == ee.MAT
    assert ee.kind_of(ee.parse("trace(f0[1] * f1)"), slots) == ee.CPLX
    assert ee.kind_of(ee.parse("real(trace(f1)) * s0"), slots) == ee.REAL
    assert ee.kind_of(ee.parse("s0 * f1 * s1"), slots) == ee.MAT
    assert ee.kind_of(ee.parse("trace(f1) * trace(f1)"), slots) == ee.CPLX
    for bad in ("f0 + trace(f1)", "trace(trace(f1))", "real(f1)", "f1 * trace(f1)", "f1[1]", "f0[4]", "f2", "shift(f1, +4)"):
        with pytest.raises(ee.ExprError):
            ee.kind_of(ee.parse(bad), slots)
    slots = [4, 1, 0]      # gauge, colour matrix, fermion
    assert ee.kind_of(ee.parse("f0[1] * shift(f2, +1)"), slots) == ee.SPINOR
    assert ee.kind_of(ee.parse("s0 * f2 + f1 * f2 * s1 + trace(f1) * f2 + f2 * trace(f1)"), slots) == ee.SPINOR
    assert ee.kind_of(ee.parse("norm2(f1 * f2)"), slots) == ee.REAL
    assert ee.kind_of(ee.parse("inner(f2, f0[3] * f2)"), slots) == ee.CPLX
    for bad in ("f2 * f1", "f2 * f2", "adj(f2)", "trace(f2)", "f2[0]", "norm2(f1)", "inner(f2, f1)", "f2 + f1", "inner(f2)"):
        with pytest.raises(ee.ExprError):
            ee.kind_of(ee.parse(bad), slots)


@pytest.mark.parametrize("dims", DIMS)
def test_plaquette_expression_is_def2(dims):
    """sum of real(trace(four links)) over the planes, normalised, is the plaquette of the C oracle (itself pinned on the
    unit field, abelian closed forms and numpy brute force: tests/test_oracle_plaquette.py)."""
    hu = synth.gauge_hot(dims, 41)
    V = synth.volume(dims)
    sp = sum(ee.total(dims, PLAQ.format(m=m, n=n), [hu]).real for m, n in ((0, 1), (0, 2), (1, 2)))
    tp = sum(ee.total(dims, PLAQ.format(m=m, n=3), [hu]).real for m in range(3))
    want = oracle.plaquette(dims, hu)
    assert abs(sp / (9 * V) - want[1]) < 1e-13 and abs(tp / (9 * V) - want[2]) < 1e-13
    # per site against the C oracle's own per-site plaquette
    v, kind = ee.evaluate(dims, PLAQ.format(m=0, n=1), [hu])
    assert kind == ee.REAL
    for lex in (0, 7, V - 1):
        assert abs(v[lex] - oracle.plaquette_site(dims, hu, lex)[0]) < 1e-13


@pytest.mark.parametrize("dims", DIMS)
def test_staple_and_blend_expressions_are_def3(dims):
    hu = synth.gauge_hot(dims, 42)
    for mu in range(3):
        nus = [n for n in range(3) if n != mu]
        text = " + ".join(UPPER.format(m=mu, n=n) + " + " + LOWER.format(m=mu, n=n) for n in nus)
        got, kind = ee.evaluate(dims, text, [hu])
        assert kind == ee.MAT
        assert np.abs(got - oracle.staple_field(dims, hu, mu, 3)).max() < 1e-13
        blend, _ = ee.evaluate(dims, f"s0 * f0[{mu}] + s1 * ({text})", [hu], [0.4, 0.6 / 4])
        assert np.abs(blend - oracle.ape_blend_field(dims, hu, mu, 0.6, 3)).max() < 1e-13


@pytest.mark.parametrize("dims", DIMS)
def test_trace_forms_match_trace_mul(dims):
    hu, hm = synth.gauge_hot(dims, 43), synth.color_matrix(dims, 44)
    got, _ = ee.evaluate(dims, "trace(adj(f0[2]) * shift(f1, -1))", [hu, hm])
    assert np.abs(got - oracle.trace_mul(dims, hu, 2, 1, hm, 0, 0, 1, -1)).max() < 1e-13
    got, _ = ee.evaluate(dims, "trace(f1 * adj(shift(f0[3], +0)))", [hu, hm])
    assert np.abs(got - oracle.trace_mul(dims, hm, 0, 0, hu, 3, 1, 0, +1)).max() < 1e-13


def test_algebraic_identities():
    dims = (4, 2, 6, 4)
    hu, hm = synth.gauge_hot(dims, 45), synth.color_matrix(dims, 46)
    ev = lambda t, s=(): ee.evaluate(dims, t, [hu, hm], s)[0]
    assert np.abs(ev("trace(f0[1] * f1)") - ev("trace(f1 * f0[1])")).max() < 1e-13                       # cyclicity
    assert np.abs(ev("adj(f0[1] * f1)") - ev("adj(f1) * adj(f0[1])")).max() < 1e-13                      # (AB)^dag
    assert np.array_equal(ev("shift(shift(f1, +2), -2)"), ev("f1"))                                      # shifts invert
    assert np.array_equal(ev("shift(f0[0] * f1, +3)"), ev("shift(f0[0], +3) * shift(f1, +3)"))           # site-local ops commute with shift
    assert np.array_equal(ev("shift(shift(f1, +0), +1)"), ev("shift(shift(f1, +1), +0)"))
    assert np.abs(ev("f0[2] * adj(f0[2])") - np.eye(3)).max() < 1e-13                                     # SU(3) links
    fro = (np.abs(hm) ** 2).sum(axis=(1, 2))
    assert np.abs(ev("real(trace(adj(f1) * f1))") - fro).max() < 1e-12 * fro.max()
    assert np.abs(ev("imag(trace(adj(f1) * f1))")).max() < 1e-13 * fro.max()
    assert np.abs(ev("s0 * f1 + s1 * f1", (0.25, 0.5)) - 0.75 * hm).max() < 1e-15 * np.abs(hm).max() * 4
    # brute force at one site: (a b)_ij and the trace, from the definitions
    x = 5
    a, b = hu[x, 1], hm[x]
    want = sum(a[i, k] * b[k, i] for i in range(3) for k in range(3))
    assert abs(ev("trace(f0[1] * f1)")[x] - want) < 1e-13


def test_minus_and_numbers_parse_and_type():
    """Binary '-' (left-associative, same level as '+'), the unary minus (binds tighter than '*') and decimal literals."""
    f0, f1, f2 = ("f", 0, None), ("f", 1, None), ("f", 2, None)
    assert ee.parse("f0 - f1 - f2") == ("-", ("-", f0, f1), f2)
    assert ee.parse("f0 - f1 + f2") == ("+", ("-", f0, f1), f2)
    assert ee.parse("f0 - f1 * f2") == ("-", f0, ("*", f1, f2))
    assert ee.parse("-f0 * f1") == ("*", ("neg", f0), f1)
    assert ee.parse("f0 - -f1") == ("-", f0, ("neg", f1))
    assert ee.parse("2 * f0") == ("*", ("num", 2.0), f0)
    assert ee.parse("f0[1] * 1.5e-3") == ("*", ("f", 0, 1), ("num", 0.0015))
    assert ee.parse(".5 + 10.") == ("+", ("num", 0.5), ("num", 10.0))
    assert ee.parse("shift(f0 - 2 * f1, -3)") == ("shift", ("-", f0, ("*", ("num", 2.0), f1)), 3, -1)
    for bad in ("f0 -", "- ", "f0[10]", "shift(f0, +12)", "1.5.2", "2 f0", "f0 - * f1", "1e"):
        with pytest.raises(ee.ExprError):
            ee.parse(bad)
    slots = [4, 1, 0]
    assert ee.kind_of(ee.parse("f0[1] - f1"), slots) == ee.MAT
    assert ee.kind_of(ee.parse("-f2"), slots) == ee.SPINOR
    assert ee.kind_of(ee.parse("f2 - 0.5 * f1 * f2"), slots) == ee.SPINOR
    assert ee.kind_of(ee.parse("0.5"), slots) == ee.REAL
    assert ee.kind_of(ee.parse("-real(trace(f1)) - 3"), slots) == ee.REAL
    for bad in ("f0 - trace(f1)", "trace(f1) - 2", "f2 - f1", "f1 - 1"):
        with pytest.raises(ee.ExprError):
            ee.kind_of(ee.parse(bad), slots)


def test_minus_and_numbers_evaluate_to_numpy_arithmetic():
    """Pinned on numpy written out here (elementwise subtraction, negation and scaling need nothing of the evaluator but the
    leaves) and on what the algebra fixes."""
    dims = (4, 2, 6, 4)
    hu, hm, hp = synth.gauge_hot(dims, 49), synth.color_matrix(dims, 50), synth.spinor(dims, 51)
    ev = lambda t, s=(): ee.evaluate(dims, t, [hu, hm, hp], s)[0]
    assert np.array_equal(ev("f0[1] - f1"), hu[:, 1] - hm)
    assert np.array_equal(ev("-f1"), -hm)
    assert np.array_equal(ev("-f2"), -hp)
    assert np.array_equal(ev("2.5 * f1"), 2.5 * hm)
    assert np.array_equal(ev("f0[0] - f1 * 0.5"), hu[:, 0] - hm * 0.5)
    assert np.array_equal(ev("f1 - f0[2] - f0[3]"), (hm - hu[:, 2]) - hu[:, 3])              # left-associative
    assert np.array_equal(ev("-f1 * f0[1]"), ev("(-f1) * f0[1]"))
    assert not ev("f1 - f1").any() and not ev("f2 - f2").any()
    assert np.array_equal(ev("f1 - s0 * f0[1]", (0.75,)), ev("f1 + s0 * f0[1]", (-0.75,)))       # a - c b = a + (-c) b
    assert np.array_equal(ev("f1 - 0.75 * f0[1]"), ev("f1 - s0 * f0[1]", (0.75,)))              # a literal is a scalar argument
    assert np.array_equal(ev("real(trace(f1 - adj(f1)))"), np.zeros(synth.volume(dims)))         # anti-Hermitian part: imaginary trace
    assert np.array_equal(ev("trace(f1) - trace(f1) * 2"), -(hm[:, 0, 0] + hm[:, 1, 1] + hm[:, 2, 2]))
    # the residual of PAPER.md:96, r = b - A x, against the C oracle's hop
    r = ev("f2 - 0.3 * (" + HOP_F2 + ")")
    want = hp - 0.3 * oracle.hop(dims, hu, hp)
    assert np.abs(r - want).max() < 1e-13 * np.abs(want).max()
    assert abs(ee.total(dims, "norm2(f2 - f2 * 0.5)", [hu, hm, hp]).real - 0.25 * oracle.norm2(dims, hp)) < 1e-12 * oracle.norm2(dims, hp)


HOP_F2 = " + ".join(f"f0[{m}] * shift(f2, +{m}) + shift(adj(f0[{m}]) * f2, -{m})" for m in range(4))
HOP = " + ".join(f"f0[{m}] * shift(f1, +{m}) + shift(adj(f0[{m}]) * f1, -{m})" for m in range(4))


@pytest.mark.parametrize("dims", DIMS)
def test_spinor_expressions_are_def5_and_def6(dims):
    """The hopping term, the fused a psi + b hop(psi), norm2 and innerProduct written as expressions equal the C oracle's
    functions (pinned on numpy brute force, plane waves, gauge covariance: tests/test_oracle_hop.py, _reductions.py)."""
    hu, hp = synth.gauge_hot(dims, 47), synth.spinor(dims, 48)
    chi, kind = ee.evaluate(dims, HOP, [hu, hp])
    assert kind == ee.SPINOR
    want = oracle.hop(dims, hu, hp)
    assert np.abs(chi - want).max() < 1e-13 * np.abs(want).max()
    axpy, _ = ee.evaluate(dims, f"s0 * f1 + s1 * ({HOP})", [hu, hp], (0.3, -0.7))
    w2 = oracle.axpy_hop(dims, 0.3, -0.7, hu, hp)
    assert np.abs(axpy - w2).max() < 1e-13 * np.abs(w2).max()
    n2 = ee.total(dims, f"norm2({HOP})", [hu, hp])
    assert abs(n2.real - oracle.norm2(dims, want)) < 1e-12 * n2.real and n2.imag == 0.0
    ip = ee.total(dims, f"inner(f1, {HOP})", [hu, hp])
    assert abs(ip - oracle.inner(dims, hp, want)) < 1e-12 * abs(n2)
    # the colour rotation leaves the spin index alone: a one-hot spinor stays in its spin component
    one = np.zeros_like(hp)
    one[:, 2, 1] = 1.0
    v, _ = ee.evaluate(dims, "f0[3] * f1", [hu, one])
    assert np.abs(v[:, [0, 1, 3]]).max() == 0.0 and np.abs(v[:, 2] - hu[:, 3, :, 1]).max() < 1e-15


# ---- the library's host-side front end (no GPU): it must accept and reject what the oracle's language does ------
VALID = [("f0[1] * f1", ee.MAT), ("trace(f0[1] * f1)", ee.CPLX), ("real(trace(f1)) * s0", ee.REAL), ("s0 * f1 * s1", ee.MAT),
         ("trace(f1) * trace(adj(f1)) + trace(f0[3])", ee.CPLX), (LOWER.format(m=0, n=2), ee.MAT), ("( f1+adj( f1 ) )*s1", ee.MAT),
         ("imag(trace(f1)) * real(trace(f0[0]))", ee.REAL), ("trace(f1) * s0", ee.CPLX),
         ("trace(s0 * f1)", ee.CPLX), ("real(trace(f1 * s0))", ee.REAL), ("trace((s0 * f1) * f0[1])", ee.CPLX),
         ("f0[1] - f1", ee.MAT), ("-f1 * f0[2] - 0.5 * f1", ee.MAT), ("real(trace(f1)) - 2.5e-1", ee.REAL), ("- - f1", ee.MAT),
         ("trace(f1 - adj(f1)) * -1", ee.CPLX), ("shift(f0[0] - 2 * f1, -3)", ee.MAT)]
INVALID = ["f0 + trace(f1)", "trace(trace(f1))", "real(f1)", "f1 * trace(f1)", "f1[1]", "f0[4]", "f2", "shift(f1, +4)", "f0 +",
           "shift(f0, 2)", "f0 f1", "(f0", "s2 * f1", "", "f0[0] * ", "adj f1", "f0 -", "f1 - 1", "trace(f1) - 2", "1.5.2", "2 f1",
           "f0[10]", "shift(f1, +12)", "1e"]


def test_library_front_end_agrees_with_the_oracle_language():
    q = pytest.importorskip("paper_1111_5596_b200")
    kinds = [q.QDP_GAUGE, q.QDP_COLOR_MATRIX]
    for text, kind in VALID:
        assert ee.kind_of(ee.parse(text), [4, 1]) == kind
        assert q.qdp_expr_jit_kind(text, kinds, 2) == kind, text
    for text in INVALID:
        with pytest.raises(q.QdpError):
            q.qdp_expr_jit_kind(text, kinds, 2)
        with pytest.raises(ee.ExprError):
            tree = ee.parse(text)
            ee.kind_of(tree, [4, 1])
            if "s2" in text:
                raise ee.ExprError("scalar argument out of range")   # the oracle takes its scalars from a Python sequence
    kinds = [q.QDP_GAUGE, q.QDP_COLOR_MATRIX, q.QDP_FERMION]
    for text, kind in [("f0[1] * shift(f2, +1)", ee.SPINOR), ("s0 * f2 + f1 * f2 * s1 + trace(f1) * f2 + f2 * trace(f1)", ee.SPINOR),
                       ("norm2(f1 * f2)", ee.REAL), ("inner(f2, f0[3] * f2)", ee.CPLX), (HOP.replace("f1", "f2"), ee.SPINOR),
                       ("f2 - 0.3 * (" + HOP_F2 + ")", ee.SPINOR), ("-f2", ee.SPINOR), ("norm2(f2 - f1 * f2)", ee.REAL)]:
        assert ee.kind_of(ee.parse(text), [4, 1, 0]) == kind
        assert q.qdp_expr_jit_kind(text, kinds, 2) == kind, text
    for text in ("f2 * f1", "f2 * f2", "adj(f2)", "trace(f2)", "f2[0]", "norm2(f1)", "inner(f2, f1)", "f2 + f1", "inner(f2)", "f2 - f1", "f2 - 1"):
        with pytest.raises(q.QdpError):
            q.qdp_expr_jit_kind(text, kinds, 2)
        with pytest.raises(ee.ExprError):
            ee.kind_of(ee.parse(text), [4, 1, 0])


def test_nvrtc_compiles_an_expression_once_without_a_gpu():
    q = pytest.importorskip("paper_1111_5596_b200")
    kinds = [q.QDP_GAUGE]
    text = "trace(f0[0] * adj(shift(f0[1], -2))) * s0"
    before = q.qdp_expr_jit_compilations()
    try:
        size = q.qdp_expr_jit_compile(text, kinds, 1, q.QDP_F64, sum_=True)
    except q.QdpError as exc:
        if "libnvrtc" in str(exc):
            pytest.skip("no libnvrtc on this machine")
        raise
    assert size > 1000 and q.qdp_expr_jit_compilations() == before + 1
    assert q.qdp_expr_jit_compile(text, kinds, 1, q.QDP_F64, sum_=True) == size      # cached
    assert q.qdp_expr_jit_compilations() == before + 1
    q.qdp_expr_jit_compile("trace( f0[0]*adj(shift(f0[1],-2)) )*s0", kinds, 1, q.QDP_F64, sum_=True)   # same tree, other spelling
    assert q.qdp_expr_jit_compilations() == before + 1
    q.qdp_expr_jit_compile(text, kinds, 1, q.QDP_F32, sum_=True)                     # another precision: another kernel
    assert q.qdp_expr_jit_compilations() == before + 2
    with pytest.raises(q.QdpError):
        q.qdp_expr_jit_compile("f0[0]", kinds, 0, q.QDP_F64, sum_=True)              # a matrix cannot be summed
    # every shape the front end accepts must also get through the compiler: a real scalar directly under a trace
    for shape in ("trace(s0 * f0[0])", "real(trace(f0[0] * s0))", "trace((s0 * f0[0]) * f0[1])",
                  "real(trace(-f0[0] - 0.5 * f0[1])) - 2", "trace(f0[0]) * -1.5e-1"):
        for prec in (q.QDP_F64, q.QDP_F32):
            assert q.qdp_expr_jit_compile(shape, kinds, 1, prec, sum_=True) > 1000, shape
