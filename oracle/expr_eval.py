"""ORACLE -- test infrastructure, not the product.

Run-time lattice expressions (second step), evaluated the slow and obvious
way: every sub-expression becomes a whole-lattice numpy array (exactly the temporaries QDP++ avoids), one node at a time,
in the order the expression is written.  Shares nothing with ``csrc/jit.cu``: own tokenizer, own recursive descent.

Grammar (the same language the library documents in ``include/qdp_b200.h``):

    expr   := term { ('+' | '-') term }  term := factor { '*' factor }
    factor := '-' factor | adj(expr) | trace(expr) | real(expr) | imag(expr) | norm2(expr) | inner(expr, expr)
            | shift(expr, +mu | -mu) | '(' expr ')' | leaf
    leaf   := f<k> [ '[' slot ']' ]  |  s<k>  |  number        (number: decimal literal, e.g. 2, 0.5, 1.5e-3)

Values: matrix field [V,3,3] complex128, spinor field [V,4,3] complex128 (a fermion argument), complex field [V]
complex128, real field [V] float64 (a scalar argument is a constant real field).  adj = conjugate transpose / complex
conjugate / identity on reals (not defined on spinors); trace over the colour indices; norm2(psi) = sum over spin and
colour of |psi|^2, inner(a, b) = sum over spin and colour of conj(a) b; shift(e, +mu)(x) = e(x + mu) with periodic wrap
(reading A3), done by ``oracle.shift`` on the evaluated array; '*' is the per-site matrix product, a matrix acting on the
colour index of every spin component of a spinor, scaling by a real or a complex number, or the product of complex
numbers; '+' adds and '-' subtracts values of equal kind, a leading '-' negates a value of any kind (it binds tighter than
'*': -a * b = (-a) * b), a number is a constant real field like a scalar argument.
"""
from __future__ import annotations

import re

import numpy as np

from . import shift as _shift, volume as _volume

MAT, CPLX, REAL, SPINOR = 0, 1, 2, 3
_NUMBER = r"(?:\d+\.\d*|\.\d+|\d+)(?:[eE][+-]?\d+)?"
_TOKEN = re.compile(r"\s*(adj|trace|real|imag|norm2|inner|shift|f\d|s\d|[()\[\],+\-*]|" + _NUMBER + ")")


class ExprError(ValueError):
    pass


def tokenize(text: str) -> list[str]:
    out, pos = [], 0
    text = text.rstrip()
    while pos < len(text):
        m = _TOKEN.match(text, pos)
        if not m:
            raise ExprError(f"bad input at {text[pos:pos + 12]!r}")
        out.append(m.group(1))
        pos = m.end()
    return out


def parse(text: str):
    """Returns a nested tuple tree: ('f', k, slot | None) | ('s', k) | ('adj'|'trace'|'real'|'imag'|'norm2', e) |
    ('inner', a, b) | ('shift', e, mu, sign) | ('+', a, b) | ('-', a, b) | ('*', a, b) | ('neg', e) | ('num', value);
    '+', '-' and '*' associate to the left, '*' binds tighter, the unary minus tighter still."""
    toks = tokenize(text)
    pos = 0

    def peek():
        return toks[pos] if pos < len(toks) else None

    def take(want=None):
        nonlocal pos
        t = peek()
        if t is None or (want is not None and t != want):
            raise ExprError(f"{want!r} expected, got {t!r}")
        pos += 1
        return t

    def expr():
        node = term()
        while peek() in ("+", "-"):
            op = take()
            node = (op, node, term())
        return node

    def term():
        node = factor()
        while peek() == "*":
            take()
            node = ("*", node, factor())
        return node

    def small_int(what):
        t = take()
        if not (len(t) == 1 and t.isdigit()):
            raise ExprError(f"{what}: one digit expected, got {t!r}")
        return int(t)

    def factor():
        t = take()
        if t == "-":
            return ("neg", factor())
        if t in ("adj", "trace", "real", "imag", "norm2"):
            take("(")
            e = expr()
            take(")")
            return (t, e)
        if t == "inner":
            take("(")
            a = expr()
            take(",")
            b = expr()
            take(")")
            return ("inner", a, b)
        if t == "shift":
            take("(")
            e = expr()
            take(",")
            sign = {"+": 1, "-": -1}.get(take())
            if sign is None:
                raise ExprError("'+' or '-' expected in shift")
            mu = small_int("direction")
            take(")")
            return ("shift", e, mu, sign)
        if t == "(":
            e = expr()
            take(")")
            return e
        if t[0] == "f" and len(t) == 2:
            slot = None                      # None: no subscript written
            if peek() == "[":
                take()
                slot = small_int("slot")
                take("]")
            return ("f", int(t[1]), slot)
        if t[0] == "s" and len(t) == 2:
            return ("s", int(t[1]))
        if t[0].isdigit() or t[0] == ".":
            return ("num", float(t))
        raise ExprError(f"operand expected, got {t!r}")

    tree = expr()
    if pos != len(toks):
        raise ExprError(f"unexpected {toks[pos]!r}")
    return tree


def kind_of(tree, field_slots) -> int:
    """Value kind of the expression; field_slots[k] = number of matrices per site of field argument k (1 colour matrix,
    4 gauge field) or 0 for a fermion field.  Raises ExprError for the combinations the language does not define."""
    op = tree[0]
    if op == "f":
        if tree[1] >= len(field_slots):
            raise ExprError("field argument out of range")
        if field_slots[tree[1]] == 0:
            if tree[2] is not None:
                raise ExprError("a fermion field has no slots")
            return SPINOR
        if (tree[2] or 0) >= field_slots[tree[1]]:
            raise ExprError("slot out of range")
        return MAT
    if op in ("s", "num"):
        return REAL
    if op == "neg":
        return kind_of(tree[1], field_slots)
    if op in ("adj", "shift"):
        if op == "shift" and not 0 <= tree[2] <= 3:
            raise ExprError("direction must be 0..3")
        k = kind_of(tree[1], field_slots)
        if op == "adj" and k == SPINOR:
            raise ExprError("adj() of a spinor is not defined")
        return k
    if op == "trace":
        if kind_of(tree[1], field_slots) != MAT:
            raise ExprError("trace() takes a matrix")
        return CPLX
    if op in ("real", "imag"):
        if kind_of(tree[1], field_slots) != CPLX:
            raise ExprError(f"{op}() takes a complex number")
        return REAL
    if op == "norm2":
        if kind_of(tree[1], field_slots) != SPINOR:
            raise ExprError("norm2() takes a spinor")
        return REAL
    a, b = kind_of(tree[1], field_slots), kind_of(tree[2], field_slots)
    if op == "inner":
        if a != SPINOR or b != SPINOR:
            raise ExprError("inner() takes two spinors")
        return CPLX
    if op in ("+", "-"):
        if a != b:
            raise ExprError(f"'{op}' needs operands of the same kind")
        return a
    if a == REAL:
        return b
    if b == REAL:
        return a
    if (a, b) in ((MAT, MAT), (CPLX, CPLX)):
        return a
    if (a, b) in ((MAT, SPINOR), (CPLX, SPINOR), (SPINOR, CPLX)):
        return SPINOR
    raise ExprError("'*' is not defined for these operand kinds")


def evaluate(dims, text: str, fields, scalars=()):
    """The expression at every site.  fields[k]: [V,3,3] (colour matrix), [V,4,3,3] (gauge) or [V,4,3] (fermion) complex
    arrays.  Returns ([V,3,3] | [V,4,3] | [V] complex128 | [V] float64, kind)."""
    V = _volume(dims)
    fields = [np.asarray(f, dtype=np.complex128) for f in fields]
    is_spinor = [f.ndim == 3 and f.shape[1:] == (4, 3) for f in fields]
    mats = [None if sp else f.reshape(V, -1, 3, 3) for f, sp in zip(fields, is_spinor)]
    tree = parse(text)
    kind = kind_of(tree, [0 if sp else m.shape[1] for m, sp in zip(mats, is_spinor)])

    def is_mat(v):
        return v.ndim == 3 and v.shape[1:] == (3, 3)

    def is_spin(v):
        return v.ndim == 3 and v.shape[1:] == (4, 3)

    def ev(t):
        op = t[0]
        if op == "f":
            return fields[t[1]].copy() if is_spinor[t[1]] else mats[t[1]][:, t[2] or 0].copy()
        if op == "s":
            return np.full(V, float(scalars[t[1]]))
        if op == "num":
            return np.full(V, t[1])
        if op == "neg":
            return -ev(t[1])
        if op == "adj":
            v = ev(t[1])
            return np.conj(np.swapaxes(v, 1, 2)) if is_mat(v) else np.conj(v)
        if op == "trace":
            v = ev(t[1])
            return v[:, 0, 0] + v[:, 1, 1] + v[:, 2, 2]
        if op == "real":
            return np.ascontiguousarray(ev(t[1]).real)
        if op == "imag":
            return np.ascontiguousarray(ev(t[1]).imag)
        if op == "norm2":
            v = ev(t[1])
            return (v.real ** 2 + v.imag ** 2).reshape(V, 12).sum(axis=1)
        if op == "inner":
            a, b = ev(t[1]), ev(t[2])
            return (np.conj(a) * b).reshape(V, 12).sum(axis=1)
        if op == "shift":
            return _shift(dims, np.ascontiguousarray(ev(t[1])), t[2], t[3])
        a, b = ev(t[1]), ev(t[2])
        if op == "+":
            return a + b
        if op == "-":
            return a - b
        if is_mat(a) and is_mat(b):
            out = np.zeros_like(a)
            for i in range(3):            # (a b)_ij = sum_k a_ik b_kj, written out
                for j in range(3):
                    for k in range(3):
                        out[:, i, j] += a[:, i, k] * b[:, k, j]
            return out
        if is_mat(a) and is_spin(b):
            out = np.zeros_like(b)
            for sp in range(4):           # (a psi)_{s,i} = sum_k a_ik psi_{s,k}: spin untouched (reading A11)
                for i in range(3):
                    for k in range(3):
                        out[:, sp, i] += a[:, i, k] * b[:, sp, k]
            return out
        if a.ndim == 3:
            return a * b[:, None, None]
        if b.ndim == 3:
            return a[:, None, None] * b
        return a * b

    return ev(tree), kind


def total(dims, text: str, fields, scalars=(), mask=None) -> complex:
    """sum over the sites (of the subset given by the boolean mask) of a real or complex expression, exactly rounded
    (math.fsum) so that the comparison bar is the GPU's, not this sum's."""
    import math
    v, kind = evaluate(dims, text, fields, scalars)
    if kind in (MAT, SPINOR):
        raise ExprError("a sum needs a real or complex expression")
    if mask is not None:
        v = v[mask]
    v = np.asarray(v, dtype=np.complex128)
    return complex(math.fsum(v.real), math.fsum(v.imag))
