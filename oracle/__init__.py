"""ORACLE -- test infrastructure, not the product.

ctypes front end of ``qdp_oracle.c``: a plain single-threaded fp64 CPU
implementation of the lattice expressions (definitions 1-6).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` leg may import this package.  It imports nothing from
``paper_1111_5596_b200`` and shares no code with the CUDA path.

Arrays: host, lexicographic sites (x0 fastest), complex128,
gauge [V,4,3,3], fermion [V,4,3], colour matrix [V,3,3].
For fp32 parity the caller passes the fp32-rounded inputs converted back to
complex128 (reading A13): the oracle always computes in fp64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qdp_oracle.c")
_LIB = os.path.join(_HERE, "libqdp_oracle.so")

ALL, EVEN, ODD = 0, 1, 2
CFLAGS = ["-O2", "-ffp-contract=off"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _get():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P, I, Z, D = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_double
        sig = {
            "orc_neighbor_table": ([P, I, I, P], None),
            "orc_parity_mask": ([P, P], None),
            "orc_shift_bytes": ([P, Z, P, P, I, I, I], None),
            "orc_plaquette_site": ([P, P, Z, P], None),
            "orc_plaquette": ([P, P, I, P], None),
            "orc_polar_unitary": ([P, P], None),
            "orc_proj_su3": ([P, P], None),
            "orc_min_eig_vdv": ([P], D),
            "orc_gram_schmidt_su3": ([P, P], None),
            "orc_matvec": ([P, P, P, I, I, I, P, I, I, I], None),
            "orc_matmul": ([P, P, I, I, P, I, I, I, P, I, I, I, I, I, I], None),
            "orc_reunitarize": ([P, I, P, P, I, I], None),
            "orc_max_retr_su3": ([P, I, P, P], None),
            "orc_project_max_retr": ([P, I, P, P, I, I], None),
            "orc_baryon_timeslices": ([P, I, P, P, P, I, I, P], None),
            "orc_trace_mul": ([P, P, P, I, I, I, P, I, I, I, I, I, I], None),
            "orc_staple_field": ([P, P, I, I, I, P], None),
            "orc_ape_blend_field": ([P, P, I, D, I, I, P], None),
            "orc_staple_site": ([P, P, Z, I, I, P], I),
            "orc_ape_blend_site": ([P, P, Z, I, D, I, P], None),
            "orc_ape_site": ([P, P, Z, I, D, I, P], None),
            "orc_ape_smear_step": ([P, P, P, D, I, I], None),
            "orc_hop_site": ([P, P, P, Z, P], None),
            "orc_hop": ([P, P, P, P, I], None),
            "orc_axpy_hop": ([P, D, D, P, P, P, I], None),
            "orc_hop_site_dirs": ([P, P, P, Z, I, P], None),
            "orc_smear_hop": ([P, D, D, P, P, P, I, I], None),
            "orc_norm2": ([P, I, P, I], D),
            "orc_inner": ([P, I, P, P, I, P], None),
            "orc_sum": ([P, I, P, I, P], None),
            "orc_inner_timeslices": ([P, I, P, P, I, P], None),
            "orc_axpby": ([P, I, D, P, D, P, P, I], None),
            "orc_gamma_matrix": ([I, P], None),
            "orc_inner_timeslices_gamma": ([P, P, P, I, I, P], None),
            # the same loops over lex sites [begin, end): bounded samples for bench.py
            "orc_shift_bytes_range": ([P, Z, P, P, I, I, I, Z, Z], None),
            "orc_plaquette_range": ([P, P, I, Z, Z, P], None),
            "orc_ape_smear_step_range": ([P, P, P, D, I, I, Z, Z], None),
            "orc_hop_range": ([P, P, P, P, I, Z, Z], None),
            "orc_axpy_hop_range": ([P, D, D, P, P, P, I, Z, Z], None),
            "orc_norm2_range": ([P, I, P, I, Z, Z], D),
            "orc_inner_range": ([P, I, P, P, I, Z, Z, P], None),
        }
        for name, (args, res) in sig.items():
            f = getattr(lib, name)
            f.argtypes, f.restype = args, res
        _lib = lib
    return _lib


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def _c128(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def volume(dims):
    return int(np.prod([int(d) for d in dims]))


def neighbor_table(dims, mu, sign):
    out = np.empty(volume(dims), dtype=np.int32)
    _get().orc_neighbor_table(_dims(dims), mu, sign, out.ctypes.data)
    return out


def parity_mask(dims):
    out = np.empty(volume(dims), dtype=np.uint8)
    _get().orc_parity_mask(_dims(dims), out.ctypes.data)
    return out


def shift(dims, src, mu, sign, subset=ALL, dst=None):
    """dst(x) = src(x + sign*mu) on the subset; any dtype, moved as bytes."""
    src = np.ascontiguousarray(src)
    V = volume(dims)
    dst = np.zeros_like(src) if dst is None else np.ascontiguousarray(dst).copy()
    _get().orc_shift_bytes(_dims(dims), src.nbytes // V, src.ctypes.data, dst.ctypes.data,
                           mu, sign, subset)
    return dst


def plaquette(dims, u, subset=ALL):
    u = _c128(u)
    out = np.empty(3)
    _get().orc_plaquette(_dims(dims), u.ctypes.data, subset, out.ctypes.data)
    return out


def plaquette_site(dims, u, lex):
    u = _c128(u)
    out = np.empty(6)
    _get().orc_plaquette_site(_dims(dims), u.ctypes.data, lex, out.ctypes.data)
    return out


def polar_unitary(V):
    V = _c128(V)
    out = np.empty((3, 3), dtype=np.complex128)
    _get().orc_polar_unitary(V.ctypes.data, out.ctypes.data)
    return out


def proj_su3(V):
    V = _c128(V)
    out = np.empty((3, 3), dtype=np.complex128)
    _get().orc_proj_su3(V.ctypes.data, out.ctypes.data)
    return out


def matmul(dims, dst, id_, a, ia, adj_a, b, ib, adj_b, mu=-1, sign=1, subset=ALL):
    """dst[:, id_] = op(a[:, ia])(x) @ op(b[:, ib])(x + sign*mu) on the subset (row f1); fields are
    [V,3,3] (index 0) or [V,4,3,3]; returns the updated copy of dst."""
    a, b, out = _c128(a), _c128(b), _c128(dst).copy()
    V = volume(dims)
    _get().orc_matmul(_dims(dims), out.ctypes.data, out.size // (9 * V), id_, a.ctypes.data, a.size // (9 * V), ia,
                      int(adj_a), b.ctypes.data, b.size // (9 * V), ib, int(adj_b), mu, sign, subset)
    return out


def matvec(dims, a, ia, adj_a, psi, mu=-1, sign=1, subset=ALL, chi=None):
    """chi(x) = op(a[:, ia])(x) psi(x + sign*mu) on the subset (row f1); a is [V,3,3] or [V,4,3,3]."""
    a, psi = _c128(a), _c128(psi)
    out = np.zeros_like(psi) if chi is None else _c128(chi).copy()
    _get().orc_matvec(_dims(dims), out.ctypes.data, a.ctypes.data, a.size // (9 * volume(dims)), ia, int(adj_a),
                      psi.ctypes.data, mu, sign, subset)
    return out


def trace_mul(dims, a, ia, adj_a, b, ib, adj_b, mu=-1, sign=1, subset=ALL, out=None):
    """out(x) = tr[op(a[:, ia])(x) @ op(b[:, ib])(x + sign*mu)] on the subset, [V] complex128 (row f1: `trace`;
    `real` of it is .real); fields are [V,3,3] (index 0) or [V,4,3,3]."""
    a, b = _c128(a), _c128(b)
    V = volume(dims)
    res = np.zeros(V, dtype=np.complex128) if out is None else _c128(out).copy()
    _get().orc_trace_mul(_dims(dims), res.ctypes.data, a.ctypes.data, a.size // (9 * V), ia, int(adj_a),
                         b.ctypes.data, b.size // (9 * V), ib, int(adj_b), mu, sign, subset)
    return res


def staple_field(dims, u, mu, t_dir=3, subset=ALL, out=None):
    """out(x) = S_mu(x), the staple sum around link mu (def. 3), as a colour-matrix field [V,3,3]."""
    u = _c128(u)
    res = np.zeros((volume(dims), 3, 3), dtype=np.complex128) if out is None else _c128(out).copy()
    _get().orc_staple_field(_dims(dims), u.ctypes.data, mu, t_dir, subset, res.ctypes.data)
    return res


def ape_blend_field(dims, u, mu, alpha, t_dir=3, subset=ALL, out=None):
    """out(x) = (1-alpha) U_mu(x) + (alpha/n) S_mu(x): the APE link before projection, [V,3,3]."""
    u = _c128(u)
    res = np.zeros((volume(dims), 3, 3), dtype=np.complex128) if out is None else _c128(out).copy()
    _get().orc_ape_blend_field(_dims(dims), u.ctypes.data, mu, alpha, t_dir, subset, res.ctypes.data)
    return res


def gram_schmidt_su3(V):
    V = _c128(V)
    out = np.empty((3, 3), dtype=np.complex128)
    _get().orc_gram_schmidt_su3(V.ctypes.data, out.ctypes.data)
    return out


POLAR, GRAM_SCHMIDT = 0, 1


def reunitarize(dims, f, method=POLAR, subset=ALL, out=None):
    """Every 3x3 matrix of the field ([V,4,3,3] or [V,3,3]) projected to SU(3) (row f2)."""
    f = _c128(f)
    res = np.zeros_like(f) if out is None else _c128(out).copy()
    nmat = f.size // (volume(dims) * 9)
    _get().orc_reunitarize(_dims(dims), nmat, f.ctypes.data, res.ctypes.data, method, subset)
    return res


def max_retr_su3(V, iters, with_trace=False):
    """Cabibbo-Marinari-style projection of one matrix (row f2): X_0 = Gram-Schmidt(V), then `iters` sweeps over the
    SU(2) subgroups (0,1), (1,2), (0,2), each maximising Re tr(X V^dag).  with_trace: also Re tr(X V^dag) after X_0 and
    after each of the 3*iters updates."""
    V = _c128(V)
    out = np.empty((3, 3), dtype=np.complex128)
    tr = np.empty(1 + 3 * iters)
    _get().orc_max_retr_su3(V.ctypes.data, int(iters), out.ctypes.data, tr.ctypes.data if with_trace else None)
    return (out, tr) if with_trace else out


def project_max_retr(dims, f, iters, subset=ALL, out=None):
    """Every 3x3 matrix of the field ([V,4,3,3] or [V,3,3]) replaced by its max-Re-tr projection after `iters` sweeps."""
    f = _c128(f)
    res = np.zeros_like(f) if out is None else _c128(out).copy()
    nmat = f.size // (volume(dims) * 9)
    _get().orc_project_max_retr(_dims(dims), nmat, f.ctypes.data, res.ctypes.data, int(iters), subset)
    return res


def baryon_timeslices(dims, q1, q2, q3, n, subset=ALL):
    """out[t, g] of orc_baryon_timeslices; q1, q2, q3: one fermion field each ([V,4,3]; no source contraction) or lists
    of three fields each (one per source colour; eps_{a'b'c'} over them)."""
    def pack(q):
        fields = [_c128(q)] if isinstance(q, np.ndarray) else [_c128(f) for f in q]
        return fields, (ctypes.c_void_p * len(fields))(*[f.ctypes.data for f in fields])
    f1, p1 = pack(q1)
    f2, p2 = pack(q2)
    f3, p3 = pack(q3)
    if not (len(f1) == len(f2) == len(f3)) or len(f1) not in (1, 3):
        raise ValueError("one or three fields per quark")
    out = np.empty((dims[3], 4), dtype=np.complex128)
    _get().orc_baryon_timeslices(_dims(dims), len(f1), p1, p2, p3, int(n), subset, out.ctypes.data)
    return out


def min_eig_vdv(V):
    V = _c128(V)
    return _get().orc_min_eig_vdv(V.ctypes.data)


def staple_site(dims, u, lex, mu, t_dir=3):
    u = _c128(u)
    out = np.empty((3, 3), dtype=np.complex128)
    n = _get().orc_staple_site(_dims(dims), u.ctypes.data, lex, mu, t_dir, out.ctypes.data)
    return out, n


def ape_blend_site(dims, u, lex, mu, alpha, t_dir=3):
    u = _c128(u)
    out = np.empty((3, 3), dtype=np.complex128)
    _get().orc_ape_blend_site(_dims(dims), u.ctypes.data, lex, mu, alpha, t_dir, out.ctypes.data)
    return out


def ape_site(dims, u, lex, mu, alpha, t_dir=3):
    u = _c128(u)
    out = np.empty((3, 3), dtype=np.complex128)
    _get().orc_ape_site(_dims(dims), u.ctypes.data, lex, mu, alpha, t_dir, out.ctypes.data)
    return out


def ape_smear_step(dims, u, alpha, t_dir=3, subset=ALL, u_out=None):
    u = _c128(u)
    out = np.zeros_like(u) if u_out is None else _c128(u_out).copy()
    _get().orc_ape_smear_step(_dims(dims), u.ctypes.data, out.ctypes.data, alpha, t_dir, subset)
    return out


def hop_site(dims, u, psi, lex):
    u, psi = _c128(u), _c128(psi)
    out = np.empty((4, 3), dtype=np.complex128)
    _get().orc_hop_site(_dims(dims), u.ctypes.data, psi.ctypes.data, lex, out.ctypes.data)
    return out


def hop(dims, u, psi, subset=ALL, chi=None):
    u, psi = _c128(u), _c128(psi)
    out = np.zeros_like(psi) if chi is None else _c128(chi).copy()
    _get().orc_hop(_dims(dims), u.ctypes.data, psi.ctypes.data, out.ctypes.data, subset)
    return out


def axpy_hop(dims, a, b, u, psi, subset=ALL, chi=None):
    u, psi = _c128(u), _c128(psi)
    out = np.zeros_like(psi) if chi is None else _c128(chi).copy()
    _get().orc_axpy_hop(_dims(dims), a, b, u.ctypes.data, psi.ctypes.data, out.ctypes.data, subset)
    return out


def smear_hop(dims, a, b, u, psi, t_dir=3, subset=ALL, chi=None):
    """chi = a psi + b sum_{mu != t_dir} [U_mu(x) psi(x+mu) + U_mu(x-mu)^dag psi(x-mu)] (row f2)."""
    u, psi = _c128(u), _c128(psi)
    out = np.zeros_like(psi) if chi is None else _c128(chi).copy()
    _get().orc_smear_hop(_dims(dims), a, b, u.ctypes.data, psi.ctypes.data, out.ctypes.data, t_dir, subset)
    return out


def hop_site_dirs(dims, u, psi, lex, t_dir=3):
    u, psi = _c128(u), _c128(psi)
    out = np.empty((4, 3), dtype=np.complex128)
    _get().orc_hop_site_dirs(_dims(dims), u.ctypes.data, psi.ctypes.data, lex, t_dir, out.ctypes.data)
    return out


def _reals(dims, f):
    return 2 * (f.size // volume(dims))


def norm2(dims, f, subset=ALL):
    f = _c128(f)
    return _get().orc_norm2(_dims(dims), _reals(dims, f), f.ctypes.data, subset)


def inner(dims, a, b, subset=ALL):
    a, b = _c128(a), _c128(b)
    out = np.empty(2)
    _get().orc_inner(_dims(dims), _reals(dims, a), a.ctypes.data, b.ctypes.data, subset,
                     out.ctypes.data)
    return complex(out[0], out[1])


def gamma_matrix(n):
    """Gamma(n) = g0^n0 g1^n1 g2^n2 g3^n3 (DeGrand-Rossi basis), complex [4,4]."""
    out = np.empty((4, 4), dtype=np.complex128)
    _get().orc_gamma_matrix(int(n), out.ctypes.data)
    return out


def inner_timeslices_gamma(dims, a, b, n, subset=ALL):
    """out[t] = sum over x3 = t of a^dag Gamma(n) b (spin matrix on the spin index), complex [L3]."""
    a, b = _c128(a), _c128(b)
    out = np.empty(2 * int(dims[3]))
    _get().orc_inner_timeslices_gamma(_dims(dims), a.ctypes.data, b.ctypes.data, int(n), subset, out.ctypes.data)
    return out[0::2] + 1j * out[1::2]


def axpby(dims, a, x, b, y, subset=ALL, dst=None):
    """dst = a x + b y on the subset (real a, b; any kind)."""
    x, y = _c128(x), _c128(y)
    out = np.zeros_like(x) if dst is None else _c128(dst).copy()
    _get().orc_axpby(_dims(dims), _reals(dims, x), a, x.ctypes.data, b, y.ctypes.data, out.ctypes.data, subset)
    return out


def inner_timeslices(dims, a, b, subset=ALL):
    """out[t] = sum over the sites of time-slice x3 = t of conj(a) . b  (row f3), complex [L3]."""
    a, b = _c128(a), _c128(b)
    out = np.empty(2 * int(dims[3]))
    _get().orc_inner_timeslices(_dims(dims), _reals(dims, a), a.ctypes.data, b.ctypes.data, subset,
                                out.ctypes.data)
    return out[0::2] + 1j * out[1::2]


def sum_field(dims, f, subset=ALL):
    f = _c128(f)
    n = _reals(dims, f)
    out = np.empty(n)
    _get().orc_sum(_dims(dims), n, f.ctypes.data, subset, out.ctypes.data)
    return out[0::2] + 1j * out[1::2]


def hot_path_sample(dims, u, psi, chi, u_out, shifted, a, b, lex_begin, lex_end):
    """One pass of the hot path restricted to the lex sites
    [lex_begin, lex_end) of a large lattice: shift, plaquette, APE step, hop on even then
    odd sites, axpy_hop, norm2, inner.  All arrays complex128 and preallocated; outputs are
    written in place.  Returns (plaquette[3], norm2, inner).  For bench.py's cpu_baseline."""
    lib, d = _get(), _dims(dims)
    lo, hi = int(lex_begin), int(lex_end)
    lib.orc_shift_bytes_range(d, psi.nbytes // volume(dims), psi.ctypes.data, shifted.ctypes.data, 0, 1, ALL, lo, hi)
    plaq = np.empty(3)
    lib.orc_plaquette_range(d, u.ctypes.data, ALL, lo, hi, plaq.ctypes.data)
    lib.orc_ape_smear_step_range(d, u.ctypes.data, u_out.ctypes.data, 0.5, 3, ALL, lo, hi)
    lib.orc_hop_range(d, u.ctypes.data, psi.ctypes.data, chi.ctypes.data, EVEN, lo, hi)
    lib.orc_hop_range(d, u.ctypes.data, psi.ctypes.data, chi.ctypes.data, ODD, lo, hi)
    ip = np.empty(2)
    lib.orc_inner_range(d, 24, psi.ctypes.data, chi.ctypes.data, ALL, lo, hi, ip.ctypes.data)
    lib.orc_axpy_hop_range(d, a, b, u.ctypes.data, psi.ctypes.data, chi.ctypes.data, ALL, lo, hi)
    n2 = lib.orc_norm2_range(d, 24, chi.ctypes.data, ALL, lo, hi)
    return plaq, n2, complex(ip[0], ip[1])
