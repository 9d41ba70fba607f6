"""ctypes binding of include/qdp_b200.h: argument marshalling only.

Function names are those of the C ABI.  Handles are small Python objects that own
the C handle (and, for fields, the torch tensor that provides the device memory).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

__all__ = [
    "QdpError", "Lattice", "Field", "LIB_PATH", "DECLARED_SYMBOLS",
    "QDP_ALL", "QDP_EVEN", "QDP_ODD", "QDP_F32", "QDP_F64",
    "QDP_COLOR_MATRIX", "QDP_GAUGE", "QDP_FERMION", "QDP_COMPLEX",
    "qdp_lattice_create", "qdp_lattice_destroy", "qdp_lattice_set_stream", "qdp_lattice_set_sweep_slab", "qdp_lattice_set_staged", "qdp_lattice_volume",
    "qdp_lattice_neighbor_table", "qdp_lattice_parity_mask", "qdp_lattice_sync",
    "qdp_field_alloc", "qdp_field_wrap", "qdp_field_free", "qdp_field_bytes",
    "qdp_field_upload", "qdp_field_download", "qdp_field_copy",
    "qdp_shift", "qdp_plaquette", "qdp_ape_smear_step", "qdp_hop", "qdp_axpy_hop", "qdp_smear_hop", "qdp_inner_timeslices", "qdp_inner_timeslices_gamma", "qdp_reunitarize", "qdp_project_max_retr", "qdp_baryon_timeslices", "qdp_matmul", "qdp_matvec", "qdp_axpby", "qdp_expr_plaquette", "qdp_expr_staple", "qdp_expr_ape_blend", "qdp_expr_trace_mul", "qdp_expr_sum_trace_mul", "qdp_expr_jit_kind", "qdp_expr_jit_compile", "qdp_expr_jit_assign", "qdp_expr_jit_sum", "qdp_expr_jit_compilations", "QDP_REUNIT_POLAR", "QDP_REUNIT_GRAM_SCHMIDT",
    "qdp_norm2", "qdp_inner", "qdp_sum", "qdp_sum_noalloc", "qdp_kernel_launch_count", "qdp_last_error",
    "qdp_set_allocator", "field_from_host", "field_to_host",
    "qdp_field_timeslice_bytes", "qdp_field_get_timeslice", "qdp_field_set_timeslice",
    "Pool", "Cached", "qdp_pool_create", "qdp_pool_destroy", "qdp_pool_alloc", "qdp_pool_free", "qdp_pool_stats",
    "qdp_pool_hook_alloc", "qdp_pool_hook_free", "qdp_pool_eviction_log", "qdp_cache_register", "qdp_cache_acquire",
    "qdp_cache_release", "qdp_cache_unregister", "qdp_cache_is_resident", "qdp_cache_id",
]

QDP_ALL, QDP_EVEN, QDP_ODD = 0, 1, 2
QDP_F32, QDP_F64 = 0, 1
QDP_COLOR_MATRIX, QDP_GAUGE, QDP_FERMION, QDP_COMPLEX = 0, 1, 2, 3
_NCOMP = {QDP_COLOR_MATRIX: 9, QDP_GAUGE: 36, QDP_FERMION: 12, QDP_COMPLEX: 1}
_SHAPE = {QDP_COLOR_MATRIX: (3, 3), QDP_GAUGE: (4, 3, 3), QDP_FERMION: (4, 3), QDP_COMPLEX: ()}

# QDP_B200_LIB selects another build of the same library (e.g. a debug or tuning build)
LIB_PATH = os.environ.get("QDP_B200_LIB") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "libqdp_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_1111_5596_b200.build` "
        "(there is no CPU fallback)")
_lib = ctypes.CDLL(LIB_PATH)

_P, _I, _D, _Z = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
_PP = ctypes.POINTER(ctypes.c_void_p)
ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
FREE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)

# every symbol include/qdp_b200.h declares: (argtypes, restype)
DECLARED_SYMBOLS = {
    "qdp_lattice_create": ([_P, _I, _PP], _I),
    "qdp_lattice_destroy": ([_P], _I),
    "qdp_lattice_set_stream": ([_P, _P], _I),
    "qdp_lattice_set_sweep_slab": ([_P, _I], _I),
    "qdp_lattice_set_staged": ([_P, _I], _I),
    "qdp_set_allocator": ([_P, _P, _P], _I),
    "qdp_lattice_neighbor_table": ([_P, _I, _I, _P], _I),
    "qdp_lattice_parity_mask": ([_P, _P], _I),
    "qdp_lattice_volume": ([_P, ctypes.POINTER(ctypes.c_int64)], _I),
    "qdp_field_alloc": ([_P, _I, _I, _PP], _I),
    "qdp_field_wrap": ([_P, _I, _I, _P, _Z, _PP], _I),
    "qdp_field_free": ([_P], _I),
    "qdp_field_bytes": ([_P, _I, _I, ctypes.POINTER(_Z)], _I),
    "qdp_field_upload": ([_P, _P], _I),
    "qdp_field_download": ([_P, _P], _I),
    "qdp_field_copy": ([_P, _P], _I),
    "qdp_shift": ([_P, _P, _I, _I, _I], _I),
    "qdp_plaquette": ([_P, _I, _P], _I),
    "qdp_ape_smear_step": ([_P, _P, _D, _I, _I], _I),
    "qdp_hop": ([_P, _P, _P, _I], _I),
    "qdp_axpy_hop": ([_P, _D, _D, _P, _P, _I, _P], _I),
    "qdp_smear_hop": ([_P, _D, _D, _P, _P, _I, _I, _P], _I),
    "qdp_inner_timeslices": ([_P, _P, _I, _P], _I),
    "qdp_inner_timeslices_gamma": ([_P, _P, _I, _I, _P], _I),
    "qdp_reunitarize": ([_P, _P, _I, _I], _I),
    "qdp_axpby": ([_P, _D, _P, _D, _P, _I, _P], _I),
    "qdp_matvec": ([_P, _P, _I, _I, _P, _I, _I, _I], _I),
    "qdp_matmul": ([_P, _I, _P, _I, _I, _P, _I, _I, _I, _I, _I], _I),
    "qdp_project_max_retr": ([_P, _P, _I, _I], _I),
    "qdp_baryon_timeslices": ([_PP, _PP, _PP, _I, _I, _I, _P], _I),
    "qdp_expr_plaquette": ([_P, _I, ctypes.POINTER(_D)], _I),
    "qdp_expr_staple": ([_P, _P, _I, _I, _I], _I),
    "qdp_expr_ape_blend": ([_P, _P, _I, _D, _I, _I], _I),
    "qdp_expr_trace_mul": ([_P, _P, _I, _I, _P, _I, _I, _I, _I, _I], _I),
    "qdp_expr_sum_trace_mul": ([_P, _I, _I, _P, _I, _I, _I, _I, _I, ctypes.POINTER(_D)], _I),
    "qdp_expr_jit_kind": ([ctypes.c_char_p, ctypes.POINTER(_I), _I, _I, ctypes.POINTER(_I)], _I),
    "qdp_expr_jit_compile": ([ctypes.c_char_p, ctypes.POINTER(_I), _I, _I, _I, _I, ctypes.POINTER(_Z)], _I),
    "qdp_expr_jit_assign": ([_P, _I, ctypes.c_char_p, _PP, _I, ctypes.POINTER(_D), _I, _I], _I),
    "qdp_expr_jit_sum": ([ctypes.c_char_p, _PP, _I, ctypes.POINTER(_D), _I, _I, ctypes.POINTER(_D)], _I),
    "qdp_expr_jit_compilations": ([], ctypes.c_int64),
    "qdp_norm2": ([_P, _I, _P], _I),
    "qdp_inner": ([_P, _P, _I, _P], _I),
    "qdp_sum": ([_P, _I, _P], _I),
    "qdp_sum_noalloc": ([ctypes.POINTER(ctypes.c_int), _I, _I, _P, _Z, _I, _P, _P], _I),
    "qdp_lattice_sync": ([_P], _I),
    "qdp_kernel_launch_count": ([], ctypes.c_int64),
    "qdp_last_error": ([], ctypes.c_char_p),
    "qdp_field_timeslice_bytes": ([_P, ctypes.POINTER(_Z)], _I),
    "qdp_field_get_timeslice": ([_P, _I, _P, _Z], _I),
    "qdp_field_set_timeslice": ([_P, _I, _P, _Z, _I], _I),
    "qdp_pool_create": ([_I, _Z, _PP], _I),
    "qdp_pool_destroy": ([_P], _I),
    "qdp_pool_alloc": ([_P, _Z, _PP], _I),
    "qdp_pool_free": ([_P, _P], _I),
    "qdp_pool_stats": ([_P, ctypes.POINTER(_Z)], _I),
    "qdp_pool_hook_alloc": ([_Z, _P], _P),
    "qdp_pool_hook_free": ([_P, _P], None),
    "qdp_cache_register": ([_P, _P, _Z, _PP], _I),
    "qdp_cache_acquire": ([_P, _I, _PP], _I),
    "qdp_cache_release": ([_P], _I),
    "qdp_cache_unregister": ([_P], _I),
    "qdp_cache_is_resident": ([_P], _I),
    "qdp_cache_id": ([_P], ctypes.c_int64),
    "qdp_pool_eviction_log": ([_P, ctypes.POINTER(ctypes.c_int64), _I, ctypes.POINTER(_I)], _I),
}
for _name, (_args, _res) in DECLARED_SYMBOLS.items():
    _f = getattr(_lib, _name)
    _f.argtypes, _f.restype = _args, _res


class QdpError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"qdp error {code}: {msg}")
        self.code = code


def _check(rc: int) -> None:
    if rc != 0:
        raise QdpError(rc, _lib.qdp_last_error().decode(errors="replace"))


def qdp_last_error() -> str:
    return _lib.qdp_last_error().decode(errors="replace")


def qdp_kernel_launch_count() -> int:
    return int(_lib.qdp_kernel_launch_count())


class Lattice:
    def __init__(self, handle: int, dims, device: int):
        self.handle, self.dims, self.device = handle, tuple(int(d) for d in dims), device
        self.volume = int(np.prod(self.dims))

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:      # _lib is None during interpreter shutdown
            _lib.qdp_lattice_destroy(h)


class Field:
    def __init__(self, handle: int, lat: Lattice, kind: int, prec: int, storage=None):
        self.handle, self.lat, self.kind, self.prec, self.storage = handle, lat, kind, prec, storage

    @property
    def host_dtype(self):
        return np.complex128 if self.prec == QDP_F64 else np.complex64

    @property
    def host_shape(self):
        return (self.lat.volume,) + _SHAPE[self.kind]

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:
            _lib.qdp_field_free(h)
        self.storage = None


def qdp_lattice_create(dims, device: int = 0) -> Lattice:
    out = ctypes.c_void_p()
    _check(_lib.qdp_lattice_create((ctypes.c_int * 4)(*[int(d) for d in dims]), device, ctypes.byref(out)))
    return Lattice(out.value, dims, device)


def qdp_lattice_destroy(lat: Lattice) -> None:
    h, lat.handle = lat.handle, None
    if h:
        _check(_lib.qdp_lattice_destroy(h))


def qdp_lattice_set_stream(lat: Lattice, cuda_stream: int | None) -> None:
    _check(_lib.qdp_lattice_set_stream(lat.handle, cuda_stream))


def qdp_lattice_set_sweep_slab(lat: Lattice, x2_extent: int) -> None:
    _check(_lib.qdp_lattice_set_sweep_slab(lat.handle, int(x2_extent)))


def qdp_lattice_set_staged(lat: Lattice, on: bool) -> None:
    _check(_lib.qdp_lattice_set_staged(lat.handle, int(bool(on))))


def qdp_lattice_sync(lat: Lattice) -> None:
    _check(_lib.qdp_lattice_sync(lat.handle))


def qdp_lattice_volume(lat: Lattice) -> int:
    out = ctypes.c_int64()
    _check(_lib.qdp_lattice_volume(lat.handle, ctypes.byref(out)))
    return out.value


def qdp_lattice_neighbor_table(lat: Lattice, mu: int, sign: int) -> np.ndarray:
    out = np.empty(lat.volume, dtype=np.int32)
    _check(_lib.qdp_lattice_neighbor_table(lat.handle, mu, sign, out.ctypes.data))
    return out


def qdp_lattice_parity_mask(lat: Lattice) -> np.ndarray:
    out = np.empty(lat.volume, dtype=np.uint8)
    _check(_lib.qdp_lattice_parity_mask(lat.handle, out.ctypes.data))
    return out


def qdp_set_allocator(alloc, free_, ctx=None) -> None:
    """alloc/free_: ctypes callbacks of type ALLOC_FN / FREE_FN (keep them alive), or None."""
    _check(_lib.qdp_set_allocator(ctypes.cast(alloc, _P) if alloc else None,
                                  ctypes.cast(free_, _P) if free_ else None, ctx))


def qdp_field_bytes(lat: Lattice, kind: int, prec: int) -> int:
    out = _Z()
    _check(_lib.qdp_field_bytes(lat.handle, kind, prec, ctypes.byref(out)))
    return out.value


def qdp_field_wrap(lat: Lattice, kind: int, prec: int, dev_ptr: int, nbytes: int, storage=None) -> Field:
    out = ctypes.c_void_p()
    _check(_lib.qdp_field_wrap(lat.handle, kind, prec, dev_ptr, nbytes, ctypes.byref(out)))
    return Field(out.value, lat, kind, prec, storage)


def qdp_field_alloc(lat: Lattice, kind: int, prec: int, use_torch: bool = True) -> Field:
    """Device memory comes from PyTorch's caching allocator (a uint8 tensor wrapped with
    qdp_field_wrap); use_torch=False lets the library allocate (qdp_field_alloc in C)."""
    if use_torch:
        import torch
        nbytes = qdp_field_bytes(lat, kind, prec)
        buf = torch.empty(nbytes, dtype=torch.uint8, device=f"cuda:{lat.device}")
        return qdp_field_wrap(lat, kind, prec, buf.data_ptr(), nbytes, storage=buf)
    out = ctypes.c_void_p()
    _check(_lib.qdp_field_alloc(lat.handle, kind, prec, ctypes.byref(out)))
    return Field(out.value, lat, kind, prec)


def qdp_field_free(f: Field) -> None:
    h, f.handle = f.handle, None
    if h:
        _check(_lib.qdp_field_free(h))
    f.storage = None


def _host_ptr(f: Field, host) -> int:
    """host: numpy array (complex64/128, C-contiguous) or a CPU torch tensor (e.g. pinned)."""
    if isinstance(host, np.ndarray):
        if host.dtype != f.host_dtype or not host.flags.c_contiguous:
            raise TypeError(f"host array must be C-contiguous {f.host_dtype}")
        if host.size != int(np.prod(f.host_shape)):
            raise ValueError("host array has the wrong number of elements")
        return host.ctypes.data
    nbytes = host.numel() * host.element_size()
    want = int(np.prod(f.host_shape)) * np.dtype(f.host_dtype).itemsize    # host AoS size: V * ncomp complex numbers
    if nbytes != want or not host.is_contiguous() or host.is_cuda:
        raise ValueError(f"host tensor must be a contiguous CPU tensor of {want} bytes (V x components, array of structures)")
    return host.data_ptr()


def qdp_field_upload(f: Field, host) -> None:
    _check(_lib.qdp_field_upload(f.handle, _host_ptr(f, host)))


def qdp_field_download(f: Field, host=None):
    if host is None:
        host = np.empty(f.host_shape, dtype=f.host_dtype)
    _check(_lib.qdp_field_download(f.handle, _host_ptr(f, host)))
    return host


def qdp_field_copy(dst: Field, src: Field) -> None:
    _check(_lib.qdp_field_copy(dst.handle, src.handle))


def field_from_host(lat: Lattice, kind: int, host: np.ndarray) -> Field:
    prec = QDP_F64 if host.dtype == np.complex128 else QDP_F32
    f = qdp_field_alloc(lat, kind, prec)
    qdp_field_upload(f, np.ascontiguousarray(host))
    return f


def field_to_host(f: Field) -> np.ndarray:
    return qdp_field_download(f)


def qdp_shift(dst: Field, src: Field, mu: int, sign: int, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_shift(dst.handle, src.handle, mu, sign, subset))


def qdp_plaquette(u: Field, subset: int = QDP_ALL) -> np.ndarray:
    out = np.empty(3)
    _check(_lib.qdp_plaquette(u.handle, subset, out.ctypes.data))
    return out


def qdp_ape_smear_step(u_out: Field, u_in: Field, alpha: float, t_dir: int = 3, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_ape_smear_step(u_out.handle, u_in.handle, float(alpha), t_dir, subset))


QDP_REUNIT_POLAR, QDP_REUNIT_GRAM_SCHMIDT = 0, 1


def qdp_matvec(chi: Field, a: Field, slot_a: int, adj_a: bool, psi: Field, mu: int = -1, sign: int = 1,
               subset: int = QDP_ALL) -> None:
    """chi(x) = op(a[slot_a])(x) psi(x + sign*mu); mu = -1: no shift."""
    _check(_lib.qdp_matvec(chi.handle, a.handle, slot_a, int(bool(adj_a)), psi.handle, mu, sign, subset))


def qdp_matmul(dst: Field, slot_d: int, a: Field, slot_a: int, adj_a: bool, b: Field, slot_b: int, adj_b: bool,
               mu: int = -1, sign: int = 1, subset: int = QDP_ALL) -> None:
    """dst[slot_d](x) = op(a[slot_a])(x) @ op(b[slot_b])(x + sign*mu); mu = -1: no shift."""
    _check(_lib.qdp_matmul(dst.handle, slot_d, a.handle, slot_a, int(bool(adj_a)), b.handle, slot_b, int(bool(adj_b)),
                           mu, sign, subset))


def qdp_expr_plaquette(u: Field, subset: int = QDP_ALL) -> np.ndarray:
    """The plaquette as one expression kernel (row f1); same normalisation as qdp_plaquette."""
    out = (_D * 3)()
    _check(_lib.qdp_expr_plaquette(u.handle, subset, out))
    return np.array(out[:], dtype=np.float64)


def qdp_expr_staple(dst: Field, u: Field, mu: int, t_dir: int = 3, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_expr_staple(dst.handle, u.handle, mu, t_dir, subset))


def qdp_expr_ape_blend(dst: Field, u: Field, mu: int, alpha: float, t_dir: int = 3, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_expr_ape_blend(dst.handle, u.handle, mu, float(alpha), t_dir, subset))


def qdp_expr_trace_mul(dst: Field, a: Field, slot_a: int, adj_a: bool, b: Field, slot_b: int, adj_b: bool,
                       mu: int = -1, sign: int = 1, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_expr_trace_mul(dst.handle, a.handle, slot_a, int(bool(adj_a)), b.handle, slot_b, int(bool(adj_b)),
                                   mu, sign, subset))


def qdp_expr_sum_trace_mul(a: Field, slot_a: int, adj_a: bool, b: Field, slot_b: int, adj_b: bool,
                           mu: int = -1, sign: int = 1, subset: int = QDP_ALL) -> complex:
    out = (_D * 2)()
    _check(_lib.qdp_expr_sum_trace_mul(a.handle, slot_a, int(bool(adj_a)), b.handle, slot_b, int(bool(adj_b)), mu, sign,
                                       subset, out))
    return complex(out[0], out[1])


def qdp_expr_jit_kind(expr: str, field_kinds, nscalars: int = 0) -> int:
    """Host-only type check of a run-time expression: 0 matrix, 1 complex, 2 real (QdpError on a syntax / kind error)."""
    kinds = (_I * max(1, len(field_kinds)))(*field_kinds)
    out = _I()
    _check(_lib.qdp_expr_jit_kind(expr.encode(), kinds, len(field_kinds), nscalars, ctypes.byref(out)))
    return out.value


def qdp_expr_jit_compile(expr: str, field_kinds, nscalars: int = 0, prec: int = QDP_F64, sum_: bool = False) -> int:
    """Compile (NVRTC, no device needed) the kernel of the expression into the cache; returns the size of its image."""
    kinds = (_I * max(1, len(field_kinds)))(*field_kinds)
    out = _Z()
    _check(_lib.qdp_expr_jit_compile(expr.encode(), kinds, len(field_kinds), nscalars, prec, int(bool(sum_)), ctypes.byref(out)))
    return out.value


def _jit_args(fields, scalars):
    fp = (ctypes.c_void_p * len(fields))(*[f.handle for f in fields])
    sc = (_D * max(1, len(scalars)))(*[float(x) for x in scalars])
    return fp, sc


def qdp_expr_jit_assign(dst: Field, slot_d: int, expr: str, fields, scalars=(), subset: int = QDP_ALL) -> None:
    fp, sc = _jit_args(fields, scalars)
    _check(_lib.qdp_expr_jit_assign(dst.handle, slot_d, expr.encode(), fp, len(fields), sc, len(scalars), subset))


def qdp_expr_jit_sum(expr: str, fields, scalars=(), subset: int = QDP_ALL) -> complex:
    fp, sc = _jit_args(fields, scalars)
    out = (_D * 2)()
    _check(_lib.qdp_expr_jit_sum(expr.encode(), fp, len(fields), sc, len(scalars), subset, out))
    return complex(out[0], out[1])


def qdp_expr_jit_compilations() -> int:
    return int(_lib.qdp_expr_jit_compilations())


def qdp_reunitarize(u_out: Field, u_in: Field, method: int = QDP_REUNIT_POLAR, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_reunitarize(u_out.handle, u_in.handle, int(method), subset))


def qdp_project_max_retr(u_out: Field, u_in: Field, iterations: int, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_project_max_retr(u_out.handle, u_in.handle, int(iterations), subset))


def qdp_baryon_timeslices(q1, q2, q3, n: int, subset: int = QDP_ALL) -> np.ndarray:
    """q1, q2, q3: a Field each (no source contraction) or a sequence of three Fields each (one per source colour).
    Returns out[t, g], complex, [L3, 4]."""
    def pack(q):
        fields = [q] if isinstance(q, Field) else list(q)
        return fields, (ctypes.c_void_p * len(fields))(*[f.handle for f in fields])
    f1, p1 = pack(q1)
    f2, p2 = pack(q2)
    f3, p3 = pack(q3)
    if not (len(f1) == len(f2) == len(f3)):
        raise ValueError("the same number of fields (1 or 3) per quark")
    L3 = f1[0].lat.dims[3]
    out = np.empty(8 * L3)
    _check(_lib.qdp_baryon_timeslices(p1, p2, p3, len(f1), int(n), subset, out.ctypes.data))
    return (out[0::2] + 1j * out[1::2]).reshape(L3, 4)


def qdp_hop(chi: Field, u: Field, psi: Field, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_hop(chi.handle, u.handle, psi.handle, subset))


def qdp_axpy_hop(chi: Field, a: float, b: float, u: Field, psi: Field, subset: int = QDP_ALL,
                 want_norm2: bool = False):
    if want_norm2:
        out = ctypes.c_double()
        _check(_lib.qdp_axpy_hop(chi.handle, float(a), float(b), u.handle, psi.handle, subset, ctypes.addressof(out)))
        return out.value
    _check(_lib.qdp_axpy_hop(chi.handle, float(a), float(b), u.handle, psi.handle, subset, None))
    return None


def qdp_smear_hop(chi: Field, a: float, b: float, u: Field, psi: Field, t_dir: int = 3, subset: int = QDP_ALL,
                  want_norm2: bool = False):
    out = ctypes.c_double()
    _check(_lib.qdp_smear_hop(chi.handle, float(a), float(b), u.handle, psi.handle, int(t_dir), subset,
                              ctypes.addressof(out) if want_norm2 else None))
    return out.value if want_norm2 else None


def qdp_axpby(dst: Field, a: float, x: Field, b: float, y: Field, subset: int = QDP_ALL, want_norm2: bool = False):
    out = ctypes.c_double()
    _check(_lib.qdp_axpby(dst.handle, float(a), x.handle, float(b), y.handle, subset,
                          ctypes.addressof(out) if want_norm2 else None))
    return out.value if want_norm2 else None


def qdp_norm2(f: Field, subset: int = QDP_ALL) -> float:
    out = ctypes.c_double()
    _check(_lib.qdp_norm2(f.handle, subset, ctypes.addressof(out)))
    return out.value


def qdp_inner(a: Field, b: Field, subset: int = QDP_ALL) -> complex:
    out = np.empty(2)
    _check(_lib.qdp_inner(a.handle, b.handle, subset, out.ctypes.data))
    return complex(out[0], out[1])


def qdp_inner_timeslices(a: Field, b: Field, subset: int = QDP_ALL) -> np.ndarray:
    """complex [L3]: sum over the sites of each time-slice x3 = t of conj(a) . b"""
    out = np.empty(2 * int(a.lat.dims[3]), dtype=np.float64)
    _check(_lib.qdp_inner_timeslices(a.handle, b.handle, subset, out.ctypes.data))
    return out[0::2] + 1j * out[1::2]


def qdp_inner_timeslices_gamma(a: Field, b: Field, n: int, subset: int = QDP_ALL) -> np.ndarray:
    """complex [L3]: sum over the sites of each time-slice of a^dag Gamma(n) b (Gamma(15) = gamma_5)"""
    out = np.empty(2 * int(a.lat.dims[3]), dtype=np.float64)
    _check(_lib.qdp_inner_timeslices_gamma(a.handle, b.handle, int(n), subset, out.ctypes.data))
    return out[0::2] + 1j * out[1::2]


def qdp_sum(f: Field, subset: int = QDP_ALL) -> np.ndarray:
    out = np.empty(2 * _NCOMP[f.kind])
    _check(_lib.qdp_sum(f.handle, subset, out.ctypes.data))
    return (out[0::2] + 1j * out[1::2]).reshape(_SHAPE[f.kind])


def qdp_sum_noalloc(dims, ncomp: int, prec: int, field_dev: int, nbytes: int, subset: int, out_dev: int,
                    cuda_stream: int | None = None) -> None:
    """qdp_sum without a lattice handle and without any allocation, for callers that may not call cudaMalloc
    (include/qdp_b200.h).  field_dev / out_dev are raw device addresses on the current device (out_dev: 2 * ncomp
    doubles); the call is asynchronous on cuda_stream.  Calls that overlap on the GPU race on the shared scratch."""
    _check(_lib.qdp_sum_noalloc((ctypes.c_int * 4)(*[int(d) for d in dims]), int(ncomp), int(prec), field_dev,
                                int(nbytes), int(subset), out_dev, cuda_stream))


def qdp_field_timeslice_bytes(f: Field) -> int:
    out = _Z()
    _check(_lib.qdp_field_timeslice_bytes(f.handle, ctypes.byref(out)))
    return out.value


def qdp_field_get_timeslice(f: Field, t: int, dev_ptr: int, nbytes: int) -> None:
    _check(_lib.qdp_field_get_timeslice(f.handle, int(t), dev_ptr, int(nbytes)))


def qdp_field_set_timeslice(f: Field, t: int, dev_ptr: int, nbytes: int, subset: int = QDP_ALL) -> None:
    _check(_lib.qdp_field_set_timeslice(f.handle, int(t), dev_ptr, int(nbytes), subset))


# ---- row f4: device memory pool and LRU residency manager (csrc/pool.cu) -----------------------
class Pool:
    def __init__(self, handle: int, device: int, nbytes: int):
        self.handle, self.device, self.nbytes = handle, device, nbytes


class Cached:
    def __init__(self, handle: int, pool: Pool, host, nbytes: int):
        self.handle, self.pool, self.host, self.nbytes = handle, pool, host, nbytes    # `host` keeps the buffer alive


def qdp_pool_create(device: int, nbytes: int) -> Pool:
    """device = -1: address-range-only pool (allocator and eviction policy without a GPU)."""
    out = ctypes.c_void_p()
    _check(_lib.qdp_pool_create(int(device), int(nbytes), ctypes.byref(out)))
    return Pool(out.value, device, nbytes)


def qdp_pool_destroy(pool: Pool) -> None:
    if pool.handle:
        _check(_lib.qdp_pool_destroy(pool.handle))     # fails (and keeps the pool) while objects are registered
        pool.handle = None


def qdp_pool_alloc(pool: Pool, nbytes: int) -> int:
    out = ctypes.c_void_p()
    _check(_lib.qdp_pool_alloc(pool.handle, int(nbytes), ctypes.byref(out)))
    return out.value


def qdp_pool_free(pool: Pool, ptr: int) -> None:
    _check(_lib.qdp_pool_free(pool.handle, ptr))


def qdp_pool_stats(pool: Pool) -> dict:
    out = (_Z * 4)()
    _check(_lib.qdp_pool_stats(pool.handle, out))
    return {"capacity": out[0], "in_use": out[1], "largest_free": out[2], "free_blocks": out[3]}


def qdp_pool_hook_alloc():
    """The pool's qdp_set_allocator-compatible entry points as raw function addresses: (alloc, free)."""
    return ctypes.cast(_lib.qdp_pool_hook_alloc, _P).value, ctypes.cast(_lib.qdp_pool_hook_free, _P).value


def qdp_pool_hook_free():
    return qdp_pool_hook_alloc()[1]


def qdp_pool_eviction_log(pool: Pool) -> list:
    n = _I()
    _check(_lib.qdp_pool_eviction_log(pool.handle, None, 0, ctypes.byref(n)))
    ids = (ctypes.c_int64 * max(1, n.value))()
    _check(_lib.qdp_pool_eviction_log(pool.handle, ids, n.value, ctypes.byref(n)))
    return [int(ids[i]) for i in range(n.value)]


def qdp_cache_register(pool: Pool, host, nbytes: int | None = None) -> Cached:
    """host: a (pinned) CPU torch tensor or a numpy array holding the object's bytes, or None with an explicit size
    for an address-range-only pool."""
    if host is None:
        ptr, size = None, int(nbytes)
    elif isinstance(host, np.ndarray):
        ptr, size = host.ctypes.data, host.nbytes
    else:
        ptr, size = host.data_ptr(), host.numel() * host.element_size()
    out = ctypes.c_void_p()
    _check(_lib.qdp_cache_register(pool.handle, ptr, size, ctypes.byref(out)))
    return Cached(out.value, pool, host, size)


def qdp_cache_acquire(c: Cached, for_write: bool = False) -> int:
    out = ctypes.c_void_p()
    _check(_lib.qdp_cache_acquire(c.handle, int(bool(for_write)), ctypes.byref(out)))
    return out.value


def qdp_cache_release(c: Cached) -> None:
    _check(_lib.qdp_cache_release(c.handle))


def qdp_cache_unregister(c: Cached) -> None:
    if c.handle:
        _check(_lib.qdp_cache_unregister(c.handle))     # a refused call ("still acquired") keeps the handle, so it can be retried
        c.handle = None


def qdp_cache_is_resident(c: Cached) -> bool:
    return bool(_lib.qdp_cache_is_resident(c.handle))


def qdp_cache_id(c: Cached) -> int:
    return int(_lib.qdp_cache_id(c.handle))
