"""Seeded synthetic lattice inputs (SURVEY.md 8(c) reading A20; recipe in DESIGN.md).

The one module both the oracle side and the CUDA side take their inputs from.
It contains no arithmetic of the method under test: only a counter-based random
number generator and the constructions of the input distributions that
BASELINE.json:configs names.  It imports neither ``oracle`` nor the CUDA package.

All arrays are host, fp64, lexicographic site order (x0 fastest):
    gauge   [V, 4, 3, 3] complex128     spinor [V, 4, 3] complex128
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synth_fields.c")
_LIB = os.path.join(_HERE, "libsynth_fields.so")

BASE_SEED = 11115596  # + config index

# field-id table (A20): one stream per logical input
FID_GAUGE = 1
FID_GAUGE_XFORM = 2
FID_SCALARS = 3
FID_SPINOR0 = 10  # + k for the k-th spinor
FID_MATRIX = 40

# BASELINE.json:configs, dims = (L0, L1, L2, L3) = (x, y, z, t), reading A1
CONFIGS = {
    "C1": (4, 4, 4, 4),
    "C2": (16, 16, 16, 32),
    "C3": (24, 24, 24, 64),
    "C4": (32, 32, 32, 64),
    "C5": (48, 48, 48, 96),
}


def build(force: bool = False) -> str:
    """Compile the generator with gcc (idempotent)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


_lib = None


def _get():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64, sz, dbl, ptr = ctypes.c_uint64, ctypes.c_size_t, ctypes.c_double, ctypes.c_void_p
        lib.syn_normal_complex.argtypes = [u64, u64, sz, ptr]
        lib.syn_uniform.argtypes = [u64, u64, sz, dbl, dbl, ptr]
        lib.syn_su3_hot.argtypes = [u64, u64, sz, ptr]
        lib.syn_su3_warm.argtypes = [u64, u64, sz, dbl, ptr]
        for f in (lib.syn_normal_complex, lib.syn_uniform, lib.syn_su3_hot, lib.syn_su3_warm):
            f.restype = None
        _lib = lib
    return _lib


def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def gauge_hot(dims, seed: int, field_id: int = FID_GAUGE) -> np.ndarray:
    """Haar-like random SU(3) links, [V,4,3,3] complex128."""
    V = volume(dims)
    out = np.empty((V, 4, 3, 3), dtype=np.complex128)
    _get().syn_su3_hot(seed, field_id, V * 4, out.ctypes.data)
    return out


def gauge_warm(dims, seed: int, eps: float = 0.2, field_id: int = FID_GAUGE) -> np.ndarray:
    """U = exp(i eps H), H traceless Hermitian Gaussian; [V,4,3,3] complex128."""
    V = volume(dims)
    out = np.empty((V, 4, 3, 3), dtype=np.complex128)
    _get().syn_su3_warm(seed, field_id, V * 4, float(eps), out.ctypes.data)
    return out


def gauge_unit(dims) -> np.ndarray:
    V = volume(dims)
    out = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    out[:, :, 0, 0] = out[:, :, 1, 1] = out[:, :, 2, 2] = 1.0
    return out


def su3_site_field(dims, seed: int, field_id: int = FID_GAUGE_XFORM) -> np.ndarray:
    """One Haar-like SU(3) per site (a gauge transformation g(x)), [V,3,3]."""
    V = volume(dims)
    out = np.empty((V, 3, 3), dtype=np.complex128)
    _get().syn_su3_hot(seed, field_id, V, out.ctypes.data)
    return out


def spinor(dims, seed: int, k: int = 0) -> np.ndarray:
    """4 spin x 3 colour complex, i.i.d. N(0,1) parts, [V,4,3] complex128."""
    V = volume(dims)
    out = np.empty((V, 4, 3), dtype=np.complex128)
    _get().syn_normal_complex(seed, FID_SPINOR0 + k, V * 12, out.ctypes.data)
    return out


def color_matrix(dims, seed: int, field_id: int = FID_MATRIX) -> np.ndarray:
    """General complex 3x3 per site (for shift / reduction tests), [V,3,3]."""
    V = volume(dims)
    out = np.empty((V, 3, 3), dtype=np.complex128)
    _get().syn_normal_complex(seed, field_id, V * 9, out.ctypes.data)
    return out


def scalars_ab(seed: int) -> tuple[float, float]:
    """Real a, b ~ U(-1,1) for chi = a psi + b hop(psi) (BASELINE.json:configs[2])."""
    out = np.empty(2, dtype=np.float64)
    _get().syn_uniform(seed, FID_SCALARS, 2, -1.0, 1.0, out.ctypes.data)
    return float(out[0]), float(out[1])


def round_to(arr: np.ndarray, prec: str) -> np.ndarray:
    """Round an fp64 complex array once to the field precision (A13); returns the
    host array in the element type the C-ABI upload expects."""
    if prec == "f64":
        return np.ascontiguousarray(arr, dtype=np.complex128)
    if prec == "f32":
        return np.ascontiguousarray(arr.astype(np.complex64))
    raise ValueError(prec)
