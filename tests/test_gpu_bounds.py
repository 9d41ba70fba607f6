"""Memory-safety evidence without compute-sanitizer (closed on this GPU pool): the small-lattice parity suite is run
against libqdp_b200_bc.so, the same library compiled with -DQDP_BOUNDS_CHECK, in which every site address the kernels
form is validated on the device (su3.cuh: site_ptr_checked) and a violation prints a QDP_BOUNDS line."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SELFTEST = """
import ctypes
import paper_1111_5596_b200 as q
from paper_1111_5596_b200 import binding
lat = q.qdp_lattice_create((2, 2, 2, 2))
f = q.qdp_field_alloc(lat, q.QDP_FERMION, q.QDP_F64)
fn = binding._lib.qdp_bc_selftest
fn.argtypes, fn.restype = [ctypes.c_void_p], ctypes.c_int
assert fn(f.handle) == 0
q.qdp_lattice_sync(lat)
print("selftest done", binding.LIB_PATH)
"""


def test_small_lattice_suite_under_the_bounds_checked_build():
    from paper_1111_5596_b200.build import BC_LIB, build
    build(bounds_check=True)
    env = dict(os.environ, QDP_B200_LIB=BC_LIB, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""))
    # the checker fires on deliberately wrong addresses (and only there)
    r = subprocess.run([sys.executable, "-c", SELFTEST], capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "libqdp_b200_bc.so" in r.stdout and r.stdout.count("QDP_BOUNDS") == 3, r.stdout
    # every op, subset, kind and precision on the tiny, ragged and anisotropic lattices (C2 left out: time); the run-time
    # expression kernels are compiled by NVRTC with the same check
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join("tests", "test_gpu_parity.py"), os.path.join("tests", "test_gpu_jit.py"),
                        "-x", "-q", "-s", "-m", "gpu",
                        "-k", "not dims5", "-p", "no:cacheprovider"],
                       capture_output=True, text=True, env=env, cwd=ROOT, timeout=3000)
    out = r.stdout + r.stderr
    assert r.returncode == 0, out[-4000:]
    assert " passed" in out and "QDP_BOUNDS" not in out, out[-4000:]
