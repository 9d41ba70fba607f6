"""Build libqdp_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1111_5596_b200.build [--force] [--verbose] [--bounds-check]
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libqdp_b200.so")
PROBE_LIB = os.path.join(HERE, "libqdp_probe.so")   # bench-only peak probes (csrc/probe.cu), not part of the C ABI
SOURCES = ["api.cu", "layout.cu", "shift.cu", "reduce.cu", "hop.cu", "plaquette.cu", "plaquette_tma.cu", "ape.cu", "reunit.cu", "matmul.cu", "expr.cu", "baryon.cu", "pool.cu", "jit.cu", "noalloc.cu"]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _deps_mtime() -> float:
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hdrs.append(os.path.join(os.path.dirname(HERE), "include", "qdp_b200.h"))
    return max(os.path.getmtime(h) for h in hdrs)


JIT_HEADERS = ["geom.cuh", "reduce.cuh", "su3.cuh", "expr.cuh"]   # what a run-time expression kernel includes (csrc/jit.cu)


def _write_jit_headers(obj_dir: str) -> None:
    """jit_headers.inc: the headers above as string literals, so that NVRTC needs no file at run time."""
    parts = []
    for h in JIT_HEADERS:
        text = open(os.path.join(CSRC, h)).read()
        assert ')QDPHDR"' not in text
        parts.append(f'static const char kJitHdr_{h.split(".")[0]}[] = R"QDPHDR(' + text + ')QDPHDR";\n')
    names = ", ".join(f'"{h}"' for h in JIT_HEADERS)
    srcs = ", ".join(f'kJitHdr_{h.split(".")[0]}' for h in JIT_HEADERS)
    parts.append(f"static const char* const kJitHeaderNames[] = {{{names}}};\n")
    parts.append(f"static const char* const kJitHeaderSources[] = {{{srcs}}};\n")
    parts.append(f"static const int kJitHeaderCount = {len(JIT_HEADERS)};\n")
    new = "".join(parts)
    path = os.path.join(obj_dir, "jit_headers.inc")
    if not os.path.exists(path) or open(path).read() != new:
        with open(path, "w") as f:
            f.write(new)


BC_LIB = os.path.join(HERE, "libqdp_b200_bc.so")    # the same library compiled with -DQDP_BOUNDS_CHECK (su3.cuh: site_ptr_checked)


def build(force: bool = False, verbose: bool = False, bounds_check: bool = False) -> str:
    """bounds_check: build libqdp_b200_bc.so, every site address validated on the device (tests/test_gpu_bounds.py
    runs the small-lattice parity suite against it through QDP_B200_LIB)."""
    obj_dir = OBJ + "_bc" if bounds_check else OBJ
    lib = BC_LIB if bounds_check else LIB
    flags = NVCC_FLAGS + (["-DQDP_BOUNDS_CHECK"] if bounds_check else [])
    os.makedirs(obj_dir, exist_ok=True)
    _write_jit_headers(obj_dir)
    flags = flags + ["-I", obj_dir]
    nvcc = _nvcc()
    hdr_t = _deps_mtime()
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(obj_dir, src.replace(".cu", ".o"))
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr_t):
            jobs.append((s, o))

    def compile_one(job):
        s, o = job
        r = subprocess.run([nvcc, *flags, "-c", s, "-o", o], capture_output=True, text=True)
        return s, r

    with ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        for s, r in ex.map(compile_one, jobs):
            if verbose or r.returncode:
                sys.stderr.write(f"== {os.path.basename(s)}\n{r.stdout}{r.stderr}\n")
            if r.returncode:
                raise RuntimeError(f"nvcc failed on {s}")
    objs = [os.path.join(obj_dir, s.replace(".cu", ".o")) for s in SOURCES]
    if jobs or force or not os.path.exists(lib):
        subprocess.check_call([nvcc, "-shared", "-o", lib, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-ldl"])
    if bounds_check:
        return lib
    probe_src = os.path.join(CSRC, "probe.cu")
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < os.path.getmtime(probe_src):
        subprocess.check_call([nvcc, *[f for f in NVCC_FLAGS if f not in ("-Xptxas", "-v")], "-shared", probe_src, "-o", PROBE_LIB])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, bounds_check="--bounds-check" in sys.argv))
