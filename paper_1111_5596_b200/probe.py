"""Peak and overlap probes (csrc/probe.cu -> libqdp_probe.so; bench-only, not part of the C ABI of include/qdp_b200.h).

    python -m paper_1111_5596_b200.probe            # prints the tables quoted in profiles/r2_microbench.md

bench.py uses dfma_rate() as the measured denominator of the fp64 ("alu") roofline view."""
from __future__ import annotations

import ctypes

from .build import PROBE_LIB

_lib = None


def _get():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(PROBE_LIB)
        D = ctypes.POINTER(ctypes.c_double)
        lib.qdp_probe_dfma.argtypes, lib.qdp_probe_dfma.restype = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int, D], ctypes.c_int
        lib.qdp_probe_mix.argtypes, lib.qdp_probe_mix.restype = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, D], ctypes.c_int
        lib.qdp_probe_dfma_chain.argtypes, lib.qdp_probe_dfma_chain.restype = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, D], ctypes.c_int
        lib.qdp_probe_bulk_rate.argtypes, lib.qdp_probe_bulk_rate.restype = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, D], ctypes.c_int
        lib.qdp_probe_overlap.argtypes, lib.qdp_probe_overlap.restype = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, D], ctypes.c_int
        _lib = lib
    return _lib


def _call(fn, *args) -> float:
    out = ctypes.c_double()
    rc = fn(*args, ctypes.byref(out))
    if rc != 0:
        raise RuntimeError(f"{fn.__name__} failed with cudaError {rc}")
    return out.value


def dfma_rate(device: int = 0, stream=None, reps: int = 5) -> float:
    """Thread-level DFMA per second of the plain fp64 pipe at saturation."""
    return _call(_get().qdp_probe_dfma, device, stream, reps)


def mix_ms_per_step(mode: int, nlds: int = 36, device: int = 0, stream=None) -> float:
    """mode: bit 0 LDS.128, bit 1 DFMA, bit 2 bulk copies into shared memory; see csrc/probe.cu."""
    return _call(_get().qdp_probe_mix, device, stream, mode, nlds)


def dfma_chain_ns(warps: int, chains: int, device: int = 0, stream=None) -> float:
    return _call(_get().qdp_probe_dfma_chain, device, stream, warps, chains)


def overlap_ms_per_step(mode: int, src: int, pipe: int, device: int = 0, stream=None) -> float:
    """8 warps/SM, per step and warp 24 128-bit loads (src 0: LDS, 1: LDG hitting L1) and 234 DFMA; see csrc/probe.cu."""
    return _call(_get().qdp_probe_overlap, device, stream, mode, src, pipe)


def bulk_bytes_per_s(blocks: int, ncopies: int = 5, device: int = 0, stream=None) -> float:
    """cp.async.bulk from an L2-resident buffer into shared memory, `blocks` active SMs; see csrc/probe.cu."""
    return _call(_get().qdp_probe_bulk_rate, device, stream, blocks, ncopies)


def main() -> None:
    import torch
    dev = torch.cuda.current_device()
    props = torch.cuda.get_device_properties(dev)
    ghz = 1.965      # clocks.max.sm of the B200s of this pool; cycles below are quoted at that clock
    r = dfma_rate(dev)
    print(f"{props.name}, {props.multi_processor_count} SMs")
    print(f"DFMA rate, 12 warps/SM x 8 chains: {r / 1e12:.2f} T DFMA/s = {r / props.multi_processor_count / (ghz * 1e9):.1f} lanes/clk/SM at {ghz} GHz")
    for warps, chains in ((1, 1), (1, 2), (1, 4), (4, 8)):
        ns = dfma_chain_ns(warps, chains, dev)
        print(f"DFMA, {warps} warp(s)/SM, {chains} chain(s): {ns * ghz:.2f} cycles per DFMA of a warp")
    print("per step: 12 warps x (N LDS.128 + 234 DFMA) [+ 92,160 B of bulk copies]; floors: 36 LDS -> 1728 cycles, DFMA 1404 cycles")
    rows = [("LDS(36) only", 1, 36), ("DFMA only", 2, 36), ("LDS(36) + DFMA", 3, 36), ("bulk copies only", 4, 36),
            ("LDS(36) + bulk", 5, 36), ("DFMA + bulk", 6, 36), ("LDS(36) + DFMA + bulk", 7, 36),
            ("LDS(28) + DFMA", 3, 28), ("LDS(24) + DFMA", 3, 24), ("LDS(18) + DFMA", 3, 18), ("LDS(28) + DFMA + bulk", 7, 28)]
    for name, mode, nl in rows:
        ms = mix_ms_per_step(mode, nl, dev)
        print(f"{name:24s} {ms * 1e3:7.3f} us/step = {ms * 1e-3 * ghz * 1e9:6.0f} cycles/step")
    print("8 warps/SM (2 per sub-partition), per step and warp 24 x 128-bit loads + 234 DFMA; floors: loads 768 cycles, DFMA 936 cycles")
    for src, sname in ((0, "LDS"), (1, "LDG, L1 hit")):
        for name, mode, pipe in (("loads only", 1, 0), ("DFMA only", 2, 0), ("loads, then DFMA (per warp)", 3, 0),
                                 ("loads of step s+1 before DFMA of step s", 3, 1)):
            ms = overlap_ms_per_step(mode, src, pipe, dev)
            print(f"{sname:12s} {name:42s} {ms * 1e3:7.3f} us/step = {ms * 1e-3 * ghz * 1e9:6.0f} cycles/step")

    print("cp.async.bulk from L2 into shared memory, 92,160 B per step and SM, two steps in flight")
    nsm = props.multi_processor_count
    for ncopies in (5, 20):
        for blocks in (8, nsm // 4, nsm // 2, nsm):
            r = bulk_bytes_per_s(blocks, ncopies, dev)
            print(f"{ncopies:2d} copies of {92160 // ncopies:5d} B, {blocks:3d} SMs: {r / 1e12:6.2f} TB/s in total = {r / blocks / (ghz * 1e9):6.1f} B/clk/SM")


if __name__ == "__main__":
    main()
