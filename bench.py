#!/usr/bin/env python
"""bench.py -- site-updates/s and achieved HBM GB/s of the hot path on one B200.

A "step" is one pass of the whole hot path over one seeded
synthetic lattice of BASELINE.json:configs[3] (C4, 32^3x64 fp64 -- the config the
north_star quotes its 70 % target on):

    shift(psi,+mu) | plaquette(u) | APE step u -> u' | hop on EVEN, hop on ODD |
    inner(psi, chi) | chi = a psi + b hop(psi) with fused norm2 | norm2(chi)

= 7 V site-updates.  `value` is site-updates/s with all inputs resident in HBM, timed with
CUDA events on the lattice's stream; `e2e` is the same pass through the C ABI from pinned
HOST buffers (upload u, psi; download u', chi inside the timed region), two lattices driven by
two host threads so that one step's upload overlaps the other's download.  Every field is
larger than the 126 MB L2, so no explicit L2 flush is needed between iterations.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1 (torchrun): the path is single-GPU by contract ("replicas only"): every
rank runs an independent replica; value = N * units / max-over-ranks time, scaling "weak".
--impl reference times the oracle (plain single-threaded C, as it stands) on host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "site-updates/s"
UNIT = "site-updates/s"
OPS_PER_STEP = 7          # shift, plaquette, ape, hop(even+odd), inner, axpy_hop+norm2, norm2
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md
# fp64 instructions per site of the fused kernels as implemented (SASS, straight-line code: every instruction
# executes once per site; profiles/r3_sass.md, counted with cuobjdump): (DFMA, DMUL, DADD).  The "alu" view of the roofline divides the
# resulting flop rate by the DFMA rate measured in the same run (paper_1111_5596_b200/csrc/probe.cu).
FP64_INSTR_PER_SITE = {
    "ape": (3310, 493, 89),          # 24 3x3 complex products, blend, three SU(3) projections
    "plaquette": (1188, 219, 18),    # 12 products + 6 traces
}


def fp64_flops_per_site(op: str) -> int:
    dfma, dmul, dadd = FP64_INSTR_PER_SITE[op]
    return 2 * dfma + dmul + dadd


def probe_dfma_rate(device: int, stream) -> float | None:
    """DFMA per second (thread-level) of the plain fp64 pipe, measured now on this device (bench-only probe library)."""
    try:
        from paper_1111_5596_b200 import probe
        return probe.dfma_rate(device, stream)
    except (OSError, RuntimeError):
        return None


def algorithmic_bytes(V: int, eb: int) -> dict:
    """every operand element read once, every result element written once.
    eb = bytes per complex (16 fp64, 8 fp32).  Per launch on V sites."""
    return {
        "shift": V * 24 * eb,              # spinor: r 12 + w 12
        "plaquette": V * 36 * eb,          # every link once
        "ape": V * 72 * eb,                # full u_out contract: 36 r + 36 w (U_3 copied through)
        "hop_even": (V // 2) * 96 * eb,    # 8 links (72) + psi 12 + chi 12 per updated site
        "hop_odd": (V // 2) * 96 * eb,
        "inner": V * 24 * eb,
        "axpy_hop_norm2": V * 60 * eb,     # u 36 + psi 12 + chi 12
        "norm2": V * 12 * eb,
    }


def measured_peak() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(config: str, prec: str, kernel: str):
    """dram__bytes_read + write per launch of `kernel` from the committed ncu --set full capture of exactly this
    (config, precision); None when no capture of that combination is committed."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f).get(f"{config}/{prec}", {}).get(kernel)
    except Exception:
        return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (pynvml)."""

    def __init__(self, index: int, period: float = 0.002):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
        }
        while not self._halt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self) -> dict:
        self._halt.set()
        self.join(timeout=1.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def rank_env() -> tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when run directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def max_over_ranks(values, dist, device) -> list[float]:
    """Element-wise MAX over ranks of a list of per-rank times (the job is as slow as its slowest
    replica); identity when not distributed.  The only cross-rank operation of the bench: the data
    path itself has no collective ("replicas only")."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(units_per_rank: int, world: int, ms: float) -> float:
    """Whole-job throughput: every rank processed units_per_rank units in (max over ranks) ms."""
    return units_per_rank * world / (ms * 1e-3)


class Workload:
    """One seeded synthetic lattice of a BASELINE config resident in HBM, and the 7-op step on it."""

    def __init__(self, q, torch, config: str, prec: str, device: int, seed: int):
        import synth
        self.q, self.torch, self.config, self.prec = q, torch, config, prec
        self.dims = synth.CONFIGS[config]
        self.V = synth.volume(self.dims)
        self.P = q.QDP_F64 if prec == "f64" else q.QDP_F32
        self.eb = 16 if prec == "f64" else 8
        self.hu = synth.round_to(synth.gauge_hot(self.dims, seed), prec)
        self.hp = synth.round_to(synth.spinor(self.dims, seed), prec)
        self.a, self.b = synth.scalars_ab(seed)
        self.stream = torch.cuda.Stream()
        self.lat = q.qdp_lattice_create(self.dims, device)
        q.qdp_lattice_set_stream(self.lat, self.stream.cuda_stream)
        self.u = q.field_from_host(self.lat, q.QDP_GAUGE, self.hu)
        self.psi = q.field_from_host(self.lat, q.QDP_FERMION, self.hp)
        self.u2 = q.qdp_field_alloc(self.lat, q.QDP_GAUGE, self.P)
        self.chi = q.qdp_field_alloc(self.lat, q.QDP_FERMION, self.P)
        self.sh = q.qdp_field_alloc(self.lat, q.QDP_FERMION, self.P)
        u, psi, u2, chi, sh, a, b = self.u, self.psi, self.u2, self.chi, self.sh, self.a, self.b
        self.ops = [
            ("shift", lambda k: q.qdp_shift(sh, psi, k % 4, 1 if (k // 4) % 2 == 0 else -1)),
            ("plaquette", lambda k: q.qdp_plaquette(u)),
            ("ape", lambda k: q.qdp_ape_smear_step(u2, u, 0.5, 3)),
            ("hop_even", lambda k: q.qdp_hop(chi, u, psi, q.QDP_EVEN)),
            ("hop_odd", lambda k: q.qdp_hop(chi, u, psi, q.QDP_ODD)),
            ("inner", lambda k: q.qdp_inner(psi, chi)),
            ("axpy_hop_norm2", lambda k: q.qdp_axpy_hop(chi, a, b, u, psi, q.QDP_ALL, want_norm2=True)),
            ("norm2", lambda k: q.qdp_norm2(chi)),
        ]
        self.results = {}

    def step(self, k, evs=None):
        for i, (name, fn) in enumerate(self.ops):
            if evs is not None:
                evs[i].record(self.stream)
            self.results[name] = fn(k)
        if evs is not None:
            evs[len(self.ops)].record(self.stream)

    def timed(self, K: int, warmup: int, barrier=None, sampler=None):
        """W untimed steps, then exactly K steps bracketed by `barrier`; CUDA events on the lattice's stream around
        every op.  Returns (total ms, per-op mean ms, kernels launched)."""
        torch, q = self.torch, self.q
        for k in range(warmup):
            self.step(k)
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(len(self.ops) + 1)] for _ in range(K)]
        (barrier or torch.cuda.synchronize)()
        launches0 = q.qdp_kernel_launch_count()
        if sampler is not None:
            sampler.start()
        for k in range(K):
            self.step(k, evs[k])
        torch.cuda.synchronize()
        self.clocks = sampler.stop() if sampler is not None else None
        launches = q.qdp_kernel_launch_count() - launches0
        (barrier or torch.cuda.synchronize)()
        total_ms = evs[0][0].elapsed_time(evs[K - 1][len(self.ops)])
        per_op_ms = {name: float(np.mean([evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(K)]))
                     for i, (name, _) in enumerate(self.ops)}
        return total_ms, per_op_ms, launches

    def op_report(self, per_op_ms: dict, peak: float) -> dict:
        alg = algorithmic_bytes(self.V, self.eb)
        rep = {}
        for name, ms in per_op_ms.items():
            gbs = alg[name] / ms / 1e6
            sites = self.V // 2 if name.startswith("hop_") else self.V
            rep[name] = {"ms": round(ms, 5), "gbs": round(gbs, 1), "frac": round(gbs / peak, 4),
                         "site_updates_per_s": sites / ms * 1e3}
        return rep

    def free(self):
        for f in (self.u, self.psi, self.u2, self.chi, self.sh):
            self.q.qdp_field_free(f)
        self.q.qdp_lattice_destroy(self.lat)


def run_ours(args) -> dict | None:
    import torch
    import synth
    from paper_1111_5596_b200.build import LIB, build as build_cuda
    if not os.path.exists(LIB) and int(os.environ.get("LOCAL_RANK", "0")) == 0:
        build_cuda()                 # fresh checkout: compile the library (no fallback: without it nothing runs)
    import paper_1111_5596_b200 as q

    rank, world, local = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    prec = args.prec
    w = Workload(q, torch, args.config, prec, local, synth.BASE_SEED + 3 + rank)
    dims, V, P, eb = w.dims, w.V, w.P, w.eb
    hu, hp, a, b = w.hu, w.hp, w.a, w.b
    stream, lat, u, psi, u2, chi, sh = w.stream, w.lat, w.u, w.psi, w.u2, w.chi, w.sh
    results = w.results

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    K = args.steps
    total_ms, per_op_ms, launches = w.timed(K, args.warmup, barrier, ClockSampler(local))
    clocks = w.clocks
    dfma_rate = probe_dfma_rate(local, stream.cuda_stream) if rank == 0 else None

    # ---- rows widened beyond the step: timed separately, not part of `value` -------
    # name -> (call, complex numbers moved per site (algorithmic), note)
    cm = q.qdp_field_alloc(lat, q.QDP_COLOR_MATRIX, P)
    plane = "real(trace(f0[{a}] * shift(f0[{b}], +{a}) * adj(shift(f0[{a}], +{b})) * adj(f0[{b}])))"
    JIT_PLAQ_S = " + ".join(plane.format(a=a, b=b) for a, b in ((0, 1), (0, 2), (1, 2)))
    JIT_PLAQ_T = " + ".join(plane.format(a=a, b=3) for a in range(3))
    JIT_HOP = " + ".join(f"f0[{m}] * shift(f1, +{m}) + shift(adj(f0[{m}]) * f1, -{m})" for m in range(4))
    JIT_STAPLE = " + ".join(f"(f0[{n}] * shift(f0[0], +{n}) * adj(shift(f0[{n}], +0)) + shift(adj(f0[{n}]) * f0[0] * shift(f0[{n}], +0), -{n}))"
                            for n in (1, 2))
    extra_defs = {
        "smear_hop": (lambda: q.qdp_smear_hop(chi, a, b, u, psi, 3), 51,
                      "qdp_smear_hop, t_dir = 3 (row f2): u 27 + psi 12 + chi 12 complex per site"),
        "ape_4d": (lambda: q.qdp_ape_smear_step(u2, u, 0.5, -1), 72,
                   "qdp_ape_smear_step, t_dir = -1 (row f2: 4-D APE, 6 staples per link, all four links projected): "
                   "36 complex read + 36 written per site"),
        "inner_timeslices": (lambda: q.qdp_inner_timeslices(psi, chi), 24,
                             "qdp_inner_timeslices (row f3): 2 x 12 complex per site, includes the host round trip"),
        "reunitarize_gs": (lambda: q.qdp_reunitarize(u2, u, q.QDP_REUNIT_GRAM_SCHMIDT), 60,
                           "qdp_reunitarize, Gram-Schmidt (row f2): 24 complex read (rows 0, 1 of four links; row 2 is "
                           "not an input) + 36 written per site"),
        "matmul": (lambda: q.qdp_matmul(u2, 0, u, 0, 0, u, 1, 1, 0, 1), 27,
                   "qdp_matmul u2[0] = u[0] * adj(u[1])(x+0) (row f1): 2 x 9 complex read + 9 written per site"),
        "axpby": (lambda: q.qdp_axpby(sh, a, psi, b, chi), 36,
                  "qdp_axpby on spinors (PAPER.md:96): 2 x 12 complex read + 12 written per site"),
        "expr_plaquette": (lambda: q.qdp_expr_plaquette(u), 36,
                           "qdp_expr_plaquette (row f1): the plaquette written as one expression of the compile-time "
                           "layer, one kernel; compare ops.plaquette (hand-fused)"),
        "jit_plaquette": (lambda: (q.qdp_expr_jit_sum(JIT_PLAQ_S, [u]), q.qdp_expr_jit_sum(JIT_PLAQ_T, [u])), 36,
                          "qdp_expr_jit_sum (row f1, run-time expressions): the spatial and the temporal planes of the plaquette "
                          "as two text expressions compiled with NVRTC on first use (cached afterwards): two kernels, so the "
                          "gauge field is really read twice, but the algorithmic bytes are those of the plaquette (36 complex "
                          "per site) and the fraction is charged for the second read; compare expr_plaquette and ops.plaquette"),
        "jit_hop": (lambda: q.qdp_expr_jit_assign(chi, 0, JIT_HOP, [u, psi]), 60,
                    "qdp_expr_jit_assign (row f1): the hopping term of def. 5 on the full lattice as a text expression with "
                    "fermion leaves (u 36 + psi 12 + chi 12 complex per site, SURVEY.md 8(d): 960 B in fp64); compare the hand-fused qdp_hop ALL (hop_all)"),
        "hop_all": (lambda: q.qdp_hop(chi, u, psi, q.QDP_ALL), 60,
                    "qdp_hop on the full lattice, hand-fused (the step times the halves and the fused axpy form): "
                    "u 36 + psi 12 + chi 12 complex per site"),
        "jit_staple": (lambda: q.qdp_expr_jit_assign(cm, 0, JIT_STAPLE, [u]), 36,
                       "qdp_expr_jit_assign (row f1): the spatial staple sum of link 0 as a text expression; the same kernel as "
                       "expr_staple, through NVRTC"),
        "expr_staple": (lambda: q.qdp_expr_staple(cm, u, 0, 3), 36,
                        "qdp_expr_staple mu = 0, spatial (row f1): the staple sum as one expression; 27 complex read "
                        "(three links) + 9 written per site"),
        "project_max_retr": (lambda: q.qdp_project_max_retr(u2, u, 3), 72,
                             "qdp_project_max_retr, 3 sweeps (row f2): 36 complex read + 36 written per site"),
        "baryon_timeslices": (lambda: q.qdp_baryon_timeslices([psi, chi, sh], [chi, sh, psi], [sh, psi, chi], 5), 36,
                              "qdp_baryon_timeslices, nsrc = 3 (row f3): the call takes nine field arguments (108 complex per site "
                              "when they are nine different propagator columns); this row passes 3 distinct spinor fields three "
                              "times each, so the bytes that must move, and are counted, are 36 complex per site; includes the "
                              "host round trip"),
        "plaquette_staged": (None, 36, "qdp_plaquette with qdp_lattice_set_staged(1): cp.async.bulk + mbarrier "
                                       "shared-memory rings (plaquette_tma.cu); compare ops.plaquette"),
    }
    extra_ms = {}
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_jit = time.perf_counter()      # first use compiles: measured once, outside every timed region
    n_jit = q.qdp_expr_jit_compilations()
    try:
        extra_defs["jit_plaquette"][0]()
        extra_defs["jit_staple"][0]()
        extra_defs["jit_hop"][0]()
        jit_compile = {"expressions": q.qdp_expr_jit_compilations() - n_jit, "seconds": round(time.perf_counter() - t_jit, 3)}
    except q.QdpError as exc:       # e.g. no libnvrtc on this machine: the run-time expression rows are skipped, nothing else
        jit_compile = {"unavailable": str(exc)[:200]}
        for name in [n for n in extra_defs if n.startswith("jit_")]:
            del extra_defs[name]

    def time_extra(fn):
        for _ in range(3):
            fn()
        ev0.record(stream)
        for _ in range(K):
            fn()
        ev1.record(stream)
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) / K

    for name, (fn, _, _) in extra_defs.items():
        if fn is not None:
            extra_ms[name] = time_extra(fn)
    q.qdp_lattice_set_staged(lat, True)
    extra_ms["plaquette_staged"] = time_extra(lambda: q.qdp_plaquette(u))
    q.qdp_lattice_set_staged(lat, False)
    q.qdp_field_free(cm)

    # ---- end to end through the C ABI from pinned host buffers ----------------------
    ke = max(1, min(args.e2e_steps, K))
    if args.no_e2e:
        ke = 0
    pin_u = torch.empty(hu.nbytes, dtype=torch.uint8, pin_memory=True)
    pin_p = torch.empty(hp.nbytes, dtype=torch.uint8, pin_memory=True)
    pin_u.numpy()[:] = hu.view(np.uint8).ravel()
    pin_p.numpy()[:] = hp.view(np.uint8).ravel()

    h2d_turn, d2h_turn = threading.Lock(), threading.Lock()

    def make_pipe(lat_, u_, psi_, u2_, chi_, sh_):
        """One lattice with its fields and pinned result buffers; returns its end-to-end step:
        upload u, psi from pinned host memory, the 7-op pass, download u', chi."""
        pin_u2 = torch.empty(hu.nbytes, dtype=torch.uint8, pin_memory=True)
        pin_chi = torch.empty(hp.nbytes, dtype=torch.uint8, pin_memory=True)

        def one(k):
            with h2d_turn:       # one pipe at a time per PCIe direction: the other pipe is downloading meanwhile
                q.qdp_field_upload(u_, pin_u)
                q.qdp_field_upload(psi_, pin_p)
            q.qdp_shift(sh_, psi_, k % 4, 1 if (k // 4) % 2 == 0 else -1)
            q.qdp_plaquette(u_)
            q.qdp_ape_smear_step(u2_, u_, 0.5, 3)
            q.qdp_hop(chi_, u_, psi_, q.QDP_EVEN)
            q.qdp_hop(chi_, u_, psi_, q.QDP_ODD)
            q.qdp_inner(psi_, chi_)
            q.qdp_axpy_hop(chi_, a, b, u_, psi_, q.QDP_ALL, want_norm2=True)
            q.qdp_norm2(chi_)
            with d2h_turn:
                q.qdp_field_download(u2_, pin_u2)
                q.qdp_field_download(chi_, pin_chi)
        return one

    # Two lattices driven by two host threads: PCIe is full duplex, so the upload of one step
    # overlaps the download of the other (a single synchronous step uses one direction at a time).
    # Every step still moves its own inputs and results; `value` = steps of both pipes / wall time.
    e2e_s, n_pipes = 0.0, args.e2e_pipes
    if ke:
        pipes = [make_pipe(lat, u, psi, u2, chi, sh)]
        extra = []      # keep the extra lattices, streams and fields alive
        for _ in range(n_pipes - 1):
            lat_b = q.qdp_lattice_create(dims, local)
            stream_b = torch.cuda.Stream()
            q.qdp_lattice_set_stream(lat_b, stream_b.cuda_stream)
            fields_b = (q.qdp_field_alloc(lat_b, q.QDP_GAUGE, P), q.qdp_field_alloc(lat_b, q.QDP_FERMION, P),
                        q.qdp_field_alloc(lat_b, q.QDP_GAUGE, P), q.qdp_field_alloc(lat_b, q.QDP_FERMION, P),
                        q.qdp_field_alloc(lat_b, q.QDP_FERMION, P))
            extra.append((lat_b, stream_b, fields_b))
            pipes.append(make_pipe(lat_b, *fields_b))
        for one in pipes:
            one(0)
        barrier()
        errors = []

        def drive(one):
            try:
                torch.cuda.set_device(local)
                for k in range(ke):
                    one(k)
            except Exception as exc:   # surfaced after the join
                errors.append(exc)
        threads = [threading.Thread(target=drive, args=(one,)) for one in pipes]
        t0 = time.perf_counter()
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        if errors:
            raise errors[0]
        barrier()

    total_ms, e2e_ms = max_over_ranks([total_ms, e2e_s * 1e3], dist, f"cuda:{local}")

    # ---- the other BASELINE configs that fit the time budget, same 7-op step, per-op roofline fractions only -------
    # (parity-test configurations, not bench lines: they do not enter `value`.)
    other = {}
    if world == 1 and not args.no_other_configs and args.config == "C4" and prec == "f64":
        peak_o, _ = measured_peak()
        # C5 (48^3 x 96, 6.1 GB fp64 gauge field) is BASELINE.json's "bandwidth at scale" configuration: few steps, its
        # host-side generation and upload dominate the ~20 s each precision adds to the run
        for cfg, pr in (("C4", "f32"), ("C3", "f64"), ("C3", "f32"), ("C5", "f64"), ("C5", "f32")):
            wo = Workload(q, torch, cfg, pr, local, synth.BASE_SEED + 3)
            ko = max(3, min(K, 10)) if cfg != "C5" else 3
            tot, per_op, _ = wo.timed(ko, 3)
            other[f"{cfg}/{pr}"] = {"ms_per_step": round(tot / ko, 5), "steps": ko,
                                    "site_updates_per_s": OPS_PER_STEP * wo.V * ko / (tot * 1e-3),
                                    "ops": {n: {"ms": r["ms"], "frac": r["frac"]} for n, r in wo.op_report(per_op, peak_o).items()}}
            wo.free()
            del wo
            torch.cuda.empty_cache()

    out = None
    if rank == 0:
        peak, peak_src = measured_peak()
        alg = algorithmic_bytes(V, eb)
        op_report = w.op_report(per_op_ms, peak)
        dom = max(per_op_ms, key=per_op_ms.get)
        dom_kernel = {"ape": "ape_kernel", "plaquette": "plaquette_kernel", "axpy_hop_norm2": "hop_kernel",
                      "hop_even": "hop_kernel", "hop_odd": "hop_kernel"}.get(dom, dom + "_kernel")
        # roofline of the dominant kernel in the metric's own unit: algorithmic bytes (SURVEY.md 8(d) per-site figure
        # x sites of one launch) / CUDA-event time / measured HBM copy peak.  A reader can recompute frac from
        # algorithmic_bytes_per_launch, ops[op].ms and peak.  The fp64-pipe ("alu") view of the same launch is beside it.
        roofline = {"bound": "hbm", "kernel": dom_kernel, "op": dom,
                    "achieved": op_report[dom]["gbs"], "peak": peak, "unit": "GB/s",
                    "frac": op_report[dom]["frac"], "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": alg[dom], "ms_per_launch": op_report[dom]["ms"],
                    "traffic": ncu_traffic(args.config, prec, dom_kernel)}
        alu = {}
        if prec == "f64" and dfma_rate:
            for name in FP64_INSTR_PER_SITE:
                tf = fp64_flops_per_site(name) * V / per_op_ms[name] / 1e9
                slots = sum(FP64_INSTR_PER_SITE[name]) * V / (per_op_ms[name] * 1e-3) / dfma_rate
                alu[name] = {"achieved": round(tf, 2), "peak": round(2 * dfma_rate / 1e12, 2), "unit": "TFLOP/s",
                             "frac": round(tf / (2 * dfma_rate / 1e12), 4), "fp64_pipe_slots_frac": round(slots, 4),
                             "peak_source": "measured in this run: DFMA-only kernel of csrc/probe.cu, "
                                            f"{dfma_rate / 1e12:.2f} T DFMA/s x 2 flop",
                             "fp64_instr_per_site": dict(zip(("dfma", "dmul", "dadd"), FP64_INSTR_PER_SITE[name]))}
            if dom in alu:
                roofline["alu"] = alu[dom]
        out = {
            "metric": METRIC, "value": whole_job_value(OPS_PER_STEP * V * K, world, total_ms), "unit": UNIT,
            "n_gpus": world, "steps": K, "warmup": args.warmup, "ms_per_step": total_ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": prec, "data": "synthetic",
            "config": {"workload": f"{args.config} {'x'.join(map(str, dims))} {prec}: shift, plaquette, "
                                   "APE step (alpha=0.5, spatial) with SU(3) reprojection, hop even+odd, "
                                   "inner, axpy_hop+norm2, norm2; hot (Haar) links",
                       "sites": V, "site_updates_per_step": OPS_PER_STEP * V,
                       "l2": "inputs larger than L2 (gauge 1.2 GB, spinor 0.4 GB vs 126 MB)",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "clocks": clocks,
            "e2e": ({"value": whole_job_value(OPS_PER_STEP * V * ke * n_pipes, world, e2e_ms), "unit": UNIT,
                     "h2d_bytes_per_step": int(hu.nbytes + hp.nbytes),
                     "d2h_bytes_per_step": int(hu.nbytes + hp.nbytes),
                     "steps": ke * n_pipes, "ms_per_step": e2e_ms / (ke * n_pipes),
                     "pipelining": f"{n_pipes} lattices x {n_pipes} host threads, one transfer per PCIe direction at a time (the upload of one "
                                   "step overlaps the download of the other); each step moves its own inputs and results"}
                    if ke else None),
            "gpu_launches": int(launches),
            "roofline": roofline,
            "ops": op_report,
            "alu": alu,
            "other_configs": other,
            "extra_ops": {name: {"ms": round(extra_ms[name], 5),
                                 "gbs": round(V * nc * eb / extra_ms[name] / 1e6, 1),
                                 "frac": round(V * nc * eb / extra_ms[name] / 1e6 / peak, 4),
                                 "note": note + "; not part of the step"}
                          for name, (_, nc, note) in extra_defs.items()},
            "jit": dict(jit_compile, note="NVRTC compilations on first use of the run-time expressions of extra_ops (jit_*), wall clock "
                                          "including their first launches; later uses hit the cache"),
            "scalars": {"plaquette": [float(x) for x in results["plaquette"]], "norm2": float(results["norm2"])},
        }
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(args, hu, hp, a, b, fraction=args.cpu_fraction)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return out


def cpu_baseline(args, hu, hp, a, b, fraction: int) -> dict:
    """The oracle as it stands, single-threaded, on a bounded sample: the first V/fraction
    lex sites (whole time-slices) of the same lattice and inputs."""
    import oracle
    import synth
    dims = synth.CONFIGS[args.config]
    V = synth.volume(dims)
    u = hu.astype(np.complex128, copy=False)
    psi = hp.astype(np.complex128, copy=False)
    chi, u_out, shifted = np.zeros_like(psi), np.zeros_like(u), np.zeros_like(psi)
    n = V // fraction
    t0 = time.perf_counter()
    oracle.hot_path_sample(dims, u, psi, chi, u_out, shifted, a, b, 0, n)
    dt = time.perf_counter() - t0
    return {"value": OPS_PER_STEP * n / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"lex sites [0, V/{fraction}) = {n} sites ({dims[3] // fraction} time-slices) of the same "
                      f"lattice, one pass of the same 7 ops, {dt:.1f} s",
            "host_cores_available": os.cpu_count()}


def run_reference(args) -> dict | None:
    """--impl reference: the oracle on host cores; each step is one time-slice-sized sample."""
    if int(os.environ.get("RANK", "0")) != 0:
        return None
    import oracle
    import synth
    dims = synth.CONFIGS[args.config]
    V = synth.volume(dims)
    seed = synth.BASE_SEED + 3
    hu = synth.round_to(synth.gauge_hot(dims, seed), args.prec).astype(np.complex128)
    hp = synth.round_to(synth.spinor(dims, seed), args.prec).astype(np.complex128)
    a, b = synth.scalars_ab(seed)
    chi, u_out, shifted = np.zeros_like(hp), np.zeros_like(hu), np.zeros_like(hp)
    n = V // dims[3]   # one time-slice per step
    nslices = dims[3]

    def step(k):
        lo = (k % nslices) * n
        oracle.hot_path_sample(dims, hu, hp, chi, u_out, shifted, a, b, lo, lo + n)

    for k in range(args.warmup):
        step(k)
    t0 = time.perf_counter()
    for k in range(args.steps):
        step(args.warmup + k)
    dt = time.perf_counter() - t0
    value = OPS_PER_STEP * n * args.steps / dt
    sample = f"one x3 time-slice ({n} sites) of {args.config} per step, 7 ops, single thread"
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.config} {'x'.join(map(str, dims))} {args.prec}: the same 7-op pass, "
                               "oracle (plain C, fp64) on host cores, bounded sample per step",
                   "sites": V, "sample_sites_per_step": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--e2e-pipes", type=int, default=2, help="lattices (host threads) pipelined in the e2e leg")
    ap.add_argument("--cpu-fraction", type=int, default=1, help="cpu_baseline runs on V/fraction sites (1: one whole pass, ~15 s)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the C4 f32 / C3 / C5 per-op block")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    out = run_reference(args) if args.impl == "reference" else run_ours(args)
    if out is not None:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
