"""x3-slab decomposition on the device (row f4 / SURVEY.md 8(e)): the time-slice face kernels and slab_shift.  Only one
GPU is available, so two ranks are emulated in one process as two slab lattices whose faces are handed over by device
copies (no kernel waits on another)."""
import numpy as np
import pytest

import oracle
import synth
from paper_1111_5596_b200 import slab

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 8, 8, 8), (4, 2, 6, 4)])
def test_loopback_shift_equals_the_periodic_shift_and_faces_round_trip(qdp, dims):
    import torch
    lat = qdp.qdp_lattice_create(dims)
    hp = synth.spinor(dims, 1401)
    src = qdp.field_from_host(lat, qdp.QDP_FERMION, hp)
    comm = slab.LoopbackComm()
    for sign in (+1, -1):
        for subset in (0, 1, 2):
            sentinel = np.full_like(hp, 3.0 - 1.0j)
            dst = qdp.field_from_host(lat, qdp.QDP_FERMION, sentinel)
            slab.slab_shift(qdp, dst, src, 3, sign, subset, comm)
            assert np.array_equal(qdp.field_to_host(dst), oracle.shift(dims, hp, 3, sign, subset, dst=sentinel))
    nbytes = qdp.qdp_field_timeslice_bytes(src)
    n = dims[0] * dims[1] * dims[2]
    assert nbytes == n * 12 * 16
    buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda:0")
    other = qdp.field_from_host(lat, qdp.QDP_FERMION, np.zeros_like(hp))
    qdp.qdp_field_get_timeslice(src, 1, buf.data_ptr(), nbytes)
    qdp.qdp_field_set_timeslice(other, 2, buf.data_ptr(), nbytes)         # slice 1 of src lands in slice 2
    got = qdp.field_to_host(other)
    assert np.array_equal(got[2 * n:3 * n], hp[n:2 * n]) and not got[:2 * n].any() and not got[3 * n:].any()
    assert abs(slab.slab_norm2(qdp, src, 0, comm) - oracle.norm2(dims, hp)) <= 1e-12 * oracle.norm2(dims, hp)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_field_get_timeslice(src, dims[3], buf.data_ptr(), nbytes)
    with pytest.raises(qdp.QdpError):
        qdp.qdp_field_get_timeslice(src, 0, buf.data_ptr(), nbytes - 16)


def test_loopback_shift_on_a_non_default_lattice_stream(qdp):
    """The lattice's kernels run on a non-blocking stream of their own while the communication runs on torch's current
    stream: slab_shift has to order the two itself (there is no implicit null-stream ordering to hide a missing wait).
    A large face and a busy current stream make a missing wait visible."""
    import torch
    dims = (16, 16, 16, 4)
    lat = qdp.qdp_lattice_create(dims)
    own = torch.cuda.Stream()
    qdp.qdp_lattice_set_stream(lat, own.cuda_stream)
    hu = synth.gauge_hot(dims, 1403)
    src = qdp.field_from_host(lat, qdp.QDP_GAUGE, hu)
    comm = slab.LoopbackComm()
    busy = torch.empty(1 << 28, dtype=torch.uint8, device="cuda")
    scratch = None
    for sign in (+1, -1):
        sentinel = np.full_like(hu, 3.0 - 1.0j)
        dst = qdp.field_from_host(lat, qdp.QDP_GAUGE, sentinel)
        qdp.qdp_lattice_sync(lat)
        for _ in range(8):
            busy.fill_(1)                                 # work queued on torch's current stream ahead of the copy
        scratch = slab.slab_shift(qdp, dst, src, 3, sign, 0, comm, scratch)
        assert np.array_equal(qdp.field_to_host(dst), oracle.shift(dims, hu, 3, sign, 0, dst=sentinel)), sign
    qdp.qdp_lattice_sync(lat)
    qdp.qdp_lattice_set_stream(lat, None)


@pytest.mark.parametrize("gdims", [(4, 4, 4, 8), (8, 8, 8, 16), (4, 2, 6, 8)])
@pytest.mark.parametrize("kind", ["fermion", "gauge"])
def test_two_emulated_ranks_reproduce_the_global_shift(qdp, gdims, kind):
    import torch
    world = 2
    ldims = slab.local_dims(gdims, world)
    n, Lt = gdims[0] * gdims[1] * gdims[2], ldims[3]
    K = qdp.QDP_FERMION if kind == "fermion" else qdp.QDP_GAUGE
    full = synth.spinor(gdims, 1402) if kind == "fermion" else synth.gauge_hot(gdims, 1402)
    lats = [qdp.qdp_lattice_create(ldims) for _ in range(world)]
    srcs = [qdp.field_from_host(lats[r], K, full[r * Lt * n:(r + 1) * Lt * n].copy()) for r in range(world)]
    nbytes = qdp.qdp_field_timeslice_bytes(srcs[0])
    for sign in (+1, -1):
        for subset in (0, 1, 2):
            sentinel = np.full_like(full, 2.0 + 5.0j)
            want = oracle.shift(gdims, full, 3, sign, subset, dst=sentinel)
            dsts = [qdp.field_from_host(lats[r], K, sentinel[r * Lt * n:(r + 1) * Lt * n].copy()) for r in range(world)]
            faces = {}
            for r in range(world):                               # every rank: local shift, pack its boundary slice
                qdp.qdp_shift(dsts[r], srcs[r], 3, sign, subset)
                plan = slab.face_plan(sign, Lt, r, world)
                buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda:0")
                qdp.qdp_field_get_timeslice(srcs[r], plan["send_slice"], buf.data_ptr(), nbytes)
                qdp.qdp_lattice_sync(lats[r])
                faces[plan["send_to"]] = buf                      # "sent"
            for r in range(world):                               # every rank: unpack what arrived
                plan = slab.face_plan(sign, Lt, r, world)
                qdp.qdp_field_set_timeslice(dsts[r], plan["fix_slice"], faces[r].data_ptr(), nbytes, subset)
                got = qdp.field_to_host(dsts[r])
                assert np.array_equal(got, want[r * Lt * n:(r + 1) * Lt * n]), (sign, subset, r)
    total = sum(qdp.qdp_norm2(s) for s in srcs)
    assert abs(total - oracle.norm2(gdims, full)) <= 1e-12 * total


class _ThreadComm:
    """Two ranks of one process, one host thread each, every rank driving a lattice of its own on the one GPU.  A face
    travels as a device tensor through a queue; only host threads wait for one another, never a kernel."""

    def __init__(self, rank, world, boxes, barrier, sums):
        self.rank, self.world, self.boxes, self.barrier, self.sums = rank, world, boxes, barrier, sums

    def sendrecv(self, send, send_to, recv, recv_from):
        import torch
        torch.cuda.current_stream().synchronize()
        self.boxes[send_to][self.rank].put(send.clone())
        recv.copy_(self.boxes[self.rank][recv_from].get(timeout=60))
        torch.cuda.current_stream().synchronize()

    def allreduce_sum(self, values):
        self.sums[self.rank] = list(values)
        self.barrier.wait(timeout=60)
        out = [sum(self.sums[r][i] for r in range(self.world)) for i in range(len(values))]
        self.barrier.wait(timeout=60)
        return out


@pytest.mark.parametrize("gdims", [(4, 4, 4, 8), (4, 2, 6, 4), (8, 8, 8, 16)])
def test_two_thread_ranks_hop_plaquette_and_ape_on_slabs(qdp, gdims):
    """slab_hop, slab_plaquette and the spatial APE step on two x3 slabs reproduce the oracle's results on the global
    lattice (hop: every subset, per-site bar; plaquette: the bar for sums; APE: the per-link bar)."""
    import queue
    import threading
    from parity import TOL_SITE, links, site_rel_err, z3_fix
    world = 2
    ldims = slab.local_dims(gdims, world)
    n, Lt = gdims[0] * gdims[1] * gdims[2], ldims[3]
    hu, hp = synth.gauge_hot(gdims, 1404), synth.spinor(gdims, 1405)
    want_hop = oracle.hop(gdims, hu, hp)
    want_plaq = oracle.plaquette(gdims, hu)
    want_ape = oracle.ape_smear_step(gdims, hu, 0.5, 3)
    mask = oracle.parity_mask(gdims)
    boxes = [[queue.Queue() for _ in range(world)] for _ in range(world)]
    barrier, sums, results, errors = threading.Barrier(world), [None] * world, [None] * world, []

    def run(rank):
        try:
            comm = _ThreadComm(rank, world, boxes, barrier, sums)
            lo, hi = rank * Lt * n, (rank + 1) * Lt * n
            lat = qdp.qdp_lattice_create(ldims)
            u = qdp.field_from_host(lat, qdp.QDP_GAUGE, hu[lo:hi].copy())
            psi = qdp.field_from_host(lat, qdp.QDP_FERMION, hp[lo:hi].copy())
            out = {}
            work = None
            for subset in (0, 1, 2):
                sentinel = np.full_like(hp[lo:hi], 7.0 - 3.0j)
                chi = qdp.field_from_host(lat, qdp.QDP_FERMION, sentinel)
                work = slab.slab_hop(qdp, chi, u, psi, subset, comm, work)
                out["hop", subset] = qdp.field_to_host(chi)
            out["plaq"], _ = slab.slab_plaquette(qdp, u, comm)
            u2 = qdp.qdp_field_alloc(lat, qdp.QDP_GAUGE, qdp.QDP_F64)
            slab.slab_ape_smear_step(qdp, u2, u, 0.5)
            out["ape"] = qdp.field_to_host(u2)
            results[rank] = out
        except BaseException as exc:      # surfaces in the main thread; the other rank then times out on its queue
            errors.append((rank, exc))
            barrier.abort()

    threads = [threading.Thread(target=run, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not errors, errors
    for rank in range(world):
        lo, hi = rank * Lt * n, (rank + 1) * Lt * n
        out = results[rank]
        for subset in (0, 1, 2):
            sel = np.ones(hi - lo, bool) if subset == 0 else (mask[lo:hi] == (subset - 1))
            got = out["hop", subset]
            assert np.all(got[~sel] == 7.0 - 3.0j), (rank, subset)                       # other sites untouched
            assert site_rel_err(got[sel], want_hop[lo:hi][sel]).max() <= TOL_SITE["f64"], (rank, subset)
        assert np.abs(out["plaq"] - want_plaq).max() <= 1e-10, (rank, out["plaq"], want_plaq)
        fixed, n_centre = z3_fix(links(out["ape"].astype(np.complex128)), links(want_ape[lo:hi]))
        assert n_centre == 0 and site_rel_err(fixed, links(want_ape[lo:hi])).max() <= TOL_SITE["f64"], rank
