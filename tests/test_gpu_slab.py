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
