"""x3-slab decomposition of a lattice over several GPUs (multi-GPU is the
paper's "future work").  One process per GPU; rank r owns the time-slices [r L3/N, (r+1) L3/N) as a lattice of its own
(qdp_lattice_create with the local extent, which must be even so that local and global parity agree).

What the decomposition changes, and nothing else:
  * shift(f, +-3): the local shift wraps inside the slab, so its boundary slice is wrong; it is overwritten with the
    neighbouring rank's boundary slice -- ONE face exchange per shift (qdp_field_get_timeslice -> send/recv ->
    qdp_field_set_timeslice).  Shifts along x0, x1, x2 are purely local.
  * global sums: all-reduce of the local doubles.
The fused neighbour-reading kernels (hop, plaquette, APE) read x3 neighbours inside their kernel and would need ghost
slices; bench.py therefore runs replicas only (BASELINE.json: one GPU), and this module covers shift and the reductions.

`comm` is a small adapter over torch.distributed (or LoopbackComm for one rank); every function here is argument
marshalling and message ordering -- the data movement on the device is the two kernels of csrc/layout.cu."""
from __future__ import annotations


def neighbor_ranks(rank: int, world: int) -> tuple[int, int]:
    """(rank owning the slab after mine in +x3, rank owning the slab before mine), periodic."""
    return (rank + 1) % world, (rank - 1) % world


def local_dims(global_dims, world: int):
    L3 = global_dims[3]
    if L3 % world or (L3 // world) % 2:
        raise ValueError(f"L3 = {L3} must split into {world} slabs of even extent")
    return (global_dims[0], global_dims[1], global_dims[2], L3 // world)


def face_plan(sign: int, local_L3: int, rank: int, world: int) -> dict:
    """Which local slice is sent to whom and which is overwritten by what arrives, for shift(f, sign * 3):
    dst(x) = src(x + sign 3): the slice that wrapped is local_L3 - 1 (sign = +1) or 0 (sign = -1)."""
    up, down = neighbor_ranks(rank, world)
    if sign > 0:      # I need slice 0 of the rank above me; the rank below me needs my slice 0
        return {"send_slice": 0, "send_to": down, "recv_from": up, "fix_slice": local_L3 - 1}
    return {"send_slice": local_L3 - 1, "send_to": up, "recv_from": down, "fix_slice": 0}


class LoopbackComm:
    """world_size 1: the neighbour is this rank."""
    rank, world = 0, 1

    def sendrecv(self, send, send_to, recv, recv_from):
        recv.copy_(send)

    def allreduce_sum(self, values):
        return list(values)


class TorchComm:
    """torch.distributed (nccl for device tensors, gloo for host tensors)."""

    def __init__(self, dist):
        self.dist, self.rank, self.world = dist, dist.get_rank(), dist.get_world_size()

    def sendrecv(self, send, send_to, recv, recv_from):
        if self.world == 1:
            recv.copy_(send)
            return
        dist = self.dist
        ops = [dist.P2POp(dist.isend, send, send_to), dist.P2POp(dist.irecv, recv, recv_from)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()

    def allreduce_sum(self, values):
        import torch
        t = torch.tensor(list(values), dtype=torch.float64)
        if self.world > 1:
            dev = "cuda" if self.dist.get_backend() == "nccl" else "cpu"
            t = t.to(dev)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return [float(x) for x in t.cpu()]


def slab_shift(q, dst, src, mu: int, sign: int, subset: int, comm, scratch=None):
    """dst(x) = src(x + sign mu) on the GLOBAL lattice; dst, src: this rank's slab fields.  Returns the scratch
    (two device byte tensors) so that callers can reuse it."""
    import torch
    q.qdp_shift(dst, src, mu, sign, subset)
    if mu != 3:
        return scratch
    lat = src.lat
    nbytes = q.qdp_field_timeslice_bytes(src)
    if scratch is None or scratch[0].numel() < nbytes:
        dev = f"cuda:{lat.device}"
        scratch = (torch.empty(nbytes, dtype=torch.uint8, device=dev), torch.empty(nbytes, dtype=torch.uint8, device=dev))
    send, recv = scratch
    plan = face_plan(sign, lat.dims[3], comm.rank, comm.world)
    q.qdp_field_get_timeslice(src, plan["send_slice"], send.data_ptr(), nbytes)
    q.qdp_lattice_sync(lat)                    # the face must be complete before the communication library reads it
    comm.sendrecv(send, plan["send_to"], recv, plan["recv_from"])
    # The communication (NCCL's kernels, or the loopback copy) runs on torch's current stream, and req.wait() only
    # orders that stream, not the host.  The unpack kernel goes to the lattice's own stream, which may be a
    # non-blocking one that has no implicit ordering with it: wait here until `recv` is really written.
    torch.cuda.current_stream(torch.device("cuda", lat.device)).synchronize()
    q.qdp_field_set_timeslice(dst, plan["fix_slice"], recv.data_ptr(), nbytes, subset)
    return scratch


def slab_norm2(q, f, subset: int, comm) -> float:
    return comm.allreduce_sum([q.qdp_norm2(f, subset)])[0]


def slab_inner(q, a, b, subset: int, comm) -> complex:
    z = q.qdp_inner(a, b, subset)
    re, im = comm.allreduce_sum([z.real, z.imag])
    return complex(re, im)
