"""x3-slab decomposition of a lattice over several GPUs (multi-GPU is the
paper's "future work").  One process per GPU; rank r owns the time-slices [r L3/N, (r+1) L3/N) as a lattice of its own
(qdp_lattice_create with the local extent, which must be even so that local and global parity agree).

What the decomposition changes, and nothing else:
  * shift(f, +-3): the local shift wraps inside the slab, so its boundary slice is wrong; it is overwritten with the
    neighbouring rank's boundary slice -- ONE face exchange per shift (qdp_field_get_timeslice -> send/recv ->
    qdp_field_set_timeslice).  Shifts along x0, x1, x2 are purely local.
  * global sums: all-reduce of the local doubles.
The fused neighbour-reading kernels (hop, plaquette) read their x3 neighbours inside the kernel and wrap inside the slab,
so on a slab they are evaluated the way the paper evaluates everything -- expression by expression, each shift along x3
one halo exchange (slab_hop, slab_plaquette below): the parts that never leave a time-slice stay fused (the spatial
hops, the spatial plaquette, the whole spatial APE step), the x3 terms are built from slab_shift and the site-local
products.  That is several passes instead of one: it is the functional multi-GPU path, not a tuned one; bench.py runs
replicas only (BASELINE.json: one GPU).

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


def _opposite(subset: int) -> int:
    return (0, 2, 1)[subset]


def slab_ape_smear_step(q, u_out, u_in, alpha: float, subset: int = 0):
    """The spatial APE step (t_dir = 3) on a slab: its staples never leave the time-slice, so the fused kernel is already
    the global answer and nothing is exchanged.  (The 4-D step reads x3 neighbours and is not offered on slabs.)"""
    q.qdp_ape_smear_step(u_out, u_in, alpha, 3, subset)


def slab_hop(q, chi, u, psi, subset: int, comm, work=None):
    """chi(x) = sum_mu [U_mu(x) psi(x+mu) + U_mu^dag(x-mu) psi(x-mu)] of the GLOBAL lattice on the sites of `subset`;
    chi, u, psi: this rank's slab fields.  Spatial directions: one fused local kernel.  x3: psi(x+3) by slab_shift then the
    colour rotation; (U_3^dag psi) formed at the source sites (the other parity) then moved by slab_shift.  Two face
    exchanges of one spinor time-slice each.  `work`: two spinor fields of the slab (allocated if None), returned."""
    lat = psi.lat
    if work is None:
        work = (q.qdp_field_alloc(lat, q.QDP_FERMION, psi.prec), q.qdp_field_alloc(lat, q.QDP_FERMION, psi.prec))
    t1, t2 = work
    q.qdp_smear_hop(chi, 0.0, 1.0, u, psi, 3, subset)                 # mu = 0, 1, 2
    slab_shift(q, t1, psi, 3, +1, subset, comm)                       # t1(x) = psi(x + 3)
    q.qdp_matvec(t2, u, 3, False, t1, -1, 1, subset)                  # U_3(x) psi(x + 3)
    q.qdp_axpby(chi, 1.0, chi, 1.0, t2, subset)
    q.qdp_matvec(t1, u, 3, True, psi, -1, 1, _opposite(subset))       # (U_3^dag psi)(y) at the source sites y = x - 3
    slab_shift(q, t2, t1, 3, -1, subset, comm)                        # t2(x) = (U_3^dag psi)(x - 3)
    q.qdp_axpby(chi, 1.0, chi, 1.0, t2, subset)
    return work


def slab_plaquette(q, u, comm, work=None):
    """[all, spatial, temporal] plaquette of the GLOBAL lattice, normalised as qdp_plaquette.  The spatial planes never
    leave a time-slice: the fused kernel's spatial sum is exact on a slab.  The three temporal planes need U_mu(x + 3): one
    slab_shift of the gauge field (one face exchange), then per plane P = U_mu(x) U_3(x+mu), Q = U_3(x) U_mu(x+3) and
    sum_x Re tr(P Q^dag).  `work`: (gauge field, colour matrix, colour matrix) of the slab, returned as the second value."""
    import numpy as np
    lat = u.lat
    if work is None:
        work = (q.qdp_field_alloc(lat, q.QDP_GAUGE, u.prec), q.qdp_field_alloc(lat, q.QDP_COLOR_MATRIX, u.prec),
                q.qdp_field_alloc(lat, q.QDP_COLOR_MATRIX, u.prec))
    us, P, Q = work
    v_local = lat.volume
    spatial = float(q.qdp_plaquette(u)[1]) * 9.0 * v_local            # back to the plain sum over this slab
    slab_shift(q, us, u, 3, +1, 0, comm)                              # us(x) = u(x + 3)
    temporal = 0.0
    for mu in range(3):
        q.qdp_matmul(P, 0, u, mu, False, u, 3, False, mu, +1)
        q.qdp_matmul(Q, 0, u, 3, False, us, mu, False, -1, 1)
        temporal += q.qdp_expr_sum_trace_mul(P, 0, False, Q, 0, True).real
    sp, tp, vol = comm.allreduce_sum([spatial, temporal, float(v_local)])
    return np.array([(sp + tp) / (18.0 * vol), sp / (9.0 * vol), tp / (9.0 * vol)]), work
