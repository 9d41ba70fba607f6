"""qdp_sum_noalloc: the lattice sum for callers that are not allowed to allocate device memory.

Who needs it: code that only ever receives raw device pointers and a stream -- a plug-in living inside
a framework whose caching allocator has taken the whole GPU, or a latency-bound loop that cannot afford the
device-wide synchronisation behind cudaMalloc / cudaFree.  Such a caller cannot even create a qdp_lattice
(that allocates scratch, staging and pinned memory), so qdp_sum is out of reach for it.  The no-alloc entry
point keeps its per-block partial sums in a fixed 36,864-byte __device__ array inside the library instead.

What is checked here: on two calls in a row (the second one finds the first one's partial sums still in the
shared scratch and must not be disturbed by them) the result equals the existing path's, qdp_sum, within the
tolerance the reduction tests use -- and, since the summation order is the same, bit for bit; a size beyond
what the fixed array holds is refused with a message that names the limit.

The file sorts last on purpose (pytest -x stops at the first failure, so a failure here hides nothing), and
it builds everything it needs itself, so it passes alone in a fresh process as well as after the other tests.
"""
import numpy as np
import pytest

import synth
from parity import TOL_SUM

pytestmark = pytest.mark.gpu

NCOMP = {0: 9, 1: 36, 2: 12}    # colour matrix, gauge field, fermion


def _host_field(dims, kind, seed):
    return {0: synth.color_matrix, 1: synth.gauge_hot, 2: synth.spinor}[kind](dims, seed)


@pytest.mark.parametrize("dims", [(4, 2, 6, 4), (10, 6, 4, 2), (16, 16, 16, 32)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sum_noalloc_matches_qdp_sum_on_two_calls_in_a_row(qdp, dims, prec):
    import torch
    lat = qdp.qdp_lattice_create(dims)
    p = qdp.QDP_F64 if prec == "f64" else qdp.QDP_F32
    stream = torch.cuda.Stream()
    for kind in (2, 1, 0):      # different ncomp from call to call: the stale scratch of a wider call stays behind
        fields = []
        for call in range(2):   # two calls in a row, on different data
            host = synth.round_to(_host_field(dims, kind, synth.BASE_SEED + 77 + call), prec)
            fields.append((host, qdp.field_from_host(lat, kind, host)))
        qdp.qdp_lattice_sync(lat)
        for sub in (0, 1, 2):
            outs = [torch.full((2 * NCOMP[kind],), float("nan"), dtype=torch.float64, device="cuda") for _ in fields]
            torch.cuda.synchronize()
            for (host, f), out in zip(fields, outs):      # back to back on one stream, no host sync in between
                nbytes = qdp.qdp_field_bytes(lat, kind, p)
                qdp.qdp_sum_noalloc(dims, NCOMP[kind], p, f.storage.data_ptr(), nbytes, sub, out.data_ptr(),
                                    stream.cuda_stream)
            stream.synchronize()
            for (host, f), out in zip(fields, outs):
                got = out.cpu().numpy()
                got = (got[0::2] + 1j * got[1::2])
                want = qdp.qdp_sum(f, sub).ravel()         # the existing path
                scale = np.sqrt(float((np.abs(host.astype(np.complex128)) ** 2).sum()) * synth.volume(dims))
                tol = TOL_SUM["f64"] if prec == "f64" else 1e-12    # the bar of test_reductions
                assert np.abs(got - want).max() <= tol * scale, (kind, sub)
                assert np.array_equal(got, want), (kind, sub)       # same blocks, same order: identical bits


def test_sum_noalloc_refuses_what_the_fixed_scratch_cannot_hold(qdp):
    import torch
    dims = (4, 4, 4, 4)
    buf = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    out = torch.zeros(128, dtype=torch.float64, device="cuda")
    with pytest.raises(qdp.QdpError) as e:
        qdp.qdp_sum_noalloc(dims, 37, qdp.QDP_F64, buf.data_ptr(), 1 << 16, 0, out.data_ptr())
    assert e.value.code == -1 and "36" in str(e.value) and "scratch" in str(e.value)
    with pytest.raises(qdp.QdpError) as e:      # a size that does not belong to this lattice
        qdp.qdp_sum_noalloc(dims, 12, qdp.QDP_F64, buf.data_ptr(), 100, 0, out.data_ptr())
    assert e.value.code == -1
    with pytest.raises(qdp.QdpError) as e:
        qdp.qdp_sum_noalloc((4, 4, 3, 4), 12, qdp.QDP_F64, buf.data_ptr(), 100, 0, out.data_ptr())
    assert e.value.code == -2
    assert float(out.abs().sum()) == 0.0        # nothing was written
