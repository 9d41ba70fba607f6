"""Host logic of the x3-slab decomposition (paper_1111_5596_b200/slab.py) under world_size 2
with the gloo backend on CPU: neighbour ranks, the face plan of a shift along x3, the exchange and the all-reduce.
The local data movement is done with numpy / the oracle here (tests may use the oracle); on the GPU it is the two
time-slice kernels, covered by tests/test_gpu_slab.py."""
import json
import os
import socket
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_plan_is_pure_logic():
    sys.path.insert(0, ROOT)
    from paper_1111_5596_b200 import slab
    assert slab.neighbor_ranks(0, 4) == (1, 3) and slab.neighbor_ranks(3, 4) == (0, 2) and slab.neighbor_ranks(0, 1) == (0, 0)
    assert slab.local_dims((8, 4, 6, 16), 4) == (8, 4, 6, 4)
    for bad in ((8, 4, 6, 16), 3), ((8, 4, 6, 12), 4):      # not divisible; odd local extent
        with pytest.raises(ValueError):
            slab.local_dims(*bad)
    assert slab.face_plan(+1, 4, 1, 4) == {"send_slice": 0, "send_to": 0, "recv_from": 2, "fix_slice": 3}
    assert slab.face_plan(-1, 4, 1, 4) == {"send_slice": 3, "send_to": 2, "recv_from": 0, "fix_slice": 0}
    c = slab.LoopbackComm()
    assert c.allreduce_sum([1.5, 2.0]) == [1.5, 2.0]


def test_shift_along_x3_and_sums_over_two_gloo_ranks(tmp_path):
    worker = tmp_path / "worker.py"
    worker.write_text(textwrap.dedent("""
        import json, sys
        import numpy as np
        import torch
        import torch.distributed as dist
        import oracle, synth
        from paper_1111_5596_b200 import slab
        dist.init_process_group("gloo")
        comm = slab.TorchComm(dist)
        gdims = (4, 2, 6, 8)
        ldims = slab.local_dims(gdims, comm.world)
        n = gdims[0] * gdims[1] * gdims[2]                       # sites per time-slice (lex order: x3 slowest)
        Lt = ldims[3]
        full = synth.spinor(gdims, 1301)
        mine = full[comm.rank * Lt * n:(comm.rank + 1) * Lt * n].copy()
        ok = True
        for sign in (+1, -1):
            for subset in (0, 1, 2):
                want = oracle.shift(gdims, full, 3, sign, subset, dst=np.full_like(full, 9.0))
                want = want[comm.rank * Lt * n:(comm.rank + 1) * Lt * n]
                dst = oracle.shift(ldims, mine, 3, sign, subset, dst=np.full_like(mine, 9.0))   # wraps inside the slab
                plan = slab.face_plan(sign, Lt, comm.rank, comm.world)
                s = plan["send_slice"]
                send = torch.from_numpy(mine[s * n:(s + 1) * n].copy())
                recv = torch.empty_like(send)
                comm.sendrecv(send, plan["send_to"], recv, plan["recv_from"])
                f = plan["fix_slice"]
                face = recv.numpy()
                if subset:                                            # write only the subset's sites of the fixed slice
                    par = oracle.parity_mask(ldims)[f * n:(f + 1) * n]
                    keep = par == (subset == 2)
                    dst[f * n:(f + 1) * n][keep] = face[keep]
                else:
                    dst[f * n:(f + 1) * n] = face
                ok = ok and np.array_equal(dst, want)
        total = comm.allreduce_sum([oracle.norm2(ldims, mine)])[0]
        ok = ok and abs(total - oracle.norm2(gdims, full)) <= 1e-12 * total
        dist.barrier()
        dist.destroy_process_group()
        with open(sys.argv[1] + f"/rank{comm.rank}.json", "w") as fh:
            json.dump({"ok": bool(ok), "rank": comm.rank, "world": comm.world}, fh)
    """))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(worker), str(tmp_path)]
    env = dict(os.environ, PYTHONPATH=ROOT + os.pathsep + os.path.join(ROOT, "tests"), OMP_NUM_THREADS="1")
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-3000:]
    outs = [json.load(open(tmp_path / f"rank{k}.json")) for k in range(2)]
    assert all(o["ok"] and o["world"] == 2 for o in outs) and [o["rank"] for o in outs] == [0, 1]
