"""Host-side logic of bench.py that needs no GPU: the N > 1 launch contract ("replicas only",
DESIGN.md section 8) under world_size 2 with the gloo backend, and the reference arm."""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(nproc, script_args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), *script_args]
    env = dict(os.environ, PYTHONPATH=ROOT, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_whole_job_value_gloo_world2(tmp_path):
    """Two gloo ranks report different times: every rank must see the MAX, and the whole-job value
    counts the units of both replicas over that time."""
    worker = tmp_path / "worker.py"
    worker.write_text(textwrap.dedent("""
        import json, sys
        import torch.distributed as dist
        import bench
        rank, world, local = bench.rank_env()
        dist.init_process_group("gloo")
        mine = [10.0 + 5.0 * rank, 100.0 - 30.0 * rank]
        got = bench.max_over_ranks(mine, dist, "cpu")
        value = bench.whole_job_value(1000, world, got[0])
        dist.barrier()
        dist.destroy_process_group()
        with open(sys.argv[1] + f"/rank{rank}.json", "w") as f:
            json.dump({"rank": rank, "world": world, "local": local, "got": got, "value": value}, f)
    """))
    r = _torchrun(2, [str(worker), str(tmp_path)])
    assert r.returncode == 0, r.stderr[-2000:]
    outs = [json.load(open(tmp_path / f"rank{k}.json")) for k in range(2)]
    for k, o in enumerate(outs):
        assert (o["rank"], o["world"], o["local"]) == (k, 2, k)
        assert o["got"] == [15.0, 100.0]                   # max over ranks of each entry
        assert abs(o["value"] - 2 * 1000 / 15e-3) < 1e-6   # both replicas' units over the slowest time


def test_reference_arm_prints_one_line_from_rank0_only():
    """`bench.py --impl reference` under torchrun with 2 ranks: rank 0 alone runs the oracle and prints
    the JSON line, the other rank exits 0 without work."""
    r = _torchrun(2, ["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1",
                      "--config", "C1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["gpu_launches"] == 0
    assert d["value"] > 0 and d["e2e"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["steps"] == 2 and d["warmup"] == 1 and d["higher_is_better"] is True


def test_single_process_defaults_and_algorithmic_bytes():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.rank_env() == (0, 1, 0) or "RANK" in os.environ
    assert bench.max_over_ranks([1.0, 2.0], None, "cpu") == [1.0, 2.0]
    V = 32 * 32 * 32 * 64
    alg = bench.algorithmic_bytes(V, 16)
    # bytes per site fp64
    assert alg["plaquette"] == V * 576 and alg["ape"] == V * 1152 and alg["axpy_hop_norm2"] == V * 960
    assert alg["hop_even"] == (V // 2) * 1536 and alg["norm2"] == V * 192 and alg["inner"] == V * 384
    assert alg["shift"] == V * 384
