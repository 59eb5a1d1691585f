"""Host-side logic of bench.py's N > 1 path (replicas only), world_size 2 on gloo.

No GPU: the ranks exchange made-up timings through the same helper bench.py uses over NCCL, and
the reference arm is launched under torch.distributed.run to check that rank 0 alone prints."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    mine = [10.0 + rank, 100.0 - rank, 5.0 * (rank + 1)]
    out = bench.max_over_ranks(mine, world, torch.device("cpu"))
    q.put((rank, out))
    dist.destroy_process_group()


def test_max_over_ranks_world2_gloo():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0] == got[1] == [11.0, 100.0, 10.0]


def test_aggregate_counts_every_replica():
    sys.path.insert(0, ROOT)
    import bench

    one = bench.aggregate_mlups(1000, 10, 2.0, 1)
    assert one == pytest.approx(1000 * 10 / 2e-3 / 1e6)
    assert bench.aggregate_mlups(1000, 10, 2.0, 4) == pytest.approx(4 * one)


def test_reference_arm_under_torchrun_prints_once():
    """`bench.py --impl reference` launched like the driver does for N = 2: rank 0 prints the one
    JSON line, rank 1 exits 0 without work."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "cfg1",
           "--steps", "3", "--warmup", "3"]
    env = dict(os.environ, OMP_NUM_THREADS="2")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["steps"] == 3
    assert d["metric"] == "MLUPS" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
