"""The N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only, no data-path collective.

What runs with more than one rank is (a) the max-over-ranks of the per-rank time and the whole-job rate
built from it, and (b) the launch contract of the reference arm (rank 0 prints one JSON line, the other
ranks exit 0 without work).  Both are exercised here without a GPU.
"""
import json
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = [10.0, 12.5][rank]                                   # rank 1 is the slow replica
    worst = bench.reduce_max(ms, dist, torch.device("cpu"))
    dist.barrier()
    out[rank] = (worst, bench.whole_job_rate(1000, 4, worst, world))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_gloo():
    import torch.multiprocessing as mp
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
        res = dict(out)
    assert res[0] == res[1]
    worst, rate = res[0]
    assert worst == 12.5
    assert rate == pytest.approx(2 * 1000 * 5 * 4 / 12.5e-3)


def test_single_rank_reduce_is_identity():
    import bench
    assert bench.reduce_max(3.25, None, None) == 3.25
    assert bench.whole_job_rate(10, 2, 1.0, 1) == pytest.approx(10 * 5 * 2 / 1e-3)


def test_reference_arm_under_torchrun_two_ranks():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl",
           "reference", "--steps", "1", "--warmup", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                     # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
