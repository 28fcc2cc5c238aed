"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): the path is "replicas only"
(DESIGN.md Sec. 7), so the only multi-rank logic is the barrier, the max-over-ranks timing and the
whole-job aggregate; rank != 0 of the reference arm exits without work."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
dist.barrier()
ms = bench.max_over_ranks(10.0 * (rank + 1), dist, torch.device("cpu"))     # rank 1 is the slow replica
assert ms == 10.0 * world, ms
v = bench.job_gflops(1e9, world, ms)
assert abs(v - world * 1e9 / (ms * 1e-3) / 1e9) < 1e-9
if rank == 0:
    print("OK %%d %%.1f %%.3f" %% (world, ms, v))
dist.destroy_process_group()
""" % ROOT


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_max_over_ranks_and_job_value_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "OK 2 20.0 100.000" in r.stdout, r.stdout


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode == 0 and r.stdout.strip() == "", (r.stdout, r.stderr[-500:])


def test_single_rank_needs_no_process_group():
    import torch
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, torch.device("cpu")) == 3.5
    assert bench.job_gflops(2e9, 1, 1.0) == pytest.approx(2000.0)
