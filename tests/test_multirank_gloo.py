"""N>1 path (replicas only, no data-path collective): the host-side logic bench.py runs
under torchrun -- rendezvous, barrier, MAX-over-ranks of the timing, whole-job rate, rank-0-only reporting --
exercised with two CPU processes over gloo."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["EV_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
dist.barrier()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")     # rank 1 is the slow replica
rate = bench.whole_job_rate(60, world, ms)
if rank == 0:
    print(json.dumps({"ms": ms, "rate": rate, "world": world}), flush=True)
dist.barrier()
dist.destroy_process_group()
"""


def _free_port():
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_replicas_max_over_ranks_and_whole_job_rate_world2(tmp_path):
    pytest.importorskip("torch")
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    env = dict(os.environ, EV_ROOT=ROOT, OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(w)]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, "exactly one JSON line, from rank 0"
    d = json.loads(lines[0])
    assert d["world"] == 2 and d["ms"] == 15.0                   # the slowest rank decides
    assert abs(d["rate"] - 2 * 60 / 15e-3) < 1e-6                # units of ALL ranks / max time


def test_reference_arm_other_ranks_exit_without_work():
    """bench.py --impl reference under torchrun: rank != 0 exits 0 before importing the oracle or torch."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], env=env,
                       capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
