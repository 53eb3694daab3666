"""N>1 host logic (replicas only) under a world_size-2 gloo group on CPU: the bench contract's
barrier + max-over-ranks timing and whole-job throughput, and the reference arm's "rank 0 only" rule."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["ELDR_ROOT"])
import torch.distributed as dist
from paper_2607_00466_b200 import replicas
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
dist.barrier()
ms = replicas.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")        # rank 1 is the slow one
dist.barrier()
out = {"rank": rank, "world": world, "ms": ms, "gbs": replicas.job_throughput_gbs(3.0e9, world, ms),
       "seed": replicas.replica_seed(100, rank)}
with open(os.path.join(os.environ["ELDR_OUT"], "rank%d.json" % rank), "w") as f:   # one file per rank: the ranks'
    json.dump(out, f)                                                           # stdout lines can interleave
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_max_over_ranks_and_job_throughput_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, ELDR_ROOT=ROOT, ELDR_OUT=str(tmp_path), MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    res = [json.loads((tmp_path / ("rank%d.json" % i)).read_text()) for i in range(2)]
    assert sorted(x["rank"] for x in res) == [0, 1]
    for x in res:
        assert x["world"] == 2
        assert x["ms"] == 15.0                                   # the slowest rank's time, on every rank
        assert x["gbs"] == pytest.approx(2 * 3.0e9 / 15.0e-3 / 1e9)   # both replicas' bytes over that time
    assert res[0]["seed"] != res[1]["seed"]


def test_single_process_needs_no_group():
    from paper_2607_00466_b200 import replicas
    assert replicas.max_over_ranks(7.5) == 7.5
    assert replicas.job_throughput_gbs(1e9, 1, 1.0) == pytest.approx(1000.0)


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the other ranks of `bench.py --impl reference` exit 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
