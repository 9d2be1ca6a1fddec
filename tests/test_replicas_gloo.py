"""Multi-process CPU test (gloo, world_size 2) of the only cross-rank logic the bench has: "replicas
only" - a timing barrier, max-over-ranks of the device time, sum-over-ranks of units."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["ARKCOS_ROOT"])
from paper_1211_3556_b200 import replicas
rank, local_rank, world = replicas.env_world()
dist = replicas.init("gloo")
assert dist is not None and dist.get_world_size() == world == 2 and dist.get_rank() == rank
replicas.barrier(dist)
# rank r "measured" (10 + 5 r) ms for (100 + r) units
t, u = replicas.aggregate(dist, 10.0 + 5.0 * rank, 100.0 + rank)
assert t == 15.0 and u == 201.0, (t, u)
v = replicas.throughput(u, t)
assert abs(v - 201.0 / 15e-3) < 1e-6
replicas.barrier(dist)
dist.destroy_process_group()
print(json.dumps({"rank": rank, "t": t, "u": u}))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_world_size_2_gloo_aggregation():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), ARKCOS_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        try:
            out, err = p.communicate(timeout=180)
        except subprocess.TimeoutExpired:
            p.kill()
            pytest.fail("gloo worker timed out")
        assert p.returncode == 0, err[-2000:]
        outs.append(out)
    assert '"t": 15.0' in outs[0] and '"u": 201.0' in outs[1]


def test_single_process_is_a_no_op():
    from paper_1211_3556_b200 import replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert replicas.env_world() == (0, 0, 1)
    assert replicas.init("gloo") is None
    replicas.barrier(None)
    assert replicas.aggregate(None, 3.0, 7.0) == (3.0, 7.0)


def test_reference_arm_runs_on_rank0_only():
    """bench.py --impl reference under torchrun: ranks != 0 exit 0 without work (tier contract)."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="1")
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert res.returncode == 0 and res.stdout.strip() == ""
