"""N > 1 plumbing of bench.py on CPU (gloo, world_size 2): the aggregation of the timing — max over ranks of the device
time, sum over ranks of the work — which both --parallel modes use (dd: the decomposed operator, strong scaling, the
default; replicas: N independent copies), and the rule that only rank 0 runs / prints the reference arm.  The exchange
of the decomposed operator itself is covered by tests/test_decomposition.py (gloo) and tests/test_gpu_dd.py."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
ms, units = bench.reduce_over_ranks([3.0, 7.5][r], [1000, 1024][r], dist, "cpu")
lone = bench.reduce_over_ranks(2.0, 10)          # no process group: passthrough
open(os.path.join({out!r}, "rank%d.json" % r), "w").write(json.dumps({{"rank": r, "ms": ms, "units": units, "lone": lone}}))
dist.destroy_process_group()
'''


def test_replica_aggregation_max_time_sum_work_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, out=str(tmp_path)))
    import socket

    with socket.socket() as sk:  # a free rendezvous port
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads((tmp_path / ("rank%d.json" % k)).read_text()) for k in (0, 1)]  # one file per rank
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["ms"] == 7.5 and l["units"] == 2024 and l["lone"] == [2.0, 10]


def test_reference_arm_only_rank0_works(tmp_path):
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
