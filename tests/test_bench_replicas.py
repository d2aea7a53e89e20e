"""bench.py's multi-rank logic on CPU (gloo, world_size 2): the path is "replicas only" (DESIGN.md
section 0, row (e)) -- every rank runs its own seeded replica, the elapsed time is the MAX over ranks,
the value is the whole-job aggregate, and only rank 0 prints.  `-m "not gpu"`."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%(port)d", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
ms = [10.0, 25.0][rank]                      # rank 1 is the slow replica
mx = bench.max_over_ranks(ms, dist, "cpu")
val = bench.aggregate_mlups(dist.get_world_size(), 1000000, 100, mx)
print(json.dumps({"rank": rank, "max_ms": mx, "value": val, "seed": bench.replica_seed(rank)}))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_aggregate_two_ranks_gloo():
    port = _free_port()
    code = WORKER % {"root": ROOT, "port": port}
    procs = [subprocess.Popen([sys.executable, "-c", code, str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["max_ms"] == 25.0                                   # max over ranks, on every rank
        assert abs(o["value"] - 2 * 1e6 * 100 / 25e-3 / 1e6) < 1e-9  # whole-job MLUPS of both replicas
    assert {o["seed"] for o in outs} == {1, 2}                       # independent seeded replicas


def test_single_rank_helpers():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.aggregate_mlups(1, 256 ** 3, 1000, 808.6) == pytest.approx(20748.0, rel=1e-3)


def test_algorithmic_bytes_match_design_table():
    """DESIGN.md section 6 table: bytes per lattice update per model"""
    import bench
    import workloads
    want = {"cfg1": 144, "cfg2": 160, "cfg3": 320, "cfg4": 304, "cfg5": 376}
    for k, v in want.items():
        a, b = bench.algorithmic_bytes(workloads.config(k))
        assert a + b == v, k
    a, b = bench.algorithmic_bytes(workloads.config("cfg4", precision=32))
    assert a + b == 152


def test_reference_arm_rank0_only_prints():
    """--impl reference under a 2-rank launch: rank 0 prints one JSON line, rank 1 exits 0 silently."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "3", "--warmup", "3", "--workload", "cfg1"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "MLUPS" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0
