"""The N > 1 path of bench.py on CPU: two gloo ranks on 127.0.0.1.  The hot path does not shard (north_star: one GPU,
no collectives; replicas only), so what exists to test is the launch contract: per-rank
replicas draw their own seeded inputs, timing is the max over ranks, and only rank 0 of the reference arm prints."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
local_ms = 100.0 + 50.0 * rank                       # rank 1 is the slow one
mx = bench.max_over_ranks(local_ms, world, torch.device("cpu"))
cfg, X, F = bench.make_inputs("c1", rank)
dist.barrier()
open(os.path.join(os.environ["HH_TEST_OUT"], "rank%%d.json" %% rank), "w").write(
    json.dumps({"rank": rank, "world": world, "max": mx, "x0": float(X[0, 0]), "f0": float(F[0, 0]), "n": len(X)}))
dist.destroy_process_group()
""" % ROOT


def test_two_gloo_ranks_replicas_and_max_over_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, OMP_NUM_THREADS="1", HH_TEST_OUT=str(tmp_path))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29531", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    rows = [json.loads((tmp_path / ("rank%d.json" % k)).read_text()) for k in range(2)]
    assert [d["rank"] for d in rows] == [0, 1] and all(d["world"] == 2 for d in rows)
    assert all(d["max"] == 150.0 for d in rows)                      # max over ranks, on every rank
    assert rows[0]["n"] == rows[1]["n"] == 2048
    assert rows[0]["x0"] != rows[1]["x0"] and rows[0]["f0"] != rows[1]["f0"]   # independent replicas, own seeds


def test_reference_arm_prints_one_line_on_rank0_only():
    env = dict(os.environ)
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1", "--steps", "1", "--warmup", "0"]
    r0 = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=dict(env, RANK="0", WORLD_SIZE="2"))
    assert r0.returncode == 0, r0.stderr[-2000:]
    line = json.loads([l for l in r0.stdout.splitlines() if l.startswith("{")][-1])
    assert line["impl"] == "reference" and line["unit"] == "particles/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    r1 = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=dict(env, RANK="1", WORLD_SIZE="2"))
    assert r1.returncode == 0 and not [l for l in r1.stdout.splitlines() if l.startswith("{")]
