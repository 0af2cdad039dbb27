"""bench.py --gpus N runs N independent replicas (a linearizable queue does not
shard); the only communication is the SUM / MAX reduction that forms the JSON line.  This drives
that reduction with two CPU processes over gloo, and checks the reference arm's rank gating."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
sums, maxes = bench.aggregate_replicas(dist, "cpu", [100.0 * (r + 1), 7.0], [0.5 + r, 3.0 - r])
if r == 0:
    print(json.dumps({{"sums": sums, "maxes": maxes, "world": dist.get_world_size()}}))
dist.destroy_process_group()
"""


def test_replica_aggregation_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29731", str(script)],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    res = json.loads(line)
    assert res["world"] == 2
    assert res["sums"] == [300.0, 14.0]          # units: SUM over ranks
    assert res["maxes"] == [1.5, 3.0]            # time: MAX over ranks


def test_single_process_aggregation_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    sums, maxes = bench.aggregate_replicas(None, "cpu", [1.0, 2.0], [3.0])
    assert sums == [1.0, 2.0] and maxes == [3.0]


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=120, env=env, cwd=ROOT)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_reference_arm_prints_the_contract_line():
    # `bench.py --impl reference` = the oracle's mutex+deque queue timed on the host cores (tier rule): one JSON line
    # with the base contract's keys plus impl / cpu_baseline / e2e, no GPU needed.
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "impl", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["value"] > 0 and line["unit"] == "Mops/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in line["config"]
