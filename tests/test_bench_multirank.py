"""The N > 1 path of bench.py on CPU (gloo, world_size 2).  The hot path does not shard (north_star: "no sharding
or collectives" -> replicas only), so what there is to cover is the launch contract: max-over-ranks timing,
whole-job aggregation, and the reference arm printing exactly one line from rank 0 under torchrun."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
ms = bench.max_over_ranks(10.0 + 5.0 * r, dist, "cpu")
assert ms == 15.0, ms
v = bench.aggregate_value(1000, dist.get_world_size(), ms)
assert abs(v - 2 * 1000 / 15e-3) < 1e-6
dist.barrier()
if r == 0:
    print("OK", ms, v)
dist.destroy_process_group()
'''


def _torchrun(args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731"] + args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_aggregation_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    assert "OK 15.0" in r.stdout


def test_reference_arm_under_torchrun_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--config", "0"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
