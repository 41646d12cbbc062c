"""The N > 1 beam-sharded path (f4) on CPU: world_size 2 over gloo.  The broadcast of the input block, the beam
partition and the merge of the per-rank candidate lists are exercised with the ORACLE standing in for the GPU
library on each rank (the kernels are per beam, so a rank's result is the oracle's for its beams); rank 0 checks
the merged list against the un-sharded oracle."""
import os
import subprocess
import sys

import numpy as np

from paper_1612_06592_b200 import shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch
import torch.distributed as dist
from paper_1612_06592_b200 import shard, synth
from oracle import lofar_oracle as oracle
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = synth.small(S=4, B=5, K=16, k0=100, T=48, dtype="ci8", stec=(8.0, 12.0), n_pulses=4, kappa=4.0)
_, _, tau = synth.geometry(w)
X = torch.from_numpy(synth.generate_block(w, 0, tau=tau)) if rank == 0 else torch.zeros((w.S, 2, w.K, w.T, 2), dtype=torch.int8)
shard.broadcast_input(X, dist, 0)
b0, b1 = shard.beam_slice(w.B, world, rank)
pipe = oracle.OraclePipeline(tau=tau[b0:b1], stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
_, sigma, cands, total = pipe.run_block(X.numpy())
rec = np.zeros(len(cands), dtype=[("series", "<u4"), ("trial", "<u4"), ("sample", "<u8"), ("env", "<f4"), ("sigma", "<f4")])
for i, c in enumerate(cands):
    rec[i] = (c.series, c.trial, c.sample, c.env, c.sigma)
merged = shard.gather_records(rec, b0, w.D, dist, 0)
if rank == 0:
    full = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
    _, _, ref, _ = full.run_block(X.numpy())
    assert len(ref) == merged.size and merged.size > 0
    for c, m in zip(ref, merged):
        assert (c.series, c.trial, c.sample) == (int(m["series"]), int(m["trial"]), int(m["sample"]))
    print("OK", merged.size)
else:
    assert merged is None
dist.destroy_process_group()
'''


def test_beam_slice_partitions_every_beam_once():
    for B in (1, 5, 8, 24, 50):
        for world in (1, 2, 3, 4, 8):
            seen = []
            for r in range(world):
                b0, b1 = shard.beam_slice(B, world, r)
                assert 0 <= b0 <= b1 <= B
                seen += list(range(b0, b1))
            assert seen == list(range(B))
            sizes = [shard.beam_slice(B, world, r)[1] - shard.beam_slice(B, world, r)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_globalise_renumbers_series_and_beams():
    rec = np.zeros(2, dtype=[("series", "<u4"), ("sample", "<u8")])
    rec["series"] = [0, 5]
    assert shard.globalise(rec, 3, 4)["series"].tolist() == [12, 17]
    ev = np.zeros(1, dtype=[("beam", "<u4"), ("count", "<u4")])
    assert shard.globalise(ev, 3, 4)["beam"].tolist() == [3]


def test_broadcast_partition_merge_world2_gloo(tmp_path):
    wfile = tmp_path / "worker.py"
    wfile.write_text(WORKER.format(root=ROOT))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29741", str(wfile)]
    r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "OK " in r.stdout
