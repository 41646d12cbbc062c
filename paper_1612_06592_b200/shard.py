"""Beam-sharded multi-GPU operation (row f4 of SURVEY.md 8(f); every node needs all station
data, the beams are spread over the GPUs).  Host-side plumbing only -- partition, the one collective (a broadcast
of the input block, the paper's data-distribution step) and the merge of the per-rank candidate lists; the
arithmetic stays in the CUDA library.  torch.distributed is the transport: NCCL between GPUs, gloo in the CPU
tests."""
from __future__ import annotations

import numpy as np


def beam_slice(B: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous beams [b0, b1) of `rank`: the first B % world ranks take one beam more."""
    base, extra = divmod(B, world)
    b0 = rank * base + min(rank, extra)
    return b0, b0 + base + (1 if rank < extra else 0)


def broadcast_input(X, dist, src: int = 0):
    """The input block reaches every rank ("all data from all stations have to be send to all nodes").
    X: a torch tensor resident where the backend works (device for NCCL, host for gloo); overwritten on ranks
    other than src."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.broadcast(X, src)
    return X


def globalise(rec: np.ndarray, b0: int, D: int) -> np.ndarray:
    """Candidate (or event) records of a rank that holds beams b0.. -> numbering of the whole beam set."""
    out = rec.copy()
    if "series" in out.dtype.names:
        out["series"] = out["series"] + b0 * D
    if "beam" in out.dtype.names:
        out["beam"] = out["beam"] + b0
    return out


def gather_records(rec: np.ndarray, b0: int, D: int, dist, dst: int = 0):
    """All ranks' records on rank dst, renumbered and in (beam, sample) order (ranks hold increasing beams, each
    list is already sorted).  Returns None on the other ranks."""
    mine = globalise(rec, b0, D)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return mine
    parts = [None] * dist.get_world_size() if dist.get_rank() == dst else None
    dist.gather_object(mine, parts, dst=dst)
    if dist.get_rank() != dst:
        return None
    return np.concatenate(parts)
