"""Data-parallel sharding of a packed document store across GPUs.

MaxSim is "embarrassingly parallel across documents ... no inter-GPU communication during scoring (only a
final concatenation of per-shard scores)".  A shard is a contiguous range of documents; ranges are
balanced by TOKENS (the HBM bytes a rank must stream), not by document count.  Queries (<= 64 KB) and PQ
codebooks / tables (<= 4 MB) are replicated.  No collective runs on the data path: the only communication is
the caller's optional gather of `scores[Q, B_rank]` and bench.py's max-over-ranks of the elapsed time.

Host logic only: no MaxSim arithmetic lives here.
"""
from __future__ import annotations

import numpy as np


def shard_bounds(offsets: np.ndarray, world_size: int) -> np.ndarray:
    """Document boundaries b[0..world_size] with b[0] = 0, b[-1] = B: rank r owns documents [b[r], b[r+1]).

    b[r] is the first document whose first token is at or after r*T/world_size (the same rule the dense
    kernel uses to cut per-CTA ranges), so every shard holds T/world_size tokens give or take one document.
    """
    off = np.asarray(offsets, dtype=np.int64)
    B, T = off.shape[0] - 1, int(off[-1])
    targets = (np.arange(world_size + 1, dtype=np.int64) * T) // world_size
    b = np.searchsorted(off[:-1], targets, side="left").astype(np.int64) if B else np.zeros(world_size + 1, np.int64)
    b[0], b[-1] = 0, B
    return np.maximum.accumulate(b)


def shard_documents(offsets: np.ndarray, world_size: int, rank: int):
    """(b_lo, b_hi, t_lo, t_hi, local_offsets) for `rank`; local_offsets is rebased to start at 0."""
    off = np.asarray(offsets, dtype=np.int64)
    b = shard_bounds(off, world_size)
    b_lo, b_hi = int(b[rank]), int(b[rank + 1])
    t_lo, t_hi = int(off[b_lo]), int(off[b_hi])
    return b_lo, b_hi, t_lo, t_hi, off[b_lo:b_hi + 1] - t_lo


def max_over_ranks(value: float, device=None) -> float:
    """MAX of a per-rank scalar over the default process group (identity when not initialised)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_scores(local_scores, world_size: int):
    """Concatenate per-shard scores[Q, B_rank] along documents on every rank (shards may differ in size)."""
    import torch
    import torch.distributed as dist

    if world_size == 1:
        return local_scores
    sizes = [torch.zeros(1, dtype=torch.int64, device=local_scores.device) for _ in range(world_size)]
    dist.all_gather(sizes, torch.tensor([local_scores.shape[1]], dtype=torch.int64, device=local_scores.device))
    parts = [torch.empty((local_scores.shape[0], int(s.item())), dtype=local_scores.dtype, device=local_scores.device)
             for s in sizes]
    mx = max(int(s.item()) for s in sizes)
    padded = torch.zeros((local_scores.shape[0], mx), dtype=local_scores.dtype, device=local_scores.device)
    padded[:, :local_scores.shape[1]] = local_scores
    bufs = [torch.empty_like(padded) for _ in range(world_size)]
    dist.all_gather(bufs, padded)
    for r in range(world_size):
        parts[r].copy_(bufs[r][:, :parts[r].shape[1]])
    return torch.cat(parts, dim=1)


def rank_seed(seed: int, rank: int) -> int:
    """Seed of rank `rank`'s synthetic shard in bench.py's weak-scaling runs (every rank owns its own B documents)."""
    return int(seed) + 1000 * int(rank)


def aggregate_throughput(units_per_rank: float, local_ms: float, device=None):
    """(whole-job units/s, max-over-ranks ms): every rank processed `units_per_rank` units in `local_ms` of device time;
    the job's time is the slowest rank's (bench.py's `value`; identity on one rank)."""
    import torch.distributed as dist

    world = dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1
    ms = max_over_ranks(local_ms, device)
    return world * units_per_rank / (ms * 1e-3), ms
