"""Host-side multi-GPU plumbing for bench.py (one process per GPU, torch.distributed).

The path shards by independent problems ("large-scale parallel evaluation ... on many
dense ... matrices"): every rank runs its own replica / share of block columns and there is no
data-path collective.  Only timing and work counters are reduced: max over ranks for time, sum for work.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of rank r's replica of a workload (weak scaling: a different geometry per GPU)."""
    return int(base_seed) + 100 * int(rank)


def aggregate(ms_total: float, work: float, device) -> tuple[float, float]:
    """(max over ranks of ms_total, sum over ranks of work).  No-op without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_total), float(work)
    t = torch.tensor([ms_total], dtype=torch.float64, device=device)
    w = torch.tensor([work], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return float(t.item()), float(w.item())


def shard_columns(dim: np.ndarray, world: int, rank: int) -> np.ndarray:
    """Longest-processing-time partition of block columns by m_i^3; returns
    the sorted column ids of `rank`.  Deterministic, so every rank computes the same partition."""
    cost = dim.astype(np.float64) ** 3
    order = np.lexsort((np.arange(len(dim)), -cost))
    load = np.zeros(world)
    owner = np.empty(len(dim), dtype=np.int64)
    for i in order:
        r = int(np.argmin(load))
        owner[i] = r
        load[r] += cost[i]
    return np.sort(np.nonzero(owner == rank)[0]).astype(np.int32)
