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


# ---- sharding one workload over ranks ---------------------------------
# Submatrices are independent units, so the block columns are partitioned over the ranks (LPT on m_i^3, shard_columns),
# H is replicated (<= 0.6 GB), every rank runs a1-a4 on its own columns, and the ONE exchange step of the path is an
# all-gather of the column-owned blocks of the result; symmetrisation and D = 1/2 (I - R) then run on the gathered
# block-sparse matrix (every rank holds the whole D afterwards, as every rank holds the whole H).

def column_value_index(n_blk, row_ptr, col_idx, val_ptr, cols) -> np.ndarray:
    """Element indices (into the block-CSR value array) of the blocks (j, i) of the listed block columns i, column by
    column, rows ascending: the layout of a rank's packed send buffer.  Integer work on host arrays."""
    row_ptr = np.asarray(row_ptr, dtype=np.int64)
    col_idx = np.asarray(col_idx, dtype=np.int64)
    val_ptr = np.asarray(val_ptr, dtype=np.int64)
    out = []
    for i in np.asarray(cols, dtype=np.int64):
        for j in col_idx[row_ptr[i]:row_ptr[i + 1]]:          # structurally symmetric: rows of column i = columns of row i
            p = row_ptr[j] + np.searchsorted(col_idx[row_ptr[j]:row_ptr[j + 1]], i)
            out.append(np.arange(val_ptr[p], val_ptr[p + 1], dtype=np.int64))
    return np.concatenate(out) if out else np.zeros(0, dtype=np.int64)


def exchange_columns(R_local: torch.Tensor, idx_by_rank, rank: int, world: int) -> torch.Tensor:
    """All-gather of column-owned blocks: every rank sends R_local[idx_by_rank[rank]] and receives the other ranks'
    blocks into the same value array.  idx_by_rank: list of int64 index tensors (on R_local's device), identical on
    every rank.  Returns R_local with every listed element filled.  NCCL over NVLink on GPUs, gloo in the CPU tests."""
    if world == 1:
        return R_local
    n_max = max(int(ix.numel()) for ix in idx_by_rank)         # all_gather wants equal sizes: pad to the largest share
    send = torch.zeros(n_max, dtype=R_local.dtype, device=R_local.device)
    send[:idx_by_rank[rank].numel()] = R_local.index_select(0, idx_by_rank[rank])
    recv = torch.empty(world * n_max, dtype=R_local.dtype, device=R_local.device)
    dist.all_gather_into_tensor(recv, send)
    for r, ix in enumerate(idx_by_rank):
        if r != rank:
            R_local.index_copy_(0, ix, recv[r * n_max:r * n_max + ix.numel()])
    return R_local


def sharded_density(sm, wl_host, A, P, x_dtype, rank: int, world: int, mu=0.0, scale_mode="global", max_iter=20,
                    tol=0.0, symmetrise=True, switch_iter=-1, state=None):
    """The whole path with the block columns sharded over `world` ranks (one process per GPU): a2-a4 on this rank's
    columns through the C ABI, exchange_columns, then symmetrise + density on the gathered matrix.  `sm` is the
    binding module, `wl_host` the host copy of the CSR arrays (index maps), A / P the device pattern (replicated).
    Returns (D, trace, state); pass `state` back in to reuse the partition, index maps and buffers."""
    dev = A.device
    if state is None:
        dim = P.dim.cpu().numpy()
        mine = shard_columns(dim, world, rank)
        order = P.order.cpu().numpy()
        pos = np.argsort(np.argsort(-P.dim_pad.cpu().numpy().astype(np.int64), kind="stable"), kind="stable")
        mine = mine[np.argsort(pos[mine], kind="stable")]                  # this rank's columns, largest first
        idx = [torch.as_tensor(column_value_index(wl_host.n_blk, wl_host.row_ptr, wl_host.col_idx, wl_host.val_ptr,
                                                  np.sort(shard_columns(dim, world, r))), device=dev) for r in range(world)]
        cols, col_off, n = sm.sm_plan_columns(P, mine)
        ne = sm.packed_elems(P, mine)
        state = dict(mine=np.sort(mine), cols=cols, col_off=col_off, n=n, ne=ne, idx=idx,
                     ws=torch.empty(sm.sm_sign_ws_bytes(P, n, ne, x_dtype), dtype=torch.uint8, device=dev),
                     R=torch.zeros(A.n_vals, dtype=torch.float64, device=dev), X=None, order=order)
    st = state
    st["X"], scale = sm.sm_gather(A, P, st["cols"], st["col_off"], st["n"], mu, scale_mode, x_dtype, X=st["X"])
    iters, res = sm.sm_sign_ns(P, st["cols"], st["col_off"], st["n"], st["ne"], x_dtype, st["X"], max_iter, tol,
                               ws=st["ws"], switch_iter=switch_iter)
    s_dtype = "f16" if switch_iter >= 0 else x_dtype
    sm.sm_scatter(A, P, st["cols"], st["col_off"], st["n"], s_dtype, st["X"], "f64", R=st["R"], symmetrise=False)
    exchange_columns(st["R"], st["idx"], rank, world)
    if symmetrise:
        sm.sm_symmetrise(A, P, st["R"])
    D, trace = sm.sm_density_from_sign(A, P, st["R"])
    st["iters"], st["residual"] = iters, res
    return D, trace, st
