"""World-size-2 gloo test (CPU) of the N>1 host logic bench.py uses: rank seeds, max/sum reduction,
and the LPT column partition."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2205_14741_b200 import dist_util


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, work = dist_util.aggregate(10.0 + 5.0 * rank, 100.0 * (rank + 1), torch.device("cpu"))
    dim = np.array([100, 400, 250, 250, 90, 410, 30, 77], dtype=np.int32)
    mine = dist_util.shard_columns(dim, world, rank)
    out[rank] = (ms, work, mine.tolist(), dist_util.rank_seed(1002, rank))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation_and_partition():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    assert out[0][:2] == out[1][:2] == (15.0, 300.0)          # max of times, sum of work
    a, b = out[0][2], out[1][2]
    assert sorted(a + b) == list(range(8)) and not set(a) & set(b)
    dim = np.array([100, 400, 250, 250, 90, 410, 30, 77], dtype=np.float64) ** 3
    la, lb = dim[a].sum(), dim[b].sum()
    assert abs(la - lb) / (la + lb) < 0.1                      # balanced by m^3
    assert out[0][3] == 1002 and out[1][3] == 1102


def _shard_worker(rank, world, port, out):
    """f4 host logic on CPU: every rank computes ITS block columns (with the oracle standing in for the GPU stages),
    the column-owned blocks are exchanged by dist_util.exchange_columns (gloo all-gather), and the assembled matrix
    must equal the one a single process computes."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle as orc
    from workloads.generator import make_config
    wl = make_config(0)
    dim = np.array([wl.blk_size[wl.col_idx[wl.row_ptr[i]:wl.row_ptr[i + 1]]].sum() for i in range(wl.n_blk)])
    idx = [torch.as_tensor(dist_util.column_value_index(wl.n_blk, wl.row_ptr, wl.col_idx, wl.val_ptr,
                                                        dist_util.shard_columns(dim, world, r))) for r in range(world)]
    mine = dist_util.shard_columns(dim, world, rank)
    d_mine, _ = orc.density_columns(wl, cols=mine)
    R = torch.from_numpy(d_mine.copy())
    dist_util.exchange_columns(R, idx, rank, world)
    out[rank] = (R.numpy().copy(), [int(ix.numel()) for ix in idx], mine.tolist())
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharded_columns_assemble_the_single_process_result():
    from oracle import oracle as orc
    from workloads.generator import make_config
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_shard_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    wl = make_config(0)
    d_all, _ = orc.density_columns(wl)
    for r in range(world):
        assert np.array_equal(out[r][0], d_all)               # bit-identical: every element comes from exactly one rank
    sizes = out[0][1]
    assert sum(sizes) == d_all.size                           # the ranks' index sets partition the value array
    assert sorted(out[0][2] + out[1][2]) == list(range(wl.n_blk))


def test_column_value_index_is_a_partition_and_matches_the_mask():
    from oracle import oracle as orc
    from workloads.generator import make_workload
    wl = make_workload(40, np.array([2, 3, 5, 4, 7] * 8), np.array([1, 1, 2, 2, 3] * 8), 5.5, seed=11)
    cols = np.array([0, 7, 13, 39])
    ix = dist_util.column_value_index(wl.n_blk, wl.row_ptr, wl.col_idx, wl.val_ptr, cols)
    mask = np.zeros(int(wl.val_ptr[-1]), bool)
    mask[ix] = True
    assert np.array_equal(mask, orc.column_mask(wl, cols)) and len(set(ix.tolist())) == ix.size
    allc = dist_util.column_value_index(wl.n_blk, wl.row_ptr, wl.col_idx, wl.val_ptr, np.arange(wl.n_blk))
    assert np.array_equal(np.sort(allc), np.arange(int(wl.val_ptr[-1])))


def test_single_process_aggregate_is_identity():
    assert dist_util.aggregate(3.5, 7.0, torch.device("cpu")) == (3.5, 7.0)
