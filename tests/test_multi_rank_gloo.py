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


def test_single_process_aggregate_is_identity():
    assert dist_util.aggregate(3.5, 7.0, torch.device("cpu")) == (3.5, 7.0)
