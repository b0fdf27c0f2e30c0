"""bench.py's N > 1 accounting ("replicas only") on CPU: two gloo ranks, the slowest rank
sets the time, the value is the sum of the replicas' work.  (The GPU path itself never exchanges data.)"""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = 2.0 + rank            # rank 1 is slower: 3.0 ms
    ms = bench.max_over_ranks(mine, dist, torch.device("cpu"))
    dist.barrier()
    out[rank] = (ms, bench.job_value(10_000_000, world, ms))
    dist.destroy_process_group()


def test_replicas_take_the_slowest_rank_and_sum_the_work():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29541 + os.getpid() % 200, out), nprocs=world, join=True)
        assert dict(out) == {0: (3.0, 2 * 10_000_000 / 3.0e-3), 1: (3.0, 2 * 10_000_000 / 3.0e-3)}


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.5, None, None) == 1.5
    assert bench.job_value(100, 1, 2.0) == 100 / 2.0e-3
