"""The N > 1 path of bench.py (replicas only) on CPU: two gloo ranks run the aggregation that
turns per-rank times and unit counts into the whole-job numbers (time = max over ranks, units = sum over ranks)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times = [10.0 + rank, 20.0 - rank, 5.0 * (rank + 1)]            # each rank is the slowest in a different entry
    t, u = bench.aggregate_over_ranks(times, 1000.0 * (rank + 1), world, torch.device("cpu"))
    dist.barrier()
    dist.destroy_process_group()
    out[rank] = (t, u)


def test_two_ranks_max_time_sum_units():
    world = 2
    port = 29500 + os.getpid() % 500
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]                                          # every rank sees the same whole-job numbers
    t, u = res[0]
    assert t == [11.0, 20.0, 10.0] and u == 3000.0


def test_single_rank_is_the_identity():
    sys.path.insert(0, ROOT)
    import bench
    t, u = bench.aggregate_over_ranks([1.5, 2.5, 3.5], 7.0, 1, torch.device("cpu"))
    assert t == [1.5, 2.5, 3.5] and u == 7.0
