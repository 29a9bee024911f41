"""N>1 host logic of bench.py on CPU (gloo, world size 2): the path does not shard
("replicas only"), so the only cross-rank step is the MAX of the timed region and
the sum of the replicas' work."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = 10.0 if rank == 0 else 25.0              # rank 1 is the slow replica
    value, ms_max = bench.aggregate_over_ranks(ms, cells_per_rank=1000, steps=4, world=world)
    dist.barrier()
    out[rank] = (value, ms_max)
    dist.destroy_process_group()


def test_replica_aggregation_takes_max_time_and_sums_work():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29531, out), nprocs=world, join=True)
    for rank in range(world):
        value, ms_max = out[rank]
        assert ms_max == 25.0
        assert value == pytest.approx(2 * 1000 * 4 / 25e-3)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    value, ms = bench.aggregate_over_ranks(8.0, 500, 2, 1)
    assert ms == 8.0 and value == pytest.approx(500 * 2 / 8e-3)
