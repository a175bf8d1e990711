"""N > 1 path of bench.py (weak scaling by independent replicas): the only cross-rank logic is the
max-over-ranks reduction of the timed region and the aggregation of the value.  Covered here with two
gloo processes on the CPU (the path has no data-path collective: DESIGN.md section 7)."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank                     # rank 1 is the slow one
    ms_max = bench.max_over_ranks(ms_local, dist, device="cpu")
    value = bench.aggregate_mlups(cells_per_rank=1000, steps=20, world=world, ms=ms_max)
    out[rank] = (ms_max, value)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_value():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29531, out), nprocs=world, join=True)
    for r in range(world):
        ms_max, value = out[r]
        assert ms_max == pytest.approx(15.0)
        assert value == pytest.approx(2 * 1000 * 20 / 15e-3 / 1e6)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, device="cpu") == 3.5
    assert bench.aggregate_mlups(64, 10, 1, 2.0) == pytest.approx(64 * 10 / 2e-3 / 1e6)
