"""`RankSlab` (one z-slab per rank of a torch.distributed group) end to end on the one GPU of the test box: two / three
processes share cuda:0 and exchange their face messages through `gloo` (host-staged, so no kernel of one process ever
waits for a kernel of another); gathered, their planes must carry the BITS of the undivided box.  What this adds to
tests/test_gpu_slabs.py (all slabs in one process) is the per-rank driver: ghost filling before init, the transfer on
the comm stream after every phase, and the matching of messages when both neighbours are the same rank."""
import os
import sys
import tempfile

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from parity_util import _np, run_gpu
from workloads import configs

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _workload(case):
    if case == "rk2_walls":
        return configs.droplet_in_gradient(nx=20, ny=18, nz=26, thermal="rk2", R=5.0, zc=10.0), 12
    return configs.perf_box(24, thermal=case, ny=20, nz=22, seed=11, r_min=4.0, r_max=6.0), 12


def _worker(rank, world, port, case, out_dir):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch.distributed as dist
    from paper_2401_03041_b200.slab import RankSlab
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    wl, steps = _workload(case)
    box = RankSlab(wl.nx, wl.ny, wl.nz, dict(wl.params))
    s, lay = box.slab, box.layout
    for (ax, fc), plane in wl.wall_T.items():
        s.set_wall_temperature_from_global(ax, fc, _np(plane))
    # every rank cuts its slab WITHOUT knowing its neighbours' planes: ghost planes start as NaN and are filled
    # by the exchange (what a rank that generated only its own part of the box does)
    def mine(a):
        if a is None:
            return None
        t = lay.extend(torch.as_tensor(_np(a)), rank).cuda()
        if s.lo:
            t.select(-3, 0).fill_(float("nan"))
        if s.hi:
            t.select(-3, t.shape[-3] - 1).fill_(float("nan"))
        return box.fill_ghosts(t)
    s.init_fields(mine(wl.phi), mine(wl.u), mine(wl.T))
    box.step(steps)
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), *s.read_fields())
    box.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(600)
@pytest.mark.parametrize("case,world,port", [("lb_d3q7", 2, 29551), ("lb_d3q19", 3, 29552), ("rk2_walls", 3, 29553)])
def test_rank_slabs_reproduce_the_undivided_box(case, world, port):
    wl, steps = _workload(case)
    want, _ = run_gpu(wl, steps)
    with tempfile.TemporaryDirectory() as d:
        mp.spawn(_worker, args=(world, port, case, d), nprocs=world, join=True)
        parts = [np.load(os.path.join(d, f"rank{r}.npz")) for r in range(world)]
        got = [np.concatenate([p[f"arr_{k}"] for p in parts], axis=-3) for k in range(4)]
    for name, g, w in zip(("phi", "u", "p", "T"), got, want):
        assert g.shape == w.shape
        assert np.array_equal(g, w), f"{name}: {np.count_nonzero(g != w)} cells differ"
