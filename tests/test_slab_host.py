"""Host side of the z-slab decomposition (paper_2401_03041_b200/slab.py): who owns which planes, how arrays are cut,
and that the point-to-point exchange delivers each face message to the right buffer of the right rank -- with gloo
processes on the CPU (world 2, where both neighbours are the same rank, and world 3)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2401_03041_b200.slab import SlabLayout, exchange_faces, fill_ghost_planes, slab_range

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_ranges_partition_the_box():
    for nz, world in ((22, 5), (400, 8), (7, 7), (128, 3), (5, 1)):
        r = [slab_range(nz, k, world) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == nz
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        sizes = [b - a for a, b in r]
        assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1
    with pytest.raises(ValueError):
        slab_range(3, 0, 4)
    with pytest.raises(ValueError):
        slab_range(8, 2, 2)


def test_layout_neighbours_and_ghosts():
    per = SlabLayout(12, 3, periodic_z=True)
    assert [per.neighbours(r) for r in range(3)] == [(2, 1), (0, 2), (1, 0)]
    assert [per.ghosts(r) for r in range(3)] == [(1, 1)] * 3
    wal = SlabLayout(12, 3, periodic_z=False)
    assert [wal.neighbours(r) for r in range(3)] == [(None, 1), (0, 2), (1, None)]
    assert [wal.ghosts(r) for r in range(3)] == [(0, 1), (1, 1), (1, 0)]
    assert SlabLayout(12, 1, True).ghosts(0) == (0, 0)       # one slab: the plain periodic wrap
    two = SlabLayout(8, 2, True)
    assert two.neighbours(0) == (1, 1) and two.neighbours(1) == (0, 0)


def test_extend_cuts_slabs_with_their_ghost_planes():
    rng = np.random.default_rng(0)
    a = rng.standard_normal((3, 10, 4, 5))
    per = SlabLayout(10, 3, True)            # planes 0-3, 4-6, 7-9
    assert np.array_equal(per.extend(a, 0), a[:, [9, 0, 1, 2, 3, 4]])
    assert np.array_equal(per.extend(a, 2), a[:, [6, 7, 8, 9, 0]])
    wal = SlabLayout(10, 3, False)
    assert np.array_equal(wal.extend(a, 0), a[:, 0:5])
    assert np.array_equal(wal.extend(a, 1), a[:, 3:8])
    assert np.array_equal(wal.extend(a, 2), a[:, 6:10])
    t = torch.from_numpy(a)
    assert torch.equal(per.extend(t, 1), t[:, 3:8])
    w = rng.standard_normal((10, 5))         # a y-wall temperature plane [nz][nx]
    assert np.array_equal(per.extend(w, 2, z_axis=-2), w[[6, 7, 8, 9, 0]])


def _worker(rank, world, port, periodic, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nz, ny, nx = 11, 3, 4
    lay = SlabLayout(nz, world, periodic)
    lower, upper = lay.neighbours(rank)
    lo, hi = lay.ghosts(rank)
    # (1) every message lands in the right buffer: message = (sender, face) tag
    tag = lambda r, face: torch.full((6,), 10.0 * r + face, dtype=torch.float64)
    recv_lo, recv_hi = torch.full((6,), -1.0, dtype=torch.float64), torch.full((6,), -1.0, dtype=torch.float64)
    exchange_faces(tag(rank, 0), tag(rank, 1), recv_lo, recv_hi, lower, upper)
    got = (recv_lo[0].item(), recv_hi[0].item())
    # (2) ghost planes of a slab cut without them are filled from the neighbours
    g = torch.from_numpy(np.random.default_rng(1).standard_normal((2, nz, ny, nx)))
    mine = lay.extend(g, rank).clone()
    if lo:
        mine[:, 0] = 0.0
    if hi:
        mine[:, -1] = 0.0
    fill_ghost_planes(mine, lo, hi, lower, upper)
    ghosts_ok = bool(torch.equal(mine, lay.extend(g, rank)))
    # (3) the step protocol on a toy transport: `up` moves one plane up per step, `down` one plane down
    #     (begin: update own planes from old ones incl. ghosts; send new boundary planes; end: ghosts <- received)
    up, down = lay.extend(g[0], rank).clone(), lay.extend(g[1], rank).clone()
    n = up.shape[0]
    for _ in range(5):
        new_up, new_down = up.clone(), down.clone()
        zs = range(lo, n - hi)
        for z in zs:                          # walls (no ghost): the toy reflects nothing, planes just stay
            new_up[z] = up[z - 1] if z - 1 >= 0 else up[z]
            new_down[z] = down[z + 1] if z + 1 < n else down[z]
        send_hi, send_lo = new_up[n - 1 - hi].contiguous(), new_down[lo].contiguous()
        r_lo, r_hi = torch.empty_like(send_hi), torch.empty_like(send_lo)
        exchange_faces(send_lo, send_hi, r_lo, r_hi, lower, upper)
        if lo:
            new_up[0] = r_lo
        if hi:
            new_down[-1] = r_hi
        up, down = new_up, new_down
    out[rank] = (got, ghosts_ok, up[lo:n - hi].numpy().copy(), down[lo:n - hi].numpy().copy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic,port", [(2, True, 29541), (3, True, 29542), (3, False, 29543)])
def test_exchange_between_ranks(world, periodic, port):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, periodic, out), nprocs=world, join=True)
    lay = SlabLayout(11, world, periodic)
    g = np.random.default_rng(1).standard_normal((2, 11, 3, 4))
    ups, downs = [], []
    for r in range(world):
        (lo_tag, hi_tag), ghosts_ok, up, down = out[r]
        lower, upper = lay.neighbours(r)
        # recv_lo holds the LOWER neighbour's send_hi (face 1), recv_hi the UPPER neighbour's send_lo (face 0)
        assert lo_tag == (10.0 * lower + 1 if lower is not None else -1.0)
        assert hi_tag == (10.0 * upper + 0 if upper is not None else -1.0)
        assert ghosts_ok
        ups.append(up); downs.append(down)
    if periodic:
        assert np.array_equal(np.concatenate(ups), np.roll(g[0], 5, axis=0))
        assert np.array_equal(np.concatenate(downs), np.roll(g[1], -5, axis=0))
