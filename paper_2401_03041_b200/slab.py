"""Block decomposition along z: the host side.

A box of nz planes is cut into `world` z-slabs.  Every slab is an ordinary `tcp_sim` with one ghost plane on
each face that has a neighbour (`tcp_set_halo`); one step is `tcp_step_begin` (boundary planes, gather, interior)
-> the transfer of one message per face -> `tcp_step_advance` (scatter; on the Runge-Kutta paths then the next
stage the same way, until no transfer is left).  This module only slices arrays, owns the
message buffers and moves the messages: between slabs of ONE process (`LocalSlabs`, a device copy; what the
single-GPU tests and `bench.py --slabs` run) or between ranks (`RankSlab`, `torch.distributed` point-to-point,
NCCL over NVLink on GPUs).  No arithmetic of the method lives here.
"""
import numpy as np
import torch

from . import binding as B


def slab_range(nz: int, rank: int, world: int):
    """Planes [z0, z1) of slab `rank`: as equal as possible, the first nz % world slabs one plane thicker."""
    if not 0 <= rank < world or world > nz:
        raise ValueError(f"cannot cut {nz} planes into {world} slabs (rank {rank})")
    q, r = divmod(nz, world)
    z0 = rank * q + min(rank, r)
    return z0, z0 + q + (1 if rank < r else 0)


class SlabLayout:
    """Who owns which planes, which faces carry a ghost plane, and who the neighbours are."""

    def __init__(self, nz: int, world: int, periodic_z: bool):
        self.nz, self.world, self.periodic_z = nz, world, bool(periodic_z)
        self.ranges = [slab_range(nz, r, world) for r in range(world)]

    def neighbours(self, rank):
        """(lower, upper) rank or None where the box ends in a wall."""
        lo = rank - 1 if rank > 0 else (self.world - 1 if self.periodic_z else None)
        hi = rank + 1 if rank < self.world - 1 else (0 if self.periodic_z else None)
        return lo, hi

    def ghosts(self, rank):
        """(lo, hi): 1 where the slab has a ghost plane.  A periodic box in one slab needs none (plain wrap)."""
        if self.world == 1:
            return 0, 0
        lo, hi = self.neighbours(rank)
        return int(lo is not None), int(hi is not None)

    def extended_planes(self, rank):
        """Global z indices of the slab's planes including its ghost planes."""
        z0, z1 = self.ranges[rank]
        lo, hi = self.ghosts(rank)
        return np.arange(z0 - lo, z1 + hi) % self.nz

    def extend(self, a, rank, z_axis=-3):
        """Slab `rank` of the global array `a` (numpy or torch) with its ghost planes."""
        idx = self.extended_planes(rank)
        if isinstance(a, torch.Tensor):
            return a.index_select(z_axis % a.dim(), torch.as_tensor(idx, device=a.device)).contiguous()
        return np.ascontiguousarray(np.take(a, idx, axis=z_axis))


def exchange_faces(send_lo, send_hi, recv_lo, recv_hi, lower, upper, group=None):
    """Point-to-point exchange of the two face messages of this rank (any backend, CPU or CUDA tensors):
    send_hi -> `upper`'s recv_lo, send_lo -> `lower`'s recv_hi.  Receives are posted in the mirrored order of the
    sends, so that with two ranks in a periodic box (lower == upper) the pairs still match up."""
    import torch.distributed as dist
    # a backend without device-to-device transport (gloo) gets the messages through host memory
    via_host = dist.get_backend(group) == "gloo" and any(t is not None and t.is_cuda for t in (send_lo, send_hi))
    dev = (recv_lo, recv_hi)
    if via_host:
        host = lambda t: None if t is None else t.cpu()        # synchronises the current stream
        send_lo, send_hi, recv_lo, recv_hi = host(send_lo), host(send_hi), host(recv_lo), host(recv_hi)
    ops = []
    if upper is not None:
        ops.append(dist.P2POp(dist.isend, send_hi, upper, group))
    if lower is not None:
        ops.append(dist.P2POp(dist.isend, send_lo, lower, group))
    if lower is not None:
        ops.append(dist.P2POp(dist.irecv, recv_lo, lower, group))
    if upper is not None:
        ops.append(dist.P2POp(dist.irecv, recv_hi, upper, group))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    if via_host:
        if lower is not None:
            dev[0].copy_(recv_lo)
        if upper is not None:
            dev[1].copy_(recv_hi)


def fill_ghost_planes(a_ext, lo, hi, lower, upper, group=None, z_axis=-3):
    """Ghost planes (first plane if `lo`, last if `hi`) of this rank's extended-box tensor <- the neighbours'
    boundary planes.  What a rank that generated only its own slab calls on phi, u, T before tcp_init_fields."""
    if not (lo or hi):
        return a_ext
    n = a_ext.shape[z_axis]
    plane = lambda k: a_ext.select(z_axis, k)
    send_lo, send_hi = plane(lo).contiguous(), plane(n - 1 - hi).contiguous()
    recv_lo, recv_hi = torch.empty_like(send_lo), torch.empty_like(send_hi)
    exchange_faces(send_lo, send_hi, recv_lo, recv_hi, lower, upper, group)
    if lo:
        plane(0).copy_(recv_lo)
    if hi:
        plane(n - 1).copy_(recv_hi)
    return a_ext


class Slab:
    """One slab on the current CUDA device: the simulation on its extended box, message buffers, comm stream."""

    def __init__(self, nx, ny, layout: SlabLayout, rank: int, params: dict, comm_stream=None, device="cuda"):
        self.layout, self.rank = layout, rank
        self.z0, self.z1 = layout.ranges[rank]
        self.lo, self.hi = layout.ghosts(rank)
        nz_ext = self.z1 - self.z0 + self.lo + self.hi
        self.sim = B.Simulation(nx, ny, nz_ext, params, device=device)
        self.comm = comm_stream if comm_stream is not None else torch.cuda.Stream(device=self.sim.device)
        n = B.tcp_halo_bytes(self.sim._h) // np.dtype(self.sim.np_dtype).itemsize
        mk = lambda on: torch.zeros(n, dtype=self.sim.torch_dtype, device=self.sim.device) if on else None
        self.send_lo, self.recv_lo, self.send_hi, self.recv_hi = mk(self.lo), mk(self.lo), mk(self.hi), mk(self.hi)
        if self.lo or self.hi:
            B.tcp_set_halo(self.sim._h, self.lo, self.hi, self.comm, self.send_lo, self.send_hi, self.recv_lo, self.recv_hi)
        # values of the message that follows each phase of a step (tcp_halo_message_bytes)
        item = np.dtype(self.sim.np_dtype).itemsize
        self.message_values = [B.tcp_halo_message_bytes(self.sim._h, p) // item for p in range(B.tcp_halo_phases(self.sim._h))]

    @property
    def halo(self):
        return bool(self.lo or self.hi)

    def interior(self, a, z_axis=-3):
        """Strip the ghost planes of an array of the extended box."""
        n = a.shape[z_axis]
        sl = [slice(None)] * a.ndim
        sl[z_axis] = slice(self.lo, n - self.hi)
        return a[tuple(sl)]

    def init_fields(self, phi, u=None, T=None):
        """Arrays of the extended box (ghost planes filled with the neighbours' values)."""
        self.sim.init_fields(phi, u, T)

    def init_from_global(self, phi, u=None, T=None):
        ext = lambda a: None if a is None else self.layout.extend(a, self.rank)
        self.sim.init_fields(ext(phi), ext(u), ext(T))

    def set_wall_temperature_from_global(self, axis, face, Tw):
        """Tw of the global box; x / y wall planes are [nz][ny] / [nz][nx] and are cut with their ghost rows."""
        if Tw is not None and axis in (0, 1):
            Tw = self.layout.extend(Tw, self.rank, z_axis=-2)
        self.sim.set_wall_temperature(axis, face, Tw)

    def set_heat_source_from_global(self, q):
        self.sim.set_heat_source(None if q is None else self.layout.extend(q, self.rank))

    def step_begin(self):
        if self.halo:
            B.tcp_step_begin(self.sim._h)
        else:
            self.sim.step(1)

    def step_advance(self) -> int:
        """After a transfer: scatter, then the next phase or the end of the step.  -> transfers left"""
        return B.tcp_step_advance(self.sim._h) if self.halo else 0

    def read_fields(self):
        """phi, u, p, T of the planes this slab owns (host arrays)."""
        return tuple(np.ascontiguousarray(self.interior(a)) for a in self.sim.read_fields())

    def close(self):
        self.sim.close()


class LocalSlabs:
    """All slabs of a box in one process on one GPU; the 'transfer' is a device copy on the shared comm stream.
    Used to check the decomposition against the undivided box and to measure what it costs on one GPU."""

    def __init__(self, nx, ny, nz, nslabs, params: dict, device="cuda"):
        periodic_z = B.make_params(params).bc[2] == B.BC["periodic"]
        self.layout = SlabLayout(nz, nslabs, periodic_z)
        self.comm = torch.cuda.Stream(device=torch.device(device))
        self.slabs = [Slab(nx, ny, self.layout, r, params, comm_stream=self.comm, device=device) for r in range(nslabs)]

    def init_fields(self, phi, u=None, T=None):
        for s in self.slabs:
            s.init_from_global(phi, u, T)

    def set_wall_temperature(self, axis, face, Tw):
        for s in self.slabs:
            s.set_wall_temperature_from_global(axis, face, Tw)

    def set_heat_source(self, q):
        for s in self.slabs:
            s.set_heat_source_from_global(q)

    def step(self, n=1):
        for _ in range(n):
            for s in self.slabs:
                s.step_begin()
            for nv in self.slabs[0].message_values:     # one transfer after every phase
                with torch.cuda.stream(self.comm):      # after every gather, before every scatter (same stream)
                    for s in self.slabs:
                        lower, upper = self.layout.neighbours(s.rank)
                        if s.hi:
                            self.slabs[upper].recv_lo[:nv].copy_(s.send_hi[:nv], non_blocking=True)
                        if s.lo:
                            self.slabs[lower].recv_hi[:nv].copy_(s.send_lo[:nv], non_blocking=True)
                for s in self.slabs:
                    s.step_advance()

    def read_fields(self):
        parts = [s.read_fields() for s in self.slabs]
        return tuple(np.concatenate([p[k] for p in parts], axis=-3) for k in range(4))

    def synchronize(self):
        for s in self.slabs:
            s.sim.synchronize()
        self.comm.synchronize()

    @property
    def launches(self):
        return sum(s.sim.launches for s in self.slabs)

    def close(self):
        for s in self.slabs:
            s.close()


class RankSlab:
    """The slab of this rank of an initialised `torch.distributed` process group (one process per GPU).
    Messages travel point-to-point on the slab's comm stream while the interior is being updated."""

    def __init__(self, nx, ny, nz_global, params: dict, group=None, device="cuda"):
        import torch.distributed as dist
        self.group = group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        periodic_z = B.make_params(params).bc[2] == B.BC["periodic"]
        self.layout = SlabLayout(nz_global, self.world, periodic_z)
        self.slab = Slab(nx, ny, self.layout, self.rank, params, device=device)
        self.lower, self.upper = self.layout.neighbours(self.rank)

    def fill_ghosts(self, a_ext, z_axis=-3):
        """Fill the ghost planes of an extended-box tensor with the neighbours' boundary planes (before init)."""
        return fill_ghost_planes(a_ext, self.slab.lo, self.slab.hi, self.lower, self.upper, self.group, z_axis)

    def step(self, n=1):
        s = self.slab
        for _ in range(n):
            s.step_begin()
            if not s.halo:
                continue
            cut = lambda t, nv: None if t is None else t[:nv]
            for nv in s.message_values:
                with torch.cuda.stream(s.comm):
                    exchange_faces(cut(s.send_lo, nv), cut(s.send_hi, nv), cut(s.recv_lo, nv), cut(s.recv_hi, nv),
                                   self.lower, self.upper, self.group)
                s.step_advance()

    def close(self):
        self.slab.close()
