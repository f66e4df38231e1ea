"""Slab decomposition of a periodic box along z ("the domain is divided in equal sub-domains ... each
one assigned to a GPU ... exchange of the borders"; scaling Tables 4-5).

One rank = one GPU = one library context holding the planes [z0, z1) of the global box plus GHOST = 2 ghost planes on either side.
A step of the update needs, at a node, the populations and densities of its 18 neighbours, and a density needs the populations of
ITS 18 neighbours: information travels two planes per step.  So the unmodified kernels are run on the slab as if it were a periodic
box of nz_local + 4 planes: whatever the slab's own wrap feeds lands in the outermost ghost planes only, and every ghost plane is
overwritten before the next step by the owner's data: `ring_exchange` ships each slab's two lowest interior planes to its lower
neighbour's upper ghosts and its two highest to the upper neighbour's lower ghosts (periodic ring).

Nothing here computes: the planes move through `lb_export_planes` / `lb_import_planes` (device to device) and between ranks through
`torch.distributed` point-to-point calls (NCCL over NVLink on GPUs).  The transport and the ring logic are engine-agnostic (any
object with export_low / export_high / import_low / import_high), which is how the CPU tests drive them without a GPU.
"""
from __future__ import annotations

import numpy as np

GHOST = 2


def slab_range(nz: int, rank: int, world: int):
    """Planes [z0, z1) of rank `rank`: equal sub-domains; nz must divide evenly and leave >= GHOST planes per rank."""
    if nz % world != 0 or nz // world < GHOST:
        raise ValueError(f"nz = {nz} does not split into {world} equal slabs of >= {GHOST} planes")
    nzl = nz // world
    return rank * nzl, (rank + 1) * nzl


def cut_with_ghosts(a, nx, ny, nz, z0, z1):
    """Planes z0 - GHOST .. z1 + GHOST - 1 (periodic) of a dense [z][y][x] field, flat."""
    if a is None:
        return None
    zz = np.arange(z0 - GHOST, z1 + GHOST) % nz
    return np.ascontiguousarray(np.asarray(a).reshape(nz, ny, nx)[zz]).reshape(-1)


class SlabBox:
    """One rank's slab on the CUDA library: the default kernel of the box shape (the one-pass TMA kernel where the tile fits; the
    planes then travel with their carried density), or `kernel`."""

    def __init__(self, nx, ny, nz, rank, world, tau_r=1.0, tau_b=1.0, G=1.2, dtype=None, cuda_stream=None, device=None, kernel=None):
        import torch
        from . import binding as B
        self.B, self.torch = B, torch
        self.nx, self.ny, self.nz, self.rank, self.world = nx, ny, nz, rank, world
        self.z0, self.z1 = slab_range(nz, rank, world)
        self.nzl = self.z1 - self.z0
        dtype = B.LB_F64 if dtype is None else dtype
        self.box = B.Box(nx, ny, self.nzl + 2 * GHOST, tau_r, tau_b, G, dtype=dtype, cuda_stream=cuda_stream)
        if kernel is not None:
            self.box.set_kernel(kernel)
        self.buffer_bytes = None
        self._tdt = torch.float64 if dtype == B.LB_F64 else torch.float32
        self._dev = device if device is not None else torch.device("cuda", torch.cuda.current_device())

    def _buffers(self):
        nbytes = self.box.plane_buffer_bytes(GHOST)                 # depends on the kernel in effect (with / without the carried density)
        if nbytes != self.buffer_bytes:
            n = nbytes // (8 if self._tdt == self.torch.float64 else 4)
            self.send_lo, self.send_hi, self.recv_lo, self.recv_hi = (self.torch.empty(n, dtype=self._tdt, device=self._dev) for _ in range(4))
            self.buffer_bytes = nbytes

    def set_fields(self, rho_r, rho_b, ux=None, uy=None, uz=None):
        """Global fields in; this rank keeps its planes and the ghosts."""
        a = [cut_with_ghosts(v, self.nx, self.ny, self.nz, self.z0, self.z1) for v in (rho_r, rho_b, ux, uy, uz)]
        self.box.set_fields(*a)

    def export_low(self):
        self._buffers()
        self.box.export_planes(GHOST, GHOST, self.send_lo.data_ptr())
        self.box.sync()
        return self.send_lo

    def export_high(self):
        self._buffers()
        self.box.export_planes(self.nzl, GHOST, self.send_hi.data_ptr())
        self.box.sync()
        return self.send_hi

    def import_low(self, t):
        self.box.import_planes(0, GHOST, t.data_ptr())

    def import_high(self, t):
        self.box.import_planes(self.nzl + GHOST, GHOST, t.data_ptr())

    def step(self, n=1):
        self.box.step(n)

    def get_populations(self):
        """The rank's own planes [z0, z1): [2][19][nzl][ny][nx].  The library keeps the post-collision state and streams when it is
        read (pull), so the populations of the outermost own planes come out of the ghost planes: exchange once more after the last
        step before calling this."""
        return self.box.get_populations()[:, :, GHOST:GHOST + self.nzl]

    def close(self):
        self.box.close()


def ring_exchange_local(slabs):
    """All ranks in one process (virtual ranks, e.g. several slabs on one GPU): ghost planes straight from the neighbours' exports."""
    R = len(slabs)
    lows = [s.export_low() for s in slabs]
    highs = [s.export_high() for s in slabs]
    for r, s in enumerate(slabs):
        s.import_low(highs[(r - 1) % R])            # my lower ghosts = the highest interior planes of the rank below
        s.import_high(lows[(r + 1) % R])            # my upper ghosts = the lowest interior planes of the rank above


def ring_exchange_dist(slab, dist, recv_lo=None, recv_hi=None):
    """One rank per process: the same exchange through torch.distributed point-to-point calls (NCCL on GPUs, gloo in the CPU tests).
    `recv_lo` / `recv_hi` default to the slab's own receive buffers."""
    rank, world = dist.get_rank(), dist.get_world_size()
    lo, hi = slab.export_low(), slab.export_high()          # (the slab's receive buffers exist from here on)
    recv_lo = slab.recv_lo if recv_lo is None else recv_lo
    recv_hi = slab.recv_hi if recv_hi is None else recv_hi
    if world == 1:
        recv_lo.copy_(hi), recv_hi.copy_(lo)
    else:
        below, above = (rank - 1) % world, (rank + 1) % world
        # order matters where the transport matches messages by order, not by tag (NCCL), and both neighbours are the same
        # rank (world = 2): my first send (high planes) is the peer's first receive (its lower ghosts)
        ops = [dist.P2POp(dist.isend, hi, above, tag=1), dist.P2POp(dist.isend, lo, below, tag=0),
               dist.P2POp(dist.irecv, recv_lo, below, tag=1), dist.P2POp(dist.irecv, recv_hi, above, tag=0)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    slab.import_low(recv_lo)
    slab.import_high(recv_hi)
