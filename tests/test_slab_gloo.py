"""Slab decomposition on CPU: the ring exchange of paper_2112_08264_b200/slab.py between two processes over gloo,
with the ORACLE as the per-rank engine (the library has no CPU path): every rank steps its slab + ghost planes, ships its outermost
interior planes to its neighbours, and the assembled result must be the oracle's on the undivided box.  Also the virtual-rank
(one process) form of the same exchange for 1, 2, 3 and 4 slabs."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

NX, NY, NZ, STEPS = 8, 6, 16, 5
TAU, G = (0.8, 1.3), 0.9


class OracleSlab:
    """The oracle on planes [z0 - 2, z1 + 2) of the global box, with the engine interface ring_exchange_* expects."""

    def __init__(self, ora, rank, world, fields):
        from paper_2112_08264_b200 import slab as S
        self.S = S
        self.z0, self.z1 = S.slab_range(NZ, rank, world)
        self.nzl = self.z1 - self.z0
        self.o = ora.Oracle(NX, NY, self.nzl + 2 * S.GHOST, TAU[0], TAU[1], G)
        self.o.set_fields(*[S.cut_with_ghosts(v, NX, NY, NZ, self.z0, self.z1) for v in fields])

    def _planes(self, a, b):
        return torch.from_numpy(np.ascontiguousarray(self.o.get_populations()[:, :, a:b]).reshape(-1).copy())

    def _put(self, a, b, t):
        f = self.o.get_populations().copy()
        f[:, :, a:b] = t.numpy().reshape(2, 19, b - a, NY, NX)
        self.o.set_populations(f.reshape(-1))

    def export_low(self):
        return self._planes(self.S.GHOST, 2 * self.S.GHOST)

    def export_high(self):
        return self._planes(self.nzl, self.nzl + self.S.GHOST)

    def import_low(self, t):
        self._put(0, self.S.GHOST, t)

    def import_high(self, t):
        self._put(self.nzl + self.S.GHOST, self.nzl + 2 * self.S.GHOST, t)

    def interior(self):
        return self.o.get_populations()[:, :, self.S.GHOST:self.S.GHOST + self.nzl]


def _fields():
    from paper_2112_08264_b200 import workloads as w
    rr, rb = w.mixture_fields(NX, NY, NZ, 77, amp=0.05)
    u = np.random.default_rng(8).uniform(-0.02, 0.02, (3, NX * NY * NZ))
    return rr, rb, u[0], u[1], u[2]


def _reference():
    from oracle import ora
    ora.build("ref")
    o = ora.Oracle(NX, NY, NZ, TAU[0], TAU[1], G)
    o.set_fields(*_fields())
    o.step(STEPS)
    return o.get_populations()


@pytest.mark.parametrize("world", [1, 2, 4, 8])
def test_virtual_ranks_reproduce_the_undivided_box(world):
    from oracle import ora
    from paper_2112_08264_b200 import slab as S
    ora.build("ref")
    slabs = [OracleSlab(ora, r, world, _fields()) for r in range(world)]
    for _ in range(STEPS):
        S.ring_exchange_local(slabs)
        for s in slabs:
            s.o.step(1)
    got = np.concatenate([s.interior() for s in slabs], axis=2)
    assert np.array_equal(got, _reference())                    # same arithmetic on the same values: bit-identical


def test_slab_ranges():
    from paper_2112_08264_b200 import slab as S
    assert [S.slab_range(16, r, 4) for r in range(4)] == [(0, 4), (4, 8), (8, 12), (12, 16)]
    with pytest.raises(ValueError):
        S.slab_range(10, 0, 4)
    with pytest.raises(ValueError):
        S.slab_range(4, 0, 4)                                    # one plane per rank: fewer than the two ghost planes a neighbour needs
    a = np.arange(16 * 2 * 3, dtype=float)
    c = S.cut_with_ghosts(a, 3, 2, 16, 0, 4).reshape(8, 2, 3)
    assert np.array_equal(c[0], a.reshape(16, 2, 3)[14]) and np.array_equal(c[7], a.reshape(16, 2, 3)[5])


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from oracle import ora
    from paper_2112_08264_b200 import slab as S
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s = OracleSlab(ora, rank, world, _fields())
    n = 38 * S.GHOST * NX * NY
    recv_lo, recv_hi = torch.empty(n, dtype=torch.float64), torch.empty(n, dtype=torch.float64)
    for _ in range(STEPS):
        S.ring_exchange_dist(s, dist, recv_lo, recv_hi)
        s.o.step(1)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, s.interior().copy()))


@pytest.mark.parametrize("world", [2, 4])
def test_ring_exchange_over_gloo(world):
    from oracle import ora
    ora.build("ref")                                             # once, before the ranks race for it
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    [p.start() for p in procs]
    got = dict(out.get(timeout=300) for _ in procs)
    [p.join(60) for p in procs]
    assert all(p.exitcode == 0 for p in procs)
    assert np.array_equal(np.concatenate([got[r] for r in range(world)], axis=2), _reference())
