"""Host-side logic of the slab decomposition on CPU: ranges, neighbours, local geometry, diagnostics
folding, and the exchange schedule over two and three gloo ranks with a stand-in slab (no CUDA involved)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2606_00641_b200 import slab  # noqa: E402


def test_ranges_and_neighbours():
    assert slab.slab_ranges(256, 8) == [(32 * r, 32 * r + 32) for r in range(8)]
    assert slab.slab_ranges(10, 3) == [(0, 4), (4, 7), (7, 10)]
    with pytest.raises(ValueError):
        slab.slab_ranges(2, 3)
    assert slab.neighbours(0, 4, True) == (3, 1) and slab.neighbours(3, 4, True) == (2, 0)
    assert slab.neighbours(0, 4, False) == (None, 1) and slab.neighbours(3, 4, False) == (2, None)
    assert slab.neighbours(0, 1, True) == (None, None)
    assert slab.neighbours(0, 2, True) == (1, 1)


def test_local_geometry():
    # config 5: periodic z, cut in 4
    g = slab.local_geometry((384, 256, 256), (2, 1, 0, 0, 0, 0), 0, 4)
    assert g["shape"] == (384, 256, 66) and g["bc"] == (2, 1, 0, 0, 3, 3)
    assert list(g["take"][[0, 1, -2, -1]]) == [255, 0, 63, 64] and g["owned"] == (1, 65) and g["halo_offset"] == -1
    g = slab.local_geometry((384, 256, 256), (2, 1, 0, 0, 0, 0), 3, 4)
    assert list(g["take"][[0, -1]]) == [191, 0] and g["halo_offset"] == 191
    # non-periodic cut axis: true faces keep their kind, no ghost there
    g = slab.local_geometry((64, 30), (1, 1, 1, 2, 0, 0), 0, 3)
    assert g["shape"] == (64, 11) and g["bc"] == (1, 1, 1, 3, 0, 0) and g["owned"] == (0, 10) and g["halo_offset"] == 0
    g = slab.local_geometry((64, 30), (1, 1, 1, 2, 0, 0), 2, 3)
    assert g["shape"] == (64, 11) and g["bc"] == (1, 1, 3, 2, 0, 0) and g["owned"] == (1, 11) and g["halo_offset"] == 19
    # every global plane is owned exactly once
    owned = []
    for r in range(3):
        g = slab.local_geometry((64, 30), (1, 1, 1, 2, 0, 0), r, 3)
        owned += list(g["take"][g["owned"][0]:g["owned"][1]])
    assert owned == list(range(30))


def test_step_pieces_and_exchange_kinds():
    # boundary planes first (those next to a ghost), the rest completes the step; every owned plane exactly once
    assert slab.step_pieces((1, 65), True, True) == ([(1, 2), (64, 65)], (2, 64))
    assert slab.step_pieces((0, 10), False, True) == ([(9, 10)], (0, 9))
    assert slab.step_pieces((1, 11), True, False) == ([(1, 2)], (2, 11))
    assert slab.step_pieces((1, 2), True, True) == ([(1, 2)], (2, 2))          # one owned plane: no interior
    assert slab.step_pieces((1, 3), True, True) == ([(1, 2), (2, 3)], (2, 2))
    assert slab.step_pieces((0, 8), False, False) == ([], (0, 8))
    for owned, lo, hi in (((1, 65), True, True), ((0, 10), False, True), ((1, 2), True, True), ((1, 3), True, True)):
        b, (i0, i1) = slab.step_pieces(owned, lo, hi)
        planes = [p for r in b for p in range(*r)] + list(range(i0, i1))
        assert sorted(planes) == list(range(*owned))
    # A/B: always the crossing populations; in place: what a pull-push step pushed goes back, a local step is followed by a refresh
    assert slab.exchange_kind(0, 0) == slab.CROSSING and slab.exchange_kind(0, 1) == slab.CROSSING
    assert slab.exchange_kind(1, 0) == slab.RETURN and slab.exchange_kind(1, 1) == slab.CROSSING


def test_combine_diag():
    K = 2
    a = np.array([1, 2, 3, 4, 5, 6, 0.1, 1.0, 0.5, 1], dtype=float)
    b = np.array([10, 20, 30, 40, 2, 9, 0.3, 0.9, 0.7, 2], dtype=float)
    out = slab.combine_diag([a, b], K)
    assert list(out) == [11, 22, 33, 44, 5, 9, 0.3, 0.9, 0.5, 3]


class FakeSlab:
    """stands in for slab.Slab: a 'plane' is just a tagged CPU tensor"""

    def __init__(self, rank, lo, hi):
        self.rank, self.lo, self.hi, self.got = rank, lo, hi, {}
        sides = [side for side, nb in ((0, lo), (1, hi)) if nb is not None]
        self.send = {s: torch.zeros(4, dtype=torch.float64) for s in sides}
        self.recv = {s: torch.zeros(4, dtype=torch.float64) for s in sides}
        self.allocations = 2 * len(sides)

    def full_buffers(self):
        self.allocations += 2 * len(self.send)
        return ({s: torch.zeros(8, dtype=torch.float64) for s in self.send}, {s: torch.zeros(8, dtype=torch.float64) for s in self.recv})

    def halo_pack(self, side, buf, what=0, next_copy=False, stream=None):
        buf.fill_(100.0 * self.rank + 10.0 * side + int(what))

    def halo_unpack(self, side, buf, what=0, next_copy=False, stream=None):
        self.got[(side, what)] = float(buf[0])


def _worker(rank, world, port, periodic, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = slab.neighbours(rank, world, periodic)
    s = FakeSlab(rank, lo, hi)
    n0 = s.allocations
    for _ in range(3):                               # crossing / return exchanges reuse the slab's buffers: nothing is allocated per step
        slab.exchange_distributed(s, dist, slab.CROSSING)
        slab.exchange_distributed(s, dist, slab.RETURN)
    assert s.allocations == n0
    slab.exchange_distributed(s, dist, slab.FULL)
    dist.barrier()
    q.put((rank, s.got))
    dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True)])
def test_exchange_schedule_over_gloo(world, periodic):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + (os.getpid() + 7 * world + int(periodic)) % 300
    procs = [ctx.Process(target=_worker, args=(r, world, port, periodic, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for r in range(world):
        lo, hi = slab.neighbours(r, world, periodic)
        for full in (slab.CROSSING, slab.FULL, slab.RETURN):
            # our low ghost holds what the low neighbour packed on ITS high side, and vice versa
            if lo is not None:
                assert res[r][(0, full)] == 100.0 * lo + 10.0 * 1 + int(full)
            else:
                assert (0, full) not in res[r]
            if hi is not None:
                assert res[r][(1, full)] == 100.0 * hi + 10.0 * 0 + int(full)
            else:
                assert (1, full) not in res[r]
