"""N > 1 host logic of bench.py on CPU: two gloo ranks, max-over-ranks timing and whole-job aggregation.
(The data path has no collective: every rank steps its own replica.)"""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r "measured" (10 + r) ms for the device leg and (30 - 5 r) ms end to end
    ms = bench.max_over_ranks([10.0 + rank, 30.0 - 5.0 * rank], world)
    dist.barrier()
    q.put((rank, ms, bench.aggregate_mlups(1000000, 20, ms[0], world)))
    dist.destroy_process_group()


def test_two_rank_max_and_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 1000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, ms, val in out:
        assert ms == [11.0, 30.0]                          # max over ranks, element-wise
        assert val == pytest.approx(2 * 1000000 * 20 / 11e-3 / 1e6)   # both replicas count, slowest rank's clock


def test_single_rank_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], 1) == [1.5, 2.5]
    assert bench.aggregate_mlups(25165824, 50, 500.0, 1) == pytest.approx(25165824 * 50 / 0.5 / 1e6)
