"""The distributed driver of the slab exchange end to end: two processes, one slab each, torch.distributed (gloo, packed
planes staged through host memory because both ranks share the one GPU of this box; their kernels never wait on one
another — the exchange happens on the host between steps).  Result against the unsharded run."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2606_00641_b200 import slab, workloads as W
    w = W.get("C5", small=True)
    res = []
    for streaming, overlap in ((0, False), (0, True), (1, True)):
        sl = slab.Slab(w, rank, world, streaming=streaming)
        ex = slab.DistributedExchange(sl, dist, via_host=True, overlap=overlap)
        sl.init(w["fields"])
        ex.prime()
        for _ in range(13):
            ex.step()
        F, dg = ex.moments()
        res.append((np.ascontiguousarray(sl.owned(F)), dg))
        sl.sim.close()
    F, dg = res[0]
    for F2, dg2 in res[1:]:             # the overlapped schedule and the in-place layout give the serial A/B result
        assert np.abs(F2 - F).max() <= 1e-13 * np.abs(F).max()
        assert np.allclose(dg2, dg, rtol=1e-11, atol=1e-14)
    q.put((rank, F, dg))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_slabs_match_unsharded():
    sys.path.insert(0, ROOT)
    from paper_2606_00641_b200 import lbmhd, slab, workloads as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29900 + os.getpid() % 90
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    Qs = np.concatenate([res[0][1], res[1][1]], axis=1)
    ds = slab.combine_diag([res[0][2], res[1][2]], 8)
    w = W.get("C5", small=True)
    ref = lbmhd.from_workload(w)
    ref.init(w["fields"])
    ref.step(13)
    Qr, dr = ref.moments()
    scale = np.abs(Qr).reshape(8, -1).max(1).reshape(8, 1, 1, 1)
    assert (np.abs(Qs - Qr) / scale).max() <= 1e-13
    assert np.allclose(ds[:16], dr[:16], rtol=1e-12, atol=1e-14) and np.allclose(ds[16:27], dr[16:27], rtol=1e-12, atol=1e-14)


def test_bench_slab_mode_two_ranks_on_one_gpu():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(29990 + os.getpid() % 9), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "4", "--warmup", "3",
           "--decomp", "slab", "--backend", "gloo", "--shape", "96x64x32", "--no-cpu-baseline"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["value"] > 0 and line["gpu_launches"] >= 4 and line["config"]["cells"] == 2 * 96 * 64 * 32
