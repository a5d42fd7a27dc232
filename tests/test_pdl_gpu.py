"""Programmatic dependent launch of the step kernels (lbmhd_ops.cuh launch_pdl, lbmhd_kernels.cuh pdl_enter):
step n+1 may be scheduled while step n drains, and must not touch memory before step n has completed.  A step that started
early would read populations the previous step has not stored yet: checked bit for bit against the same run with plain
launches (LBMHD_PDL=0), on grids of several waves so that consecutive steps do overlap at their ends, both streaming modes,
both step kernels, with other kernels (moments, halo packs) between the steps."""
import os

import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from test_parity_gpu import gpu_from_workload

pytestmark = pytest.mark.gpu


@pytest.fixture
def env():
    saved = dict(os.environ)
    yield os.environ
    os.environ.clear()
    os.environ.update(saved)


def run(w, pdl, streaming, precision, chunks):
    os.environ["LBMHD_PDL"] = pdl
    os.environ["LBMHD_PERSIST"] = "0"
    g = gpu_from_workload(w, precision=precision, streaming=streaming)
    g.init(w["fields"])
    mids = []
    for n in chunks:
        g.step(n)
        mids.append(g.moments()[1])          # a plain launch between two chains of dependent launches
    path = g.step_path
    pops = g.populations()
    g.close()
    return pops, mids, path


@pytest.mark.parametrize("name,path", [("C2i", "PATH_ONE"), ("C3", "PATH_MULTI"), ("C2", None)])
@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision", [64, 32])
def test_dependent_launches_equal_plain_launches(env, name, path, streaming, precision):
    from paper_2606_00641_b200 import lbmhd
    w = W.get(name)
    chunks = [37, 1, 62]
    p0, m0, path0 = run(w, "0", streaming, precision, chunks)
    p1, m1, path1 = run(w, "1", streaming, precision, chunks)
    assert path0 == path1 and (path is None or path1 == getattr(lbmhd, path))
    assert np.array_equal(p0, p1)
    for a, b in zip(m0, m1):
        assert np.array_equal(a, b)


def test_dependent_launches_on_a_3d_lattice_with_a_body(env):
    """D3Q19 with the moving sphere (per-step arguments change from launch to launch) and non-periodic faces"""
    w = W.config5(shape=(128, 32, 32))
    for streaming in (0, 1):
        p0, m0, _ = run(w, "0", streaming, 64, [25, 25])
        p1, m1, _ = run(w, "1", streaming, 64, [25, 25])
        assert np.array_equal(p0, p1)
        assert np.array_equal(m0[-1], m1[-1])
