"""Parity of the multi-cell kernels (step_kernel_multi: several adjacent cells per thread on interior tiles, DESIGN.md
§5.5) and of the 2-CTA cluster split of the RESIST rows (step_kernel_cl, §5.6) against the oracle.

The library takes the multi-cell kernel only on grids large enough to fill the GPU; LBMHD_MULTI=1 forces it so that
grids the oracle finishes in seconds reach it.  nx = 292: one 128-cell tile (fp32 short lattices), three 64-cell tiles,
a ragged 4-cell tail; the sphere cuts through multi-cell tiles (those fall back to the one-cell paths piece by piece)."""
import os

import numpy as np
import pytest

from parity_util import TOL64, TOL32
from test_parity_gpu import compare, random_workload, divb_workload, resist_workload, full_workload

pytestmark = pytest.mark.gpu


@pytest.fixture
def env():
    saved = dict(os.environ)
    yield os.environ
    os.environ.clear()
    os.environ.update(saved)


GRIDS = [("D1Q3", (292,), (1, 1, 0, 0, 0, 0)), ("D1Q3", (292,), (0,) * 6),
         ("D2Q5", (292, 9), (2, 1, 0, 0, 0, 0)), ("D2Q9", (292, 9), (0,) * 6), ("D2Q9", (292, 7), (1, 1, 1, 1, 0, 0)),
         ("D3Q7", (292, 6, 5), (0, 0, 1, 1, 0, 0)), ("D3Q19", (292, 6, 5), (2, 1, 0, 0, 0, 0)),
         ("D3Q19", (292, 5, 6), (0, 0, 0, 0, 1, 1)),
         # nx a multiple of the tile widths (64, 128), every x-boundary kind
         ("D1Q3", (384,), (1, 2, 0, 0, 0, 0)), ("D2Q5", (384, 6), (0,) * 6), ("D2Q9", (384, 6), (2, 1, 1, 1, 0, 0)),
         ("D2Q9", (256, 7), (1, 2, 0, 0, 0, 0)), ("D3Q7", (384, 5, 4), (1, 1, 0, 0, 0, 0)), ("D3Q19", (384, 5, 4), (2, 1, 0, 0, 0, 0)),
         ("D3Q19", (128, 5, 6), (0,) * 6), ("D3Q19", (256, 4, 5), (1, 2, 0, 0, 1, 1))]


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", GRIDS)
def test_multi_cell_ideal(env, lattice, shape, bc, precision, tol, streaming):
    env["LBMHD_MULTI"] = "1"
    w = random_workload("IDEAL", lattice, shape, bc, seed=101)
    compare(w, 9, tol=tol, precision=precision, streaming=streaming)
    compare(w, 4, tol=tol, precision=precision, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", [GRIDS[0], GRIDS[2], GRIDS[4], GRIDS[5], GRIDS[6], GRIDS[8], GRIDS[10], GRIDS[13], GRIDS[15]])
def test_multi_cell_other_schemes(env, lattice, shape, bc, precision, tol, streaming):
    env["LBMHD_MULTI"] = "1"
    compare(random_workload("INCRES", lattice, shape, bc, seed=102), 7, tol=tol, precision=precision, streaming=streaming)
    compare(divb_workload(lattice, shape, bc, seed=103), 7, tol=tol, precision=precision, streaming=streaming)
    compare(resist_workload(lattice, shape, bc, seed=104), 7, tol=tol, precision=precision, streaming=streaming)
    compare(full_workload(lattice, shape, bc, seed=111), 7, tol=tol, precision=precision, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
def test_multi_cell_with_sphere(env, precision, tol, streaming):
    env["LBMHD_MULTI"] = "1"
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=np.array([150.0, 8.0, 7.0]), radius=5.0, u_solid=np.array([-0.3, 0.0, 0.0]), dipole_dir=mh,
               B_surface=0.03, width=1.5)
    for lattice in ("D3Q19", "D3Q7"):
        for nx in (292, 384):
            compare(random_workload("IDEAL", lattice, (nx, 16, 14), (2, 1, 0, 0, 0, 0), seed=105, sphere=sph), 8, tol=tol,
                    precision=precision, streaming=streaming)


def test_multi_cell_is_taken_and_matches_one_cell(env):
    """the forced multi-cell run and the one-cell run (LBMHD_PAIR=0) agree to rounding; both are the C-ABI path"""
    from paper_2606_00641_b200 import lbmhd
    w = random_workload("IDEAL", "D3Q19", (292, 6, 5), (0,) * 6, seed=106)
    out = []
    for knobs in ({"LBMHD_MULTI": "1"}, {"LBMHD_PAIR": "0"}):
        env.pop("LBMHD_MULTI", None)
        env.pop("LBMHD_PAIR", None)
        env.update(knobs)
        g = lbmhd.from_workload(w)
        g.init(w["fields"])
        assert g.step_path == -1
        g.step(6)
        assert g.step_path == (lbmhd.PATH_MULTI if "LBMHD_MULTI" in knobs else lbmhd.PATH_ONE)
        out.append(g.moments()[0])
        g.close()
    assert np.abs(out[0] - out[1]).max() <= 1e-13 * np.abs(out[1]).max()


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("lattice,shape", [("D1Q3", (292,)), ("D2Q5", (292, 9)), ("D2Q9", (292, 9)), ("D3Q7", (292, 6, 5)),
                                           ("D3Q19", (292, 6, 5))])
def test_forced_multi_path_is_the_one_that_ran(env, lattice, shape, precision):
    """the knob the parity cases above rely on really selects step_kernel_multi (every lattice and precision has one for K = 8)"""
    from paper_2606_00641_b200 import lbmhd
    env["LBMHD_MULTI"] = "1"
    w = random_workload("IDEAL", lattice, shape, (0,) * 6, seed=109)
    for streaming in (0, 1):
        g = lbmhd.from_workload(w, precision=precision, streaming=streaming)
        g.init(w["fields"])
        g.step(2)
        assert g.step_path == lbmhd.PATH_MULTI
        g.close()


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("cluster", ["1", "0"])
def test_resist_cluster_split_and_plain(env, cluster, streaming):
    """RESIST on D3Q19, fp64: rows split over a 2-CTA cluster (default) and the plain 17-row block"""
    from paper_2606_00641_b200 import lbmhd
    env["LBMHD_CLUSTER"] = cluster
    w0 = resist_workload("D3Q19", (64, 6, 5), (0,) * 6, seed=110)
    g = lbmhd.from_workload(w0, streaming=streaming)
    g.init(w0["fields"])
    g.step(1)
    assert g.step_path == (lbmhd.PATH_CLUSTER if cluster == "1" else lbmhd.PATH_ONE)
    g.close()
    compare(resist_workload("D3Q19", (200, 12, 9), (2, 1, 0, 0, 0, 0), seed=107), 11, streaming=streaming)
    compare(resist_workload("D3Q19", (45, 11, 10), (1, 1, 1, 1, 1, 1), seed=108), 6, streaming=streaming)
