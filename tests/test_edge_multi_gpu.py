"""Parity of step_kernel_multi<.., EDGE = true> (rows made of whole multi-cell tiles, the x-face cells inside the end tiles:
periodic wrap, zero-gradient substitution, frozen inflow cell) against the oracle.  It is what lbmhd_step takes
whenever nx is a multiple of the tile width (64 or 128 cells) and the grid is large enough for the multi-cell kernel;
LBMHD_MULTI=1 lets the small grids of these tests reach that kernel, LBMHD_EDGE_MULTI=0 gives the 32-cell edge tiles back."""
import os

import numpy as np
import pytest

from parity_util import TOL64, TOL32
from test_parity_gpu import compare, random_workload, divb_workload, resist_workload

pytestmark = pytest.mark.gpu


@pytest.fixture
def env():
    saved = dict(os.environ)
    yield os.environ
    os.environ.clear()
    os.environ.update(saved)


GRIDS = [("D3Q7", (384, 6, 5), (0,) * 6), ("D3Q7", (384, 5, 4), (1, 1, 0, 0, 0, 0)), ("D3Q7", (256, 6, 5), (2, 1, 1, 1, 0, 0)),
         ("D3Q7", (512, 4, 5), (1, 2, 0, 0, 1, 1)), ("D3Q19", (384, 5, 4), (2, 1, 0, 0, 0, 0)), ("D3Q19", (256, 5, 6), (0,) * 6),
         ("D2Q9", (384, 6), (1, 1, 1, 1, 0, 0)), ("D2Q9", (256, 7), (1, 2, 0, 0, 0, 0)), ("D2Q5", (384, 6), (0,) * 6),
         ("D1Q3", (384,), (1, 2, 0, 0, 0, 0)), ("D1Q3", (512,), (0,) * 6)]


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(32, TOL32), (64, TOL64)])
@pytest.mark.parametrize("lattice,shape,bc", GRIDS)
def test_edge_tiles_ideal(env, lattice, shape, bc, precision, tol, streaming):
    env["LBMHD_MULTI"] = "1"
    env["LBMHD_EDGE_MULTI"] = "1"
    w = random_workload("IDEAL", lattice, shape, bc, seed=601)
    compare(w, 9, tol=tol, precision=precision, streaming=streaming)
    compare(w, 4, tol=tol, precision=precision, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(32, TOL32), (64, TOL64)])
@pytest.mark.parametrize("lattice,shape,bc", [GRIDS[1], GRIDS[2], GRIDS[4], GRIDS[6]])
def test_edge_tiles_other_schemes(env, lattice, shape, bc, precision, tol, streaming):
    env["LBMHD_MULTI"] = "1"
    env["LBMHD_EDGE_MULTI"] = "1"
    compare(random_workload("INCRES", lattice, shape, bc, seed=602), 7, tol=tol, precision=precision, streaming=streaming)
    compare(divb_workload(lattice, shape, bc, seed=603), 7, tol=tol, precision=precision, streaming=streaming)
    compare(resist_workload(lattice, shape, bc, seed=604), 7, tol=tol, precision=precision, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
def test_edge_tiles_equal_the_plain_layout(env, streaming):
    """the same run with the face cells in 32-cell edge tiles (LBMHD_EDGE_MULTI=0): equal to rounding"""
    from paper_2606_00641_b200 import lbmhd
    env["LBMHD_MULTI"] = "1"
    w = random_workload("IDEAL", "D3Q7", (384, 6, 5), (2, 1, 0, 0, 0, 0), seed=605)
    out = []
    for knob in ("1", "0"):
        env["LBMHD_EDGE_MULTI"] = knob
        g = lbmhd.from_workload(w, precision=32, streaming=streaming)
        g.init(w["fields"])
        g.step(9)
        assert g.step_path == lbmhd.PATH_MULTI
        out.append(g.moments()[0])
        g.close()
    assert np.abs(out[0] - out[1]).max() <= 1e-5 * np.abs(out[1]).max()


def test_edge_tiles_with_sphere_and_step_in_pieces(env):
    env["LBMHD_MULTI"] = "1"
    env["LBMHD_EDGE_MULTI"] = "1"
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=np.array([30.0, 8.0, 7.0]), radius=5.0, u_solid=np.array([-0.3, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03)
    w = random_workload("IDEAL", "D3Q7", (384, 16, 14), (2, 1, 0, 0, 0, 0), seed=606, sphere=sph)      # the sphere reaches the first tile
    for streaming in (0, 1):
        compare(w, 8, tol=TOL32, precision=32, streaming=streaming)
