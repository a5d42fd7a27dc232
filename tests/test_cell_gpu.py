"""Parity of the cell-per-thread kernel (step_kernel_cell: one thread owns a cell and all its K population
sets; the short lattices D1Q3 / D2Q5 / D3Q7) against the oracle.  The library takes it on grids large enough to fill the GPU;
LBMHD_CELL=2 forces it so that grids the oracle finishes in seconds reach it.  Shapes: rows longer than one cell tile plus a
ragged tail, row counts that are not a multiple of the tile's row count, every boundary kind, the sphere cutting through
cell tiles (those fall back to the one-cell-per-(cell, variable) paths piece by piece)."""
import os

import numpy as np
import pytest

from parity_util import TOL64, TOL32
from test_parity_gpu import compare, random_workload, divb_workload, gpu_from_workload

pytestmark = pytest.mark.gpu


@pytest.fixture
def env():
    saved = dict(os.environ)
    yield os.environ
    os.environ.clear()
    os.environ.update(saved)


GRIDS = [("D1Q3", (600,), (1, 1, 0, 0, 0, 0)), ("D1Q3", (517,), (0,) * 6), ("D1Q3", (640,), (2, 1, 0, 0, 0, 0)),
         ("D2Q5", (292, 9), (2, 1, 0, 0, 0, 0)), ("D2Q5", (292, 10), (0,) * 6), ("D2Q5", (256, 13), (1, 1, 1, 1, 0, 0)),
         ("D3Q7", (292, 6, 5), (0, 0, 1, 1, 0, 0)), ("D3Q7", (200, 11, 6), (2, 1, 0, 0, 0, 0)), ("D3Q7", (192, 9, 7), (1, 2, 1, 1, 1, 1))]


def used_path(w, precision=64, streaming=0):
    g = gpu_from_workload(w, precision=precision, streaming=streaming)
    g.init(w["fields"])
    g.step(1)
    p = g.step_path
    g.close()
    return p


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", GRIDS)
def test_cell_kernel_ideal(env, lattice, shape, bc, precision, tol, streaming):
    from paper_2606_00641_b200 import lbmhd
    env["LBMHD_CELL"] = "2"
    w = random_workload("IDEAL", lattice, shape, bc, seed=201)
    assert used_path(w, precision, streaming) == lbmhd.PATH_CELL
    compare(w, 9, tol=tol, precision=precision, streaming=streaming)
    compare(w, 4, tol=tol, precision=precision, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", [GRIDS[0], GRIDS[3], GRIDS[5], GRIDS[7], GRIDS[8]])
def test_cell_kernel_other_schemes(env, lattice, shape, bc, precision, tol, streaming):
    from paper_2606_00641_b200 import lbmhd
    env["LBMHD_CELL"] = "2"
    D = len(shape)
    wi = random_workload("INCRES", lattice, shape if D < 3 else (shape[0] + 64, shape[1], shape[2]), bc, seed=202)
    if wi["shape"][0] >= 64 + 32 * (1 + 2 * D):      # INCRES tiles are 32 (1 + 2 D) cells wide
        assert used_path(wi, precision, streaming) == lbmhd.PATH_CELL
    compare(wi, 7, tol=tol, precision=precision, streaming=streaming)
    wd = divb_workload(lattice, (max(shape[0], 200),) + tuple(shape[1:]), bc, seed=203)
    assert used_path(wd, precision, streaming) == lbmhd.PATH_CELL
    compare(wd, 7, tol=tol, precision=precision, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
def test_cell_kernel_with_sphere(env, precision, tol, streaming):
    """the sphere crosses cell tiles: touched tiles take the fallback, the others the cell path"""
    env["LBMHD_CELL"] = "2"
    cen = np.array([150.3, 10.1, 6.2])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=5.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03, width=1.5)
    w = random_workload("IDEAL", "D3Q7", (292, 20, 12), (2, 1, 0, 0, 0, 0), seed=204, sphere=sph)
    compare(w, 14, tol=tol, precision=precision, streaming=streaming)
    w2 = random_workload("IDEAL", "D2Q5", (292, 24), (2, 1, 1, 1, 0, 0), seed=205, sphere=dict(sph, centre=np.array([150.3, 12.1, 0.0])))
    compare(w2, 14, tol=tol, precision=precision, streaming=streaming)


def test_cell_kernel_masked_grid_falls_back(env):
    env["LBMHD_CELL"] = "2"
    rng = np.random.default_rng(206)
    shape = (292, 12)
    mask = (rng.random((1, 12, 292)) < 0.05).astype(np.uint8) * 2
    w = random_workload("IDEAL", "D2Q5", shape, (1, 1, 0, 0, 0, 0), seed=207)
    compare(w, 8, obstacle=(mask, np.array([0.03, -0.02, 0.0]), None))


def test_cell_kernel_step_in_pieces(env):
    """plane ranges (slab overlap) through the cell kernel: 2D ranges that cut a tile's row group"""
    env["LBMHD_CELL"] = "2"
    for lattice, shape, bc in (("D2Q5", (292, 23), (1, 1, 1, 1, 0, 0)), ("D3Q7", (200, 9, 8), (2, 1, 0, 0, 0, 0))):
        for streaming in (0, 1):
            w = random_workload("IDEAL", lattice, shape, bc, seed=208)
            a, b = gpu_from_workload(w, streaming=streaming), gpu_from_workload(w, streaming=streaming)
            nH = shape[-1]
            for g in (a, b):
                g.init(w["fields"])
            for _ in range(4):
                a.step(1)
                b.step_part(nH - 3, nH, False)
                b.step_part(0, 2, False)
                b.step_part(2, nH - 3, True)
            # rows change between the cell path and the fallback paths with the partition: equal up to rounding, not bitwise
            Qa, Qb = a.moments()[0], b.moments()[0]
            assert np.abs(Qa - Qb).max() <= 1e-13 * np.abs(Qa).max()
            a.close()
            b.close()
