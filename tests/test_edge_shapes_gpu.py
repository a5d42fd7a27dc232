"""Degenerate and ragged shapes: tiny grids (3 cells on a non-periodic axis, one tile or less in x), odd sizes, every
boundary combination, both streaming modes, all lattices and schemes — a seeded sweep against the oracle."""
import numpy as np
import pytest

from test_parity_gpu import compare, random_workload, divb_workload, resist_workload, full_workload
from parity_util import TOL64, TOL32

pytestmark = pytest.mark.gpu


def random_case(rng):
    lattice = rng.choice(["D1Q3", "D2Q9", "D3Q19", "D2Q5", "D3Q7"])
    D = {"D1Q3": 1, "D2Q9": 2, "D3Q19": 3, "D2Q5": 2, "D3Q7": 3}[lattice]
    scheme = rng.choice(["IDEAL", "INCRES", "IDEAL_DIVB", "RESIST"])
    bc = [0] * 6
    shape = []
    for a in range(D):
        kind = rng.integers(0, 4)          # 0 periodic, 1 zerograd/zerograd, 2 inflow/zerograd, 3 zerograd/inflow
        bc[2 * a], bc[2 * a + 1] = [(0, 0), (1, 1), (2, 1), (1, 2)][kind]
        if a == 0:
            n = int(rng.choice([3, 4, 5, 31, 32, 33, 63, 64, 65, 70, 97, 130]))
        else:
            n = int(rng.choice([1, 2, 3, 4, 5, 7])) if kind == 0 else int(rng.choice([3, 4, 5, 7]))
        shape.append(n)
    return scheme, lattice, tuple(shape), tuple(bc)


@pytest.mark.parametrize("seed", range(60))
def test_random_small_shapes(seed):
    rng = np.random.default_rng(9000 + seed)
    scheme, lattice, shape, bc = random_case(rng)
    streaming = int(rng.integers(0, 2))
    precision = 64 if rng.random() < 0.75 else 32
    if scheme == "IDEAL_DIVB":
        w = divb_workload(lattice, shape, bc, seed=seed)
    elif scheme == "RESIST":
        w = resist_workload(lattice, shape, bc, seed=seed)
    else:
        w = random_workload(scheme, lattice, shape, bc, seed=seed)
    steps = int(rng.integers(1, 7))
    compare(w, steps, tol=TOL64 if precision == 64 else TOL32, precision=precision, streaming=streaming)


@pytest.mark.parametrize("seed", range(20))
def test_random_small_shapes_full_scheme(seed):
    """the same sweep for the 8 + 6 D sets of the full dissipative scheme (blocks of up to 26 variable rows)"""
    rng = np.random.default_rng(9500 + seed)
    _, lattice, shape, bc = random_case(rng)
    streaming = int(rng.integers(0, 2))
    precision = 64 if rng.random() < 0.75 else 32
    steps = int(rng.integers(1, 7))
    compare(full_workload(lattice, shape, bc, seed=seed), steps, tol=TOL64 if precision == 64 else TOL32, precision=precision,
            streaming=streaming)


def test_single_cell_rows_and_zero_steps():
    """periodic axes of length 1 and 2 (a cell is its own neighbour), n_steps = 0"""
    for shape in [(40, 1), (40, 2), (33, 1, 1), (33, 2, 1), (33, 1, 2)]:
        lat = "D2Q9" if len(shape) == 2 else "D3Q19"
        for streaming in (0, 1):
            compare(random_workload("IDEAL", lat, shape, (0,) * 6, seed=5), 5, streaming=streaming)
            compare(random_workload("IDEAL", lat, shape, (0,) * 6, seed=5), 0, streaming=streaming)
