"""In-place (AA pattern) streaming: one population copy, same results as the A/B path and the oracle at every
step count (both layouts P0 / P1 visible through lbmhd_moments and lbmhd_get_populations)."""
import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from parity_util import oracle_from_workload, field_errors, TOL64
from test_parity_gpu import CASES, compare, random_workload, gpu_from_workload
from test_oracle_pins import zyx

pytestmark = pytest.mark.gpu
INPLACE = 1


@pytest.mark.parametrize("scheme,lattice,shape,bc", CASES)
def test_inplace_random_state_parity(scheme, lattice, shape, bc):
    w = random_workload(scheme, lattice, shape, bc, seed=4321)
    compare(w, 20, streaming=INPLACE)
    compare(w, 7, streaming=INPLACE)          # odd count: the state is left in layout P1


@pytest.mark.parametrize("name", ["C1", "C2", "C2i", "C3", "C4", "C5"])
def test_inplace_config_parity_100_steps(name):
    errs = compare(W.get(name, small=True), 100, streaming=INPLACE)
    print(name, "in place, max field error", errs.max())


def test_inplace_every_step_and_populations():
    """step by step: moments and the exported canonical populations agree with the oracle in both layouts"""
    w = random_workload("IDEAL", "D3Q19", (70, 9, 8), (2, 1, 1, 1, 0, 0), seed=11)
    o = oracle_from_workload(w)
    g = gpu_from_workload(w, streaming=INPLACE)
    o.init(w["fields"])
    g.init(w["fields"])
    for step in range(1, 8):
        o.step(1)
        g.step(1)
        assert (field_errors(g.moments()[0], o.moments()[0]) <= TOL64).all(), step
        po, pg = o.populations(), g.populations()
        # frozen cells are re-materialised as f^eq of their state (A10); everything else element by element
        assert np.abs(pg - po).max() <= 1e-13, step
    g.close()


def test_inplace_masked_obstacle_and_sphere():
    rng = np.random.default_rng(5)
    shape = (70, 12, 10)
    s = zyx(shape)
    w = random_workload("IDEAL", "D3Q19", shape, (1, 1) + (0,) * 4, seed=6)
    mask = (rng.random(s) < 0.05).astype(np.uint8) * 2
    mask[rng.random(s) < 0.02] = 1
    Bs = 0.1 * (rng.random((3,) + s) - 0.5)
    compare(w, 15, obstacle=(mask, np.array([0.03, -0.02, 0.01]), Bs), streaming=INPLACE)
    cen = np.array([36.0, 12.0, 10.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03)
    w2 = random_workload("IDEAL", "D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=7, sphere=sph)
    compare(w2, 13, streaming=INPLACE)


def test_inplace_halves_the_population_footprint():
    from paper_2606_00641_b200 import lbmhd
    ab = lbmhd.workspace_bytes(lbmhd.make_params("IDEAL", "D3Q19", (384, 256, 256), streaming=0))
    ip = lbmhd.workspace_bytes(lbmhd.make_params("IDEAL", "D3Q19", (384, 256, 256), streaming=1))
    assert ip < 0.6 * ab and ip < 37e9
