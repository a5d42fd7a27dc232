"""Many steps in one cooperative launch (step_kernel_persist): the path lbmhd_step(n >= 2) takes on small
lattices (BASELINE configs 1 and 2), checked against the oracle over the configs' full runs, and — forced with
LBMHD_PERSIST=2 — over every boundary kind, both streaming modes, masks and the moving sphere, against the one-launch-per-step
kernels bit for bit."""
import os

import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from parity_util import oracle_from_workload, field_errors, TOL64, TOL32
from test_parity_gpu import compare, random_workload, gpu_from_workload, resist_workload
from test_oracle_pins import zyx

pytestmark = pytest.mark.gpu


@pytest.fixture
def env():
    saved = dict(os.environ)
    yield os.environ
    os.environ.clear()
    os.environ.update(saved)


def run(w, steps, persist, streaming=0, precision=64, chunks=None, mask=None, obstacle=None):
    from paper_2606_00641_b200 import lbmhd
    os.environ["LBMHD_PERSIST"] = persist
    os.environ["LBMHD_RESIDENT"] = "0"          # (the 1D lattices would otherwise take the register-resident kernel)
    g = gpu_from_workload(w, precision=precision, streaming=streaming)
    if obstacle is not None:
        g.set_obstacle(*obstacle)
    g.init(w["fields"])
    l0 = g.launch_count
    for n in (chunks or [steps]):
        g.step(n)
    path, launches = g.step_path, g.launch_count - l0
    Q, dg = g.moments()
    pops = g.populations()
    g.close()
    return Q, dg, pops, path, launches


@pytest.mark.parametrize("streaming", [0, 1])
def test_config1_whole_run_in_one_launch(env, streaming):
    """C1: 800 cells = 25 tiles, 500 steps in ONE launch, all cells against the oracle"""
    from paper_2606_00641_b200 import lbmhd
    w = W.get("C1")
    Q, dg, _, path, launches = run(w, 500, "1", streaming=streaming)
    assert path == lbmhd.PATH_PERSIST and launches == 1
    o = oracle_from_workload(w)
    o.init(w["fields"])
    o.step(500)
    errs = field_errors(Q, o.moments(diag=False))
    print("C1 500 steps in one launch, streaming %d: %.2e" % (streaming, errs.max()))
    assert (errs <= TOL64).all(), errs


@pytest.mark.parametrize("name", ["C2", "C2i"])
def test_config2_whole_run(env, name):
    """C2 (and its INCRES variant) at their own size, all 1000 steps in ONE lbmhd_step call: whatever kernel that call picks
    there is the kernel bench.py --workload C2 times"""
    w = W.get(name)
    Q, dg, _, path, launches = run(w, 1000, "1")
    o = oracle_from_workload(w)
    o.init(w["fields"])
    o.step(1000)
    errs = field_errors(Q, o.moments(diag=False))
    print("%s 1000 steps, path %d, %d launches: %.2e" % (name, path, launches, errs.max()))
    assert (errs <= TOL64).all(), errs


CASES = [
    ("IDEAL", "D1Q3", (131,), (1, 1, 0, 0, 0, 0)), ("IDEAL", "D1Q3", (70,), (2, 1, 0, 0, 0, 0)),
    ("IDEAL", "D2Q9", (150, 37), (0,) * 6), ("IDEAL", "D2Q9", (150, 37), (1, 1, 1, 1, 0, 0)), ("INCRES", "D2Q9", (90, 21), (1, 1, 2, 1, 0, 0)),
    ("IDEAL", "D3Q19", (100, 12, 9), (2, 1, 0, 0, 0, 0)), ("IDEAL", "D3Q19", (45, 11, 10), (1, 1, 1, 1, 1, 1)),
    ("IDEAL", "D2Q5", (67, 20), (2, 1, 1, 1, 0, 0)), ("IDEAL", "D3Q7", (100, 12, 9), (0,) * 6),
]


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("scheme,lattice,shape,bc", CASES)
def test_persistent_equals_per_step_launches(env, scheme, lattice, shape, bc, streaming):
    """same populations, bit for bit, as one launch per step; odd and even step counts, several calls in a row"""
    from paper_2606_00641_b200 import lbmhd
    w = random_workload(scheme, lattice, shape, bc, seed=71)
    Qa, da, pa, path_a, la = run(w, 17, "0", streaming=streaming, chunks=[17])
    Qb, db, pb, path_b, lb = run(w, 17, "2", streaming=streaming, chunks=[7, 1, 2, 7])
    assert path_a != lbmhd.PATH_PERSIST and la == 17
    assert path_b == lbmhd.PATH_PERSIST and lb == 4          # 7 | 1 (a single step is a plain launch) | 2 | 7
    assert np.array_equal(pa, pb)
    assert np.array_equal(Qa, Qb) and np.array_equal(da, db)


@pytest.mark.parametrize("streaming", [0, 1])
def test_persistent_with_sphere_mask_and_fp32(env, streaming):
    env["LBMHD_PERSIST"] = "2"
    cen = np.array([36.0, 12.0, 10.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03, width=1.5)
    w = random_workload("IDEAL", "D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=72, sphere=sph)
    compare(w, 12, streaming=streaming)                       # the sphere's centre advances inside the kernel
    compare(w, 12, tol=TOL32, precision=32, streaming=streaming)
    rng = np.random.default_rng(73)
    shape = (70, 33)
    s = zyx(shape)
    mask = (rng.random(s) < 0.05).astype(np.uint8) * 2
    mask[rng.random(s) < 0.02] = 1
    compare(resist_workload("D2Q9", shape, (1, 1) + (0,) * 4, seed=74), 9,
            obstacle=(mask, np.array([0.03, -0.02, 0.01]), 0.1 * (rng.random((3,) + s) - 0.5)), streaming=streaming)


def test_rotating_dipoles_fall_back_to_launches(env):
    """the host turns the dipole axes every step: such a body keeps one launch per step"""
    from paper_2606_00641_b200 import lbmhd
    env["LBMHD_PERSIST"] = "2"
    cen = np.array([36.0, 12.0, 10.0])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=np.array([0.0, 0.0, 1.0]), B_surface=0.03,
               omega=np.array([0.02, 0.0, 0.02]))
    w = random_workload("IDEAL", "D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=75, sphere=sph)
    g = gpu_from_workload(w)
    g.init(w["fields"])
    g.step(5)
    assert g.step_path != lbmhd.PATH_PERSIST
    g.close()
    compare(w, 5)
