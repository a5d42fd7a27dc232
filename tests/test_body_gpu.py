"""Body integrals of the CUDA path against the oracle (A21): force, torque, work,
injected and enclosed magnetic field.  `compare` of test_parity_gpu.py checks them in every parity case that has a
solid; here: the reference point of masked bodies, read-and-reset, the per-step series written to device memory,
fp32, and the sharded run."""
import numpy as np
import pytest

from paper_2606_00641_b200 import lbmhd, slab
from parity_util import oracle_from_workload, TOL64, TOL32
from test_oracle_pins import zyx
from test_parity_gpu import assert_body_close, gpu_from_workload, random_workload

pytestmark = pytest.mark.gpu


def sphere_workload(scheme, lattice, shape, seed, bc=(2, 1, 0, 0, 0, 0), width=1.5, omega=(0.02, 0.0, 0.02)):
    D = len(shape)
    cen = np.array([shape[0] / 2.0 + 0.3, shape[1] / 2.0 + 0.1, shape[2] / 2.0 + 0.2 if D == 3 else 0.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    om = np.array(omega if D == 3 else (0.0, 0.0, omega[0]))
    sph = dict(centre=cen, radius=min(shape) / 4.0, u_solid=np.array([-0.05, 0.02, 0.0]), dipole_dir=mh, B_surface=0.03,
               width=width, omega=om)
    return random_workload(scheme, lattice, shape, bc, seed=seed, sphere=sph)


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("scheme,lattice,shape", [("IDEAL", "D3Q19", (72, 24, 20)), ("IDEAL", "D2Q9", (90, 40)), ("INCRES", "D2Q9", (90, 40)),
                                                  ("IDEAL", "D3Q7", (72, 24, 20)), ("INCRES", "D3Q19", (40, 20, 16))])
def test_sphere_body_series(scheme, lattice, shape, streaming):
    """per-step series: one read-and-reset per step into a device tensor, no host synchronisation in the loop"""
    import torch
    w = sphere_workload(scheme, lattice, shape, seed=31)
    o = oracle_from_workload(w)
    g = gpu_from_workload(w, streaming=streaming)
    g.body_enable(True)
    o.init(w["fields"])
    g.init(w["fields"])
    steps = 9
    series = torch.zeros(steps, 14, dtype=torch.float64, device="cuda")
    want = np.zeros((steps, 14))
    for s in range(steps):
        g.step(1)
        g.body_read(reset=True, out=series[s])
        o.step(1)
        want[s] = o.body_read(reset=True)
    torch.cuda.synchronize()
    got = series.cpu().numpy()
    _, do = o.moments()
    qmax = do[2 * o.K:3 * o.K].max()
    for s in range(steps):
        assert_body_close(got[s], want[s], TOL64, qmax, max(shape))
    assert np.abs(want[:, 0:3]).max() > 1e-4 and np.abs(want[:, 3:6]).max() > 1e-4      # not trivially zero
    assert np.all(g.body_read() == 0.0)
    g.close()


@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
def test_masked_body_reference_point(precision, tol):
    rng = np.random.default_rng(41)
    shape = (70, 14, 12)
    s = zyx(shape)
    w = random_workload("IDEAL", "D3Q19", shape, (1, 1) + (0,) * 4, seed=42)
    mask = np.zeros(s, dtype=np.uint8)
    mask[3:9, 4:11, 20:41] = 2
    d = np.ones(s)
    d[mask == 2] = rng.random(int((mask == 2).sum())) * 0.9
    Bs = 0.05 * (rng.random((3,) + s) - 0.5)
    ref = np.array([30.5, 7.25, 6.0])
    o = oracle_from_workload(w)
    g = gpu_from_workload(w, precision=precision)
    for sim in (o, g):
        sim.set_obstacle(mask, np.array([0.02, -0.01, 0.015]), Bs)
        sim.set_porosity(d)
    o.set_body_reference(ref)
    g.body_enable(True, ref)
    o.init(w["fields"])
    g.init(w["fields"])
    o.step(6)
    g.step(6)
    _, do = o.moments()
    bo, bg = o.body_read(), g.body_read()
    assert_body_close(bg, bo, tol, do[2 * o.K:3 * o.K].max(), max(shape))
    assert np.abs(bo[3:6]).max() > 1e-3
    g.close()


def test_body_read_needs_enable():
    w = random_workload("IDEAL", "D2Q9", (40, 12), (0,) * 6, seed=3)
    g = gpu_from_workload(w)
    g.init(w["fields"])
    with pytest.raises(lbmhd.LbmhdError):
        g.body_read()
    g.close()


@pytest.mark.parametrize("parts", [2, 3])
def test_sharded_body_integrals_add_up(parts):
    """slabs accumulate over their owned cells only (ghost planes do no work): the sum over slabs is the unsharded value"""
    w = sphere_workload("IDEAL", "D3Q19", (48, 16, 18), seed=51, bc=(2, 1, 0, 0, 0, 0))
    o = oracle_from_workload(w)
    grp = slab.LocalSlabGroup(w, parts)
    grp.body_enable(True)
    o.init(w["fields"])
    grp.init(w["fields"])
    o.step(7)
    grp.step(7)
    _, do = o.moments()
    assert_body_close(grp.body_read(), o.body_read(), TOL64, do[2 * o.K:3 * o.K].max(), 48)
    grp.close()


def dipoles(R):
    """four dipoles inside a body of radius R; cores >= 0.45 R keep the capped field below ~0.1 (lattice units)"""
    return dict(offsets=R / 5.0 * np.array([[1.5, 0.0, 0.5], [-1.0, 2.0, 0.0], [0.0, -1.5, -2.0], [0.5, 0.5, 2.5]]),
                dirs=np.array([[0.0, 0.0, 1.0], [0.6, 0.0, 0.8], [1.0, 0.0, 0.0], [0.0, -0.8, 0.6]]),
                B_surface=np.array([0.01, -0.008, 0.006, 0.009]), cores=R * np.array([0.5, 0.6, 0.45, 0.7]))


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape", [("D3Q19", (72, 24, 20)), ("D2Q9", (90, 40))])
def test_dipole_ensemble_parity(lattice, shape, precision, tol, streaming):
    """four shifted, capped dipoles fixed in the frame of the tumbling sphere"""
    from test_parity_gpu import compare
    w = sphere_workload("IDEAL", lattice, shape, seed=61)
    w["sphere"]["dipoles"] = dipoles(w["sphere"]["radius"])
    compare(w, 11, tol=tol, precision=precision, streaming=streaming)


def test_dipole_ensemble_sharded():
    w = sphere_workload("IDEAL", "D3Q19", (48, 16, 18), seed=62)
    w["sphere"]["dipoles"] = dipoles(w["sphere"]["radius"])
    o = oracle_from_workload(w)
    grp = slab.LocalSlabGroup(w, 3)
    o.init(w["fields"])
    grp.init(w["fields"])
    o.step(6)
    grp.step(6)
    Qo, _ = o.moments()
    Qg, _ = grp.moments()
    from parity_util import field_errors
    assert (field_errors(Qg, Qo) <= TOL64).all()
    grp.close()


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("scheme,lattice,shape", [("IDEAL", "D3Q19", (70, 14, 12)), ("INCRES", "D2Q9", (80, 30))])
def test_rotating_masked_body_parity(scheme, lattice, shape, streaming):
    """u^B = u_solid + omega x (x - centre) at the cells of a masked body with porosity"""
    from parity_util import field_errors
    rng = np.random.default_rng(71)
    D = len(shape)
    s = zyx(shape)
    w = random_workload(scheme, lattice, shape, (1, 1) + (0,) * 4, seed=72)
    mask = np.zeros(s, dtype=np.uint8)
    mask[..., 4:11, 20:41] = 2
    d = np.ones(s)
    d[mask == 2] = rng.random(int((mask == 2).sum())) * 0.9
    Bs = 0.05 * (rng.random((3,) + s) - 0.5)
    cen = np.array([30.5, 7.25, 6.0 if D == 3 else 0.0])
    om = np.array([0.002, -0.003, 0.004]) if D == 3 else np.array([0.0, 0.0, 0.004])
    o = oracle_from_workload(w)
    g = gpu_from_workload(w, streaming=streaming)
    for sim in (o, g):
        sim.set_obstacle(mask, np.array([0.02, -0.01, 0.015 if D == 3 else 0.0]), Bs)
        sim.set_porosity(d)
        sim.set_obstacle_rotation(om, cen)
    o.set_body_reference(cen)
    g.body_enable(True, cen)
    o.init(w["fields"])
    g.init(w["fields"])
    o.step(8)
    g.step(8)
    Qo, do = o.moments()
    assert (field_errors(g.moments()[0], Qo) <= TOL64).all()
    assert_body_close(g.body_read(), o.body_read(), TOL64, do[2 * o.K:3 * o.K].max(), max(shape))
    g.close()
