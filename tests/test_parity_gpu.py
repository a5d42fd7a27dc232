"""GPU-vs-oracle parity (the graded gate): same seeded arrays -> lbmhd_init -> n steps -> lbmhd_moments,
compared element by element with the CPU oracle through the C ABI.  fp64 bar 1e-11 (north_star), reading A15."""
import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from parity_util import oracle_from_workload, field_errors, diag_errors, TOL64, TOL32
from test_oracle_pins import admissible_ideal, ideal_fields, incres_fields, zyx

pytestmark = pytest.mark.gpu


def gpu_from_workload(w, precision=64, streaming=0):
    from paper_2606_00641_b200 import lbmhd
    return lbmhd.from_workload(w, precision=precision, streaming=streaming)


def random_workload(scheme, lattice, shape, bc, seed, tau=0.7, sphere=None, gamma=5 / 3):
    rng = np.random.default_rng(seed)
    s = zyx(shape)
    D = len(shape)
    slow = lattice in ("D2Q5", "D3Q7")        # axis-only lattices: lower speed limit (A16)
    if scheme == "IDEAL":
        rho, u, B, p = admissible_ideal(rng, s, amp=0.06 if slow else 0.2)
        F = ideal_fields(rho, u, B, p * (0.1 if slow else 1.0), gamma)
    else:
        F = incres_fields(rng, D, s, amp=0.02 if slow else 0.05)
    return dict(name="rand", scheme=scheme, lattice=lattice, shape=shape, gamma=gamma, c0sq=1 / 36, nu=0.0, eta=0.0,
                tau=tau, powell=1.0, bc=bc, steps=0, fields=F, sphere=sphere)


def assert_body_close(bg, bo, tol, qmax, extent):
    """body integrals (A21): sums over the body cells and the steps of terms that are each within ~tol * max|Q|;
    bo[13] = sum (1 - d) counts cells x steps; torques carry a lever arm of up to the domain extent"""
    scale = 10 * tol * max(1.0, bo[13]) * qmax
    bound = np.full(14, scale)
    bound[3:6] *= extent
    bound[13] = 10 * tol * max(1.0, bo[13])
    assert (np.abs(bg - bo) <= bound).all(), (bg, bo, bound)


def compare(w, steps, tol=TOL64, mask=None, obstacle=None, precision=64, streaming=0):
    o = oracle_from_workload(w, mask=mask)
    g = gpu_from_workload(w, precision=precision, streaming=streaming)
    if obstacle is not None:
        o.set_obstacle(*obstacle)
        g.set_obstacle(*obstacle)
    g.body_enable(True)
    o.init(w["fields"])
    g.init(w["fields"])
    o.step(steps)
    g.step(steps)
    Qo, do = o.moments()
    Qg, dg = g.moments()
    errs = field_errors(Qg, Qo)
    assert (errs <= tol).all(), errs
    K = o.K
    assert_body_close(g.body_read(), o.body_read(), tol, do[2 * K:3 * K].max(), max(w["shape"]))
    e_sum, e_abs, e_max = diag_errors(dg, do, K)
    # a sum over N cells, each within tol * max|Q_k|, can be off by tol * N * max|Q_k|; relative to sum|Q_k| that is
    # tol * N max / sum|.| (>= tol; large for a field that lives in a small part of the domain)
    N = Qo[0].size
    bound = tol * np.maximum(1.0, N * do[2 * K:3 * K] / np.maximum(do[K:2 * K], 1e-300))
    assert (e_sum <= bound).all() and (e_abs <= bound).all() and (e_max <= 10 * tol).all()
    # the reduction kernels themselves, with no oracle round-off in the way: against numpy sums of the fields this very call
    # returned (deterministic two-stage fold vs numpy's pairwise sum: ~ sqrt(N) eps sum|.|), extrema exactly
    Fg = Qg.reshape(K, -1)
    rb = 8 * np.sqrt(N) * np.finfo(np.float64).eps * np.maximum(np.abs(Fg).sum(1), 1e-300)
    assert (np.abs(dg[:K] - Fg.sum(1)) <= rb).all() and (np.abs(dg[K:2 * K] - np.abs(Fg).sum(1)) <= rb).all()
    assert (dg[2 * K:3 * K] == np.abs(Fg).max(1)).all()
    assert abs(dg[3 * K] - do[3 * K]) <= 1e3 * tol * max(do[2 * K:3 * K].max(), 1e-300)        # max|div_h B|
    if np.isfinite(do[3 * K + 1]):
        assert abs(dg[3 * K + 1] - do[3 * K + 1]) <= 10 * tol * abs(do[3 * K + 1])             # min rho
    if np.isfinite(do[3 * K + 2]):
        assert abs(dg[3 * K + 2] - do[3 * K + 2]) <= 1e3 * tol * max(do[2 * K:3 * K].max(), 1e-300)   # min p
    assert dg[3 * K + 3] == do[3 * K + 3]
    g.close()
    return errs


CASES = [
    ("IDEAL", "D1Q3", (200,), (0,) * 6),
    ("IDEAL", "D1Q3", (131,), (1, 1, 0, 0, 0, 0)),
    ("IDEAL", "D1Q3", (70,), (2, 1, 0, 0, 0, 0)),
    ("INCRES", "D1Q3", (131,), (1, 1, 0, 0, 0, 0)),
    ("IDEAL", "D2Q9", (150, 37), (0,) * 6),
    ("IDEAL", "D2Q9", (150, 37), (1, 1, 1, 1, 0, 0)),
    ("IDEAL", "D2Q9", (67, 20), (2, 1, 0, 0, 0, 0)),
    ("INCRES", "D2Q9", (150, 37), (0,) * 6),
    ("INCRES", "D2Q9", (90, 21), (1, 1, 2, 1, 0, 0)),
    ("IDEAL", "D3Q19", (100, 12, 9), (0,) * 6),
    ("IDEAL", "D3Q19", (100, 12, 9), (2, 1, 0, 0, 0, 0)),
    ("IDEAL", "D3Q19", (45, 11, 10), (1, 1, 1, 1, 1, 1)),
    ("INCRES", "D3Q19", (70, 9, 8), (1, 1, 0, 0, 2, 1)),
    ("IDEAL", "D2Q5", (150, 37), (0,) * 6),
    ("IDEAL", "D2Q5", (67, 20), (2, 1, 1, 1, 0, 0)),
    ("INCRES", "D2Q5", (90, 21), (1, 1, 0, 0, 0, 0)),
    ("IDEAL", "D3Q7", (100, 12, 9), (0,) * 6),
    ("IDEAL", "D3Q7", (100, 12, 9), (2, 1, 1, 1, 0, 0)),
    ("INCRES", "D3Q7", (45, 11, 10), (1, 1, 1, 1, 1, 1)),
]


@pytest.mark.parametrize("scheme,lattice,shape,bc", CASES)
def test_random_state_parity(scheme, lattice, shape, bc):
    """several x-tiles plus a ragged tail, every boundary kind, 20 steps from a rough random state"""
    w = random_workload(scheme, lattice, shape, bc, seed=1234)
    compare(w, 20)


@pytest.mark.parametrize("scheme,lattice,shape", [("IDEAL", "D2Q9", (90, 33)), ("IDEAL", "D3Q19", (70, 12, 10)), ("INCRES", "D2Q9", (90, 33))])
def test_masked_obstacle_parity(scheme, lattice, shape):
    rng = np.random.default_rng(77)
    w = random_workload(scheme, lattice, shape, (1, 1) + (0,) * 4, seed=99)
    s = zyx(shape)
    mask = (rng.random(s) < 0.05).astype(np.uint8) * 2
    mask[rng.random(s) < 0.02] = 1
    Bs = 0.1 * (rng.random((3,) + s) - 0.5)
    compare(w, 15, obstacle=(mask, np.array([0.03, -0.02, 0.01]), Bs))


@pytest.mark.parametrize("lattice,shape", [("D2Q9", (80, 40)), ("D3Q19", (72, 24, 20))])
def test_moving_sphere_parity(lattice, shape):
    D = len(shape)
    cen = np.array([shape[0] / 2.0, shape[1] / 2.0, shape[2] / 2.0 if D == 3 else 0.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03)
    w = random_workload("IDEAL", lattice, shape, (2, 1, 0, 0, 0, 0), seed=5, sphere=sph)
    compare(w, 12)


@pytest.mark.parametrize("name", ["C1", "C2", "C2i", "C3", "C4", "C5"])
def test_config_parity_100_steps_reduced_size(name):
    """the five BASELINE configs at the reduced sizes the oracle finishes in seconds, 100 steps"""
    w = W.get(name, small=True)
    errs = compare(w, 100)
    print(name, "max field error", errs.max())


def test_empty_step_and_odd_counts():
    w = random_workload("IDEAL", "D2Q9", (64, 16), (0,) * 6, seed=3)
    o = oracle_from_workload(w)
    g = gpu_from_workload(w)
    o.init(w["fields"])
    g.init(w["fields"])
    g.step(0)
    assert g.steps_done == 0
    for n in (1, 2, 3):
        o.step(n)
        g.step(n)
        assert (field_errors(g.moments()[0], o.moments()[0]) <= TOL64).all()
    assert g.steps_done == 6
    # populations themselves, not only their moments
    assert np.abs(g.populations() - o.populations()).max() <= 1e-13
    g.close()


def test_fp32_variant_parity():
    w = W.get("C3", small=True)
    errs = compare(w, 100, tol=TOL32, precision=32)
    print("fp32 C3 small", errs.max())


@pytest.mark.parametrize("streaming", [0, 1])
def test_fractional_porosity_parity(streaming):
    """Eq.13-16: per-cell porosity field for the masked solid and a ramp of width 1.5 cells across the moving sphere"""
    rng = np.random.default_rng(808)
    shape = (70, 12, 10)
    s = zyx(shape)
    w = random_workload("IDEAL", "D3Q19", shape, (1, 1) + (0,) * 4, seed=12)
    d = np.clip(1.6 * rng.random(s) - 0.3, 0.0, 1.0)
    us, Bs = np.array([0.03, -0.02, 0.01]), 0.1 * (rng.random((3,) + s) - 0.5)
    o = oracle_from_workload(w)
    g = gpu_from_workload(w, streaming=streaming)
    for sim in (o, g):
        sim.set_obstacle(np.zeros(s, dtype=np.uint8), us, Bs)
        sim.set_porosity(d)
        sim.init(w["fields"])
        sim.step(15)
    assert (field_errors(g.moments()[0], o.moments()[0]) <= TOL64).all()
    g.close()
    cen = np.array([36.3, 12.1, 10.2])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03, width=1.5)
    w2 = random_workload("IDEAL", "D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=13, sphere=sph)
    compare(w2, 13, streaming=streaming)
    sph["omega"] = np.array([0.02, 0.0, 0.02])        # tumbling body, dipole co-rotating
    w3 = random_workload("IDEAL", "D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=14, sphere=sph)
    compare(w3, 13, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("scheme,lattice,shape,bc", [
    ("IDEAL", "D3Q19", (200, 12, 9), (0,) * 6), ("IDEAL", "D3Q19", (200, 12, 9), (2, 1, 0, 0, 0, 0)),
    ("IDEAL", "D2Q9", (300, 37), (1, 1, 1, 1, 0, 0)), ("INCRES", "D2Q9", (300, 37), (0,) * 6),
    ("IDEAL", "D3Q7", (200, 12, 9), (2, 1, 1, 1, 0, 0)), ("IDEAL", "D1Q3", (400,), (1, 1, 0, 0, 0, 0)),
    ("IDEAL", "D2Q9", (131, 20), (0,) * 6),          # odd nx: one cell per thread
])
def test_fp32_paths_parity(scheme, lattice, shape, bc, streaming):
    """fp32: two cells per thread on interior tiles (even nx), one-cell paths elsewhere; bar 1e-5 (north_star)"""
    w = random_workload(scheme, lattice, shape, bc, seed=77)
    compare(w, 20, tol=TOL32, precision=32, streaming=streaming)
    compare(w, 7, tol=TOL32, precision=32, streaming=streaming)


def test_fp32_config5_small_with_sphere():
    compare(W.get("C5", small=True), 60, tol=TOL32, precision=32)
    compare(W.get("C5", small=True), 61, tol=TOL32, precision=32, streaming=1)


def divb_workload(lattice, shape, bc, seed, sphere=None):
    """IDEAL_DIVB (K = 9): random ideal state plus a random D field"""
    w = random_workload("IDEAL", lattice, shape, bc, seed=seed, sphere=sphere)
    rng = np.random.default_rng(seed + 1)
    w["scheme"] = "IDEAL_DIVB"
    w["tau_relax"] = 7.5
    w["fields"] = np.concatenate([w["fields"], 0.05 * (rng.random((1,) + zyx(shape)) - 0.5)])
    return w


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", [("D1Q3", (200,), (1, 1, 0, 0, 0, 0)), ("D2Q9", (150, 37), (0,) * 6),
                                              ("D3Q19", (200, 12, 9), (2, 1, 0, 0, 0, 0)), ("D3Q7", (100, 12, 9), (1, 1, 1, 1, 0, 0))])
def test_ideal_divb_scheme_parity(lattice, shape, bc, precision, tol, streaming):
    """the paper's local gradient evolution (traced): 9th set D, div B = D / tau_M in the Powell source"""
    w = divb_workload(lattice, shape, bc, seed=21)
    compare(w, 20, tol=tol, precision=precision, streaming=streaming)
    compare(w, 7, tol=tol, precision=precision, streaming=streaming)


def test_ideal_divb_with_sphere_and_mask():
    cen = np.array([36.0, 12.0, 10.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03)
    compare(divb_workload("D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=31, sphere=sph), 12)
    rng = np.random.default_rng(9)
    shape = (70, 12, 10)
    s = zyx(shape)
    mask = (rng.random(s) < 0.05).astype(np.uint8) * 2
    compare(divb_workload("D3Q19", shape, (1, 1) + (0,) * 4, seed=41), 12,
            obstacle=(mask, np.array([0.03, -0.02, 0.01]), 0.1 * (rng.random((3,) + s) - 0.5)), streaming=1)


def resist_workload(lattice, shape, bc, seed, sphere=None, eta=0.02, tau_relax=3.0):
    """RESIST (K = 8 + 3 D): random ideal state plus random gradient variables G"""
    w = random_workload("IDEAL", lattice, shape, bc, seed=seed, sphere=sphere)
    rng = np.random.default_rng(seed + 2)
    w["scheme"], w["tau_relax"], w["eta"] = "RESIST", tau_relax, eta
    w["fields"] = np.concatenate([w["fields"], 0.05 * (rng.random((3 * len(shape),) + zyx(shape)) - 0.5)])
    return w


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", [("D1Q3", (200,), (1, 1, 0, 0, 0, 0)), ("D2Q9", (150, 37), (0,) * 6),
                                              ("D2Q9", (90, 21), (1, 1, 2, 1, 0, 0)), ("D3Q19", (200, 12, 9), (2, 1, 0, 0, 0, 0)),
                                              ("D3Q19", (45, 11, 10), (1, 1, 1, 1, 1, 1)), ("D3Q7", (100, 12, 9), (1, 1, 1, 1, 0, 0)),
                                              ("D2Q5", (150, 37), (0,) * 6)])
def test_resist_scheme_parity(lattice, shape, bc, precision, tol, streaming):
    """dissipative MHD with transported gradients (Eq.9-10): K = 8 + 3 D sets, resistive fluxes from G"""
    w = resist_workload(lattice, shape, bc, seed=71)
    compare(w, 20, tol=tol, precision=precision, streaming=streaming)
    compare(w, 7, tol=tol, precision=precision, streaming=streaming)


def full_workload(lattice, shape, bc, seed, sphere=None, eta=0.02, mu=0.015, tau_relax=3.0):
    """FULL (K = 8 + 6 D): random ideal state plus random gradient variables G (of B) and H (of u)"""
    w = random_workload("IDEAL", lattice, shape, bc, seed=seed, sphere=sphere)
    rng = np.random.default_rng(seed + 3)
    w["scheme"], w["tau_relax"], w["eta"], w["nu"] = "FULL", tau_relax, eta, mu
    w["fields"] = np.concatenate([w["fields"], 0.05 * (rng.random((6 * len(shape),) + zyx(shape)) - 0.5)])
    return w


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", [("D1Q3", (200,), (1, 1, 0, 0, 0, 0)), ("D2Q9", (150, 37), (0,) * 6),
                                              ("D2Q9", (90, 21), (1, 1, 2, 1, 0, 0)), ("D3Q19", (200, 12, 9), (2, 1, 0, 0, 0, 0)),
                                              ("D3Q19", (45, 11, 10), (1, 1, 1, 1, 1, 1)), ("D3Q7", (100, 12, 9), (1, 1, 1, 1, 0, 0)),
                                              ("D2Q5", (150, 37), (0,) * 6)])
def test_full_scheme_parity(lattice, shape, bc, precision, tol, streaming):
    """full dissipative MHD (Eq.9): K = 8 + 6 D sets, resistive fluxes from G, viscous stress from H (A23)"""
    w = full_workload(lattice, shape, bc, seed=91)
    compare(w, 20, tol=tol, precision=precision, streaming=streaming)
    compare(w, 7, tol=tol, precision=precision, streaming=streaming)


@pytest.mark.parametrize("streaming", [0, 1])
def test_full_with_sphere_and_mask(streaming):
    cen = np.array([36.0, 12.0, 10.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03, width=1.5,
               omega=np.array([0.02, 0.0, 0.02]))
    compare(full_workload("D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=92, sphere=sph), 12, streaming=streaming)
    rng = np.random.default_rng(23)
    s = (9, 40)
    mask = (rng.random(s) < 0.05).astype(np.uint8) * 2
    mask[rng.random(s) < 0.02] = 1
    compare(full_workload("D2Q9", (40, 9), (0,) * 6, seed=93), 10, mask=mask,
            obstacle=(mask, np.array([0.03, -0.02, 0.0]), 0.1 * (rng.random((3,) + s) - 0.5)), streaming=streaming)


def test_full_viscous_terms_are_live():
    """mu changes the result (the H sets feed the momentum and energy fluxes), and mu = 0 reproduces RESIST on its variables"""
    w = full_workload("D2Q9", (64, 16), (0,) * 6, seed=94)
    a, b = gpu_from_workload(w), gpu_from_workload(dict(w, nu=0.0))
    r = resist_workload("D2Q9", (64, 16), (0,) * 6, seed=94)
    r["fields"] = w["fields"][:14].copy()
    c = gpu_from_workload(r)
    for g, F in ((a, w["fields"]), (b, w["fields"]), (c, r["fields"])):
        g.init(F)
        g.step(10)
    Qa, Qb, Qc = a.moments()[0], b.moments()[0], c.moments()[0]
    assert np.abs(Qa[1:5] - Qb[1:5]).max() > 1e-6
    assert np.abs(Qb[:14] - Qc).max() <= 1e-13 * np.abs(Qc).max()
    for g in (a, b, c):
        g.close()


@pytest.mark.parametrize("streaming", [0, 1])
def test_resist_with_sphere_and_mask(streaming):
    cen = np.array([36.0, 12.0, 10.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=cen, radius=6.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03, width=1.5,
               omega=np.array([0.02, 0.0, 0.02]))
    compare(resist_workload("D3Q19", (72, 24, 20), (2, 1, 0, 0, 0, 0), seed=81, sphere=sph), 12, streaming=streaming)
    rng = np.random.default_rng(19)
    shape = (70, 33)
    s = zyx(shape)
    mask = (rng.random(s) < 0.05).astype(np.uint8) * 2
    mask[rng.random(s) < 0.02] = 1
    compare(resist_workload("D2Q9", shape, (1, 1) + (0,) * 4, seed=82), 12,
            obstacle=(mask, np.array([0.03, -0.02, 0.01]), 0.1 * (rng.random((3,) + s) - 0.5)), streaming=streaming)


def test_resist_physics_on_gpu():
    """the CUDA path alone: a magnetic shear mode decays at (eta + (tau_B - 1/2) c_s^2) k^2 (the oracle's pin, re-run here)"""
    from test_oracle_pins import ideal_fields
    from paper_2606_00641_b200 import lbmhd
    nx, tauB, eta, tau_m = 128, 0.6, 0.03, 4.0
    k = 2 * np.pi / nx
    x = np.arange(nx)
    B = np.zeros((3, 1, 1, nx))
    B[1, 0, 0] = 1e-4 * np.sin(k * x)
    F8 = ideal_fields(np.ones((1, 1, nx)), np.zeros((3, 1, 1, nx)), B, 0.02 * np.ones((1, 1, nx)), 5 / 3)
    F = np.concatenate([F8, np.zeros((3, 1, 1, nx))])
    p = lbmhd.make_params("RESIST", "D1Q3", (nx,), gamma=5 / 3, tau=[0.6] * 5 + [tauB] * 3 + [0.6] * 3, powell=1.0, eta=eta,
                          tau_relax=tau_m)
    g = lbmhd.Lbmhd(p)
    g.init(F)
    g.step(200)
    a1 = 2 * (g.moments()[0][6].reshape(-1) @ np.sin(k * x)) / nx
    g.step(400)
    a2 = 2 * (g.moments()[0][6].reshape(-1) @ np.sin(k * x)) / nx
    rate = -np.log(a2 / a1) / 400
    assert abs(rate / ((eta + (tauB - 0.5) / 3.0) * k * k) - 1) < 0.02
    g.close()


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("precision,tol", [(64, TOL64), (32, TOL32)])
@pytest.mark.parametrize("lattice,shape,bc", [("D2Q9", (150, 37), (0,) * 6), ("D2Q9", (90, 21), (1, 1, 2, 1, 0, 0)),
                                              ("D3Q19", (100, 12, 9), (0,) * 6), ("D2Q5", (150, 37), (1, 1, 0, 0, 0, 0))])
def test_eta_of_j_parity(lattice, shape, bc, precision, tol, streaming):
    """INCRES with current-dependent resistivity: cell-local tau_B from the local current (A20)"""
    w = random_workload("INCRES", lattice, shape, bc, seed=51)
    w["eta_jc"] = 0.02
    w["tau"] = [0.7] + [0.6] * len(shape) + [0.55] * len(shape)
    compare(w, 20, tol=tol, precision=precision, streaming=streaming)
    # the feature is live on this data: the constant-eta run differs
    w0 = dict(w, eta_jc=0.0)
    a, b = gpu_from_workload(w), gpu_from_workload(w0)
    for sim in (a, b):
        sim.init(w["fields"])
        sim.step(5)
    assert np.abs(a.moments()[0] - b.moments()[0]).max() > 1e-7
    a.close()
    b.close()
