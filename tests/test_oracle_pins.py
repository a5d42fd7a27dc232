"""Pins P1-P4, P6 of the CPU oracle: what the paper and the mathematics fix.

Nothing here calls the CUDA path.  Expected values are closed forms, invariants, hand-evaluated
states, or the independent numpy restatement in tests/np_vlbm.py.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from np_vlbm import NpVLBM, lattice_np, flux_ideal

LATS = {"D1Q3": orc.D1Q3, "D2Q9": orc.D2Q9, "D3Q19": orc.D3Q19, "D2Q5": orc.D2Q5, "D3Q7": orc.D3Q7}
SHAPES = {"D1Q3": (6,), "D2Q9": (5, 4), "D3Q19": (5, 4, 3), "D2Q5": (5, 4), "D3Q7": (5, 4, 3)}


def admissible_ideal(rng, shape_zyx, amp=0.2):
    """random subsonic-on-the-lattice ideal-MHD state, [8, z, y, x]"""
    rho = 1.0 + 0.3 * rng.random(shape_zyx)
    u = amp * (rng.random((3,) + shape_zyx) - 0.5)
    B = amp * (rng.random((3,) + shape_zyx) - 0.5)
    p = 0.02 + 0.01 * rng.random(shape_zyx)
    return rho, u, B, p


def ideal_fields(rho, u, B, p, gamma):
    E = p / (gamma - 1) + 0.5 * rho * (u * u).sum(0) + 0.5 * (B * B).sum(0)
    return np.concatenate([rho[None], rho[None] * u, E[None], B])


def incres_fields(rng, D, shape_zyx, amp=0.05):
    P = 0.01 * (rng.random(shape_zyx) - 0.5)
    u = amp * (rng.random((D,) + shape_zyx) - 0.5)
    B = amp * (rng.random((D,) + shape_zyx) - 0.5)
    return np.concatenate([P[None], u, B])


def zyx(shape_xyz):
    s = list(shape_xyz) + [1] * (3 - len(shape_xyz))
    return (s[2], s[1], s[0])


# ---------------------------------------------------------------- lattice identities (A2)
@pytest.mark.parametrize("lat", list(LATS))
def test_lattice_identities(lat):
    D, Q, c, w, cs2 = orc.lattice(LATS[lat])
    Dn, cn, wn, cs2n = lattice_np(lat)
    assert D == Dn and Q == len(wn)
    assert np.array_equal(c, cn)                 # direction order of reading A2
    assert np.allclose(w, wn, rtol=0, atol=1e-17)
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs((w[:, None] * c).sum(0)).max() < 1e-16
    M2 = np.einsum("i,ia,ib->ab", w, c, c)
    assert np.allclose(M2[:D, :D], cs2 * np.eye(D), atol=1e-16)
    M3 = np.einsum("i,ia,ib,ic->abc", w, c, c, c)
    assert np.abs(M3).max() < 1e-16
    # opposite pairs are consecutive: opp(2j-1) = 2j
    for i in range(1, Q, 2):
        assert np.array_equal(c[i], -c[i + 1])
    expected_cs2 = 0.25 if lat == "D3Q7" else 1.0 / 3.0
    assert abs(cs2 - expected_cs2) < 1e-16


# ---------------------------------------------------------------- flux: hand-evaluated states (Eq.8, Eq.11)
def test_flux_hand_values():
    p = orc.make_params(orc.IDEAL, orc.D3Q19, (4, 4, 4), gamma=1.4)
    # rho=1, u=(1,0,0), p=1, B=0: E = 1/0.4 + 1/2 = 3
    Phi = orc.flux(p, [1, 1, 0, 0, 3.0, 0, 0, 0])
    assert np.allclose(Phi[0], [1, 0, 0], atol=1e-15)
    assert np.allclose(Phi[1], [2, 0, 0], atol=1e-15)      # rho u u + p
    assert np.allclose(Phi[2], [0, 1, 0], atol=1e-15)      # p on the diagonal
    assert np.allclose(Phi[3], [0, 0, 1], atol=1e-15)
    assert np.allclose(Phi[4], [4, 0, 0], atol=1e-15)      # (E + p) u
    assert np.abs(Phi[5:]).max() == 0
    # rho=1, u=0, p=1, B=(1,2,3): |B|^2/2 = 7, E = 2.5 + 7, p_tot = 8
    Phi = orc.flux(p, [1, 0, 0, 0, 9.5, 1, 2, 3])
    assert np.allclose(Phi[1], [8 - 1, -2, -3], atol=1e-14)
    assert np.allclose(Phi[2], [-2, 8 - 4, -6], atol=1e-14)
    assert np.allclose(Phi[3], [-3, -6, 8 - 9], atol=1e-14)
    assert np.abs(Phi[4]).max() < 1e-15 and np.abs(Phi[5:]).max() < 1e-15
    # induction: u=(0,1,0), B=(1,0,0): Phi_{Bx},y = u_y B_x = 1, Phi_{By},x = -B_x u_y = -1
    E = 2.5 + 0.5 + 0.5
    Phi = orc.flux(p, [1, 0, 1, 0, E, 1, 0, 0])
    assert np.allclose(Phi[5], [0, 1, 0], atol=1e-15)
    assert np.allclose(Phi[6], [-1, 0, 0], atol=1e-15)
    assert np.allclose(Phi[7], [0, 0, 0], atol=1e-15)
    # energy flux with u.B != 0: u=(1,0,0), B=(1,1,0): uB=1, B2=2, E=2.5+.5+1=4, pt=2
    Phi = orc.flux(p, [1, 1, 0, 0, 4.0, 1, 1, 0])
    assert np.allclose(Phi[4], [(4 + 2) * 1 - 1 * 1, -1 * 1, 0], atol=1e-14)


def test_flux_rotation_and_galilean():
    """Eq.11 is a tensor equation: rotating the state by 90 degrees about z rotates the flux."""
    rng = np.random.default_rng(7)
    p = orc.make_params(orc.IDEAL, orc.D3Q19, (4, 4, 4), gamma=5 / 3)
    R = np.array([[0, -1, 0], [1, 0, 0], [0, 0, 1]], dtype=float)
    for _ in range(5):
        rho, u, B, pr = [a.reshape(a.shape[:-3]) for a in admissible_ideal(rng, (1, 1, 1), amp=1.0)]
        Qv = ideal_fields(rho.reshape(()), u.reshape(3), B.reshape(3), pr.reshape(()), 5 / 3).reshape(8)
        Qr = Qv.copy()
        Qr[1:4] = R @ Qv[1:4]
        Qr[5:8] = R @ Qv[5:8]
        F, Fr = orc.flux(p, Qv), orc.flux(p, Qr)
        assert np.allclose(Fr[0], R @ F[0], atol=1e-14)
        assert np.allclose(Fr[4], R @ F[4], atol=1e-14)
        assert np.allclose(Fr[1:4], R @ F[1:4] @ R.T, atol=1e-14)
        assert np.allclose(Fr[5:8], R @ F[5:8] @ R.T, atol=1e-14)
        # induction flux is antisymmetric, so its trace vanishes (used by reading A6)
        assert np.allclose(F[5:8], -F[5:8].T, atol=1e-15)
        # independent tensor-form writing
        Fn = flux_ideal(Qv.reshape(8, 1), 5 / 3, 3)[:, :, 0]
        assert np.allclose(F, Fn, rtol=1e-14, atol=1e-15)


# ---------------------------------------------------------------- P1 equilibrium moments (Eq.3-4)
@pytest.mark.parametrize("lat", list(LATS))
@pytest.mark.parametrize("scheme", ["IDEAL", "INCRES"])
def test_P1_equilibrium_moments(lat, scheme):
    rng = np.random.default_rng(11)
    D, Q, c, w, cs2 = orc.lattice(LATS[lat])
    p = orc.make_params(orc.IDEAL if scheme == "IDEAL" else orc.INCRES, LATS[lat], SHAPES[lat], gamma=1.4, c0sq=0.1)
    for _ in range(20):
        if scheme == "IDEAL":
            rho, u, B, pr = admissible_ideal(rng, (1, 1, 1), amp=1.0)
            Qv = ideal_fields(rho, u, B, pr, 1.4).reshape(8)
        else:
            Qv = incres_fields(rng, D, (1, 1, 1), amp=1.0).reshape(-1)
        feq = orc.equilibrium(p, Qv)
        Phi = orc.flux(p, Qv)
        scale = np.abs(Qv).max() + np.abs(Phi).max()
        assert np.abs(feq.sum(1) - Qv).max() <= 2e-15 * scale            # zeroth moment = Q_k
        first = feq @ c.astype(float)                                    # [K, 3]
        assert np.abs(first - Phi).max() <= 2e-15 * scale                # first moment = Phi_k exactly
        assert D == 3 or np.abs(Phi[:, D:]).max() == 0


# ---------------------------------------------------------------- helpers to drive both writings
def make_pair(scheme, lat, shape_xyz, tau, gamma=5 / 3, c0sq=1 / 12, powell=1.0, bc=(0,) * 6, mask=None):
    p = orc.make_params(orc.IDEAL if scheme == "IDEAL" else orc.INCRES, LATS[lat], shape_xyz, gamma=gamma,
                        c0sq=c0sq, tau=tau, powell=powell, bc=bc)
    o = orc.Oracle(p, mask=mask)
    n = NpVLBM(scheme, lat, zyx(shape_xyz), tau, gamma=gamma, c0sq=c0sq, powell=powell, bc=bc, mask=mask)
    return o, n


def random_fields(rng, scheme, lat, shape_xyz, gamma=5 / 3):
    D = lattice_np(lat)[0]
    s = zyx(shape_xyz)
    if scheme == "IDEAL":
        rho, u, B, p = admissible_ideal(rng, s)
        return ideal_fields(rho, u, B, p, gamma)
    return incres_fields(rng, D, s)


# ---------------------------------------------------------------- P6 brute force: two writings agree
@pytest.mark.parametrize("lat", list(LATS))
@pytest.mark.parametrize("scheme", ["IDEAL", "INCRES"])
def test_P6_numpy_bruteforce_periodic(lat, scheme):
    rng = np.random.default_rng(101)
    D = lattice_np(lat)[0]
    K = 8 if scheme == "IDEAL" else 1 + 2 * D
    tau = 0.5 + 0.5 * rng.random(K)
    tau[(5 if scheme == "IDEAL" else 1 + D):] = 0.77          # A7: one tau for the B sets
    o, n = make_pair(scheme, lat, SHAPES[lat], tau, powell=1.0)
    F = random_fields(rng, scheme, lat, SHAPES[lat])
    o.init(F)
    n.init(F)
    assert np.abs(o.populations() - n.g).max() < 1e-15
    for s in range(5):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-14, s
    Qo = o.moments(diag=False)
    assert np.abs(Qo - n.moments()).max() < 1e-14
    assert np.abs(o.source_log() - n.src_acc).max() < 1e-13
    # the Powell source was live in this test (random B is not solenoidal)
    if D > 1:
        assert np.abs(n.src_acc).max() > 1e-6


@pytest.mark.parametrize("lat,bc", [
    ("D1Q3", (1, 1, 0, 0, 0, 0)),
    ("D2Q9", (1, 1, 1, 1, 0, 0)),
    ("D2Q9", (2, 1, 0, 0, 0, 0)),
    ("D2Q5", (1, 1, 1, 1, 0, 0)),
    ("D3Q19", (2, 1, 0, 0, 0, 0)),
    ("D3Q19", (1, 1, 1, 1, 1, 1)),
    ("D3Q7", (2, 1, 1, 1, 0, 0)),
])
@pytest.mark.parametrize("scheme", ["IDEAL", "INCRES"])
def test_P6_numpy_bruteforce_boundaries_and_solids(lat, bc, scheme):
    """ZEROGRAD / INFLOW faces (A9, A10), FROZEN and SOLID mask cells (A8, A11) against the array writing."""
    rng = np.random.default_rng(202)
    shape = {"D1Q3": (9,), "D2Q9": (6, 5), "D2Q5": (6, 5), "D3Q19": (6, 5, 4), "D3Q7": (6, 5, 4)}[lat]
    s = zyx(shape)
    mask = np.zeros(s, dtype=np.uint8)
    flat = mask.reshape(-1)
    pick = rng.choice(flat.size, size=3, replace=False)
    flat[pick[0]] = 2
    flat[pick[1]] = 2
    flat[pick[2]] = 1
    o, n = make_pair(scheme, lat, shape, 0.8, bc=bc, mask=mask)
    us = np.array([0.03, -0.02, 0.01])
    Bs = 0.1 * (rng.random((3,) + s) - 0.5)
    o.set_obstacle(mask, us, Bs)
    n.u_solid, n.B_solid = us, Bs
    F = random_fields(rng, scheme, lat, shape)
    o.init(F)
    n.init(F)
    for st in range(6):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-14, st


@pytest.mark.parametrize("lat", ["D2Q9", "D3Q19"])
def test_P6_numpy_bruteforce_moving_sphere(lat):
    """analytic moving sphere + capped dipole (A12) against the array writing, incl. a cell at r = 0"""
    rng = np.random.default_rng(303)
    shape = (12, 10) if lat == "D2Q9" else (12, 10, 9)
    bc = (2, 1, 0, 0, 0, 0)
    o, n = make_pair("IDEAL", lat, shape, 0.7, bc=bc)
    cen = np.array([6.0, 5.0, 4.0 if lat == "D3Q19" else 0.0])
    us = np.array([-0.25, 0.0, 0.0])          # reaches the integer centre (5,5,4) after 4 steps -> r = 0 cell
    mh = np.array([0.3, -0.5, 0.8])
    mh /= np.linalg.norm(mh)
    o.set_sphere(cen, 3.0, us, mh, 0.03)
    n.sphere = (cen, 3.0, us, mh, 0.03, 0)
    F = random_fields(rng, "IDEAL", lat, shape)
    o.init(F)
    n.init(F)
    for st in range(6):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-14, st
    # solid cells carry exactly rho u^B and B^B after the collision (P9)
    Q = o.moments(diag=False)
    d, uB, BB = n._solid.__func__(_at(n, n.t - 1))
    sol = d < 1
    assert sol.sum() > 10
    for b in range(3):
        assert np.abs(Q[1 + b][sol] - Q[0][sol] * uB[b][sol]).max() < 1e-15
        assert np.abs(Q[5 + b][sol] - BB[b][sol]).max() < 1e-15


class _at:
    """view of an NpVLBM with its step counter set back (solid state used by the LAST step)"""
    def __init__(self, n, t):
        self.__dict__.update(n.__dict__)
        self.t = t


# ---------------------------------------------------------------- fractional porosity (Eq.13-16, NEXT-3)
@pytest.mark.parametrize("lat,scheme", [("D2Q9", "IDEAL"), ("D3Q19", "IDEAL"), ("D2Q9", "INCRES"), ("D3Q7", "IDEAL")])
def test_P6_numpy_bruteforce_fractional_porosity(lat, scheme):
    rng = np.random.default_rng(404)
    shape = (7, 6) if lattice_np(lat)[0] == 2 else (7, 6, 5)
    s = zyx(shape)
    o, n = make_pair(scheme, lat, shape, 0.8, bc=(1, 1) + (0,) * 4)
    d = np.clip(1.6 * rng.random(s) - 0.3, 0.0, 1.0)          # zeros, ones and everything between
    us = np.array([0.03, -0.02, 0.01])
    Bs = 0.1 * (rng.random((3,) + s) - 0.5)
    o.set_obstacle(np.zeros(s, dtype=np.uint8), us, Bs)
    o.set_porosity(d)
    n.u_solid, n.B_solid, n.d_field = us, Bs, d
    F = random_fields(rng, scheme, lat, shape)
    if lat == "D3Q7":
        F[1:4] *= 0.3
        F[5:8] *= 0.3
    o.init(F)
    n.init(F)
    for st in range(6):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-14, st
    assert np.abs(o.source_log() - n.src_acc).max() < 1e-13


def test_P6_numpy_bruteforce_smooth_sphere():
    rng = np.random.default_rng(505)
    shape = (14, 12, 10)
    o, n = make_pair("IDEAL", "D3Q19", shape, 0.7, bc=(2, 1, 0, 0, 0, 0))
    cen, us = np.array([7.3, 6.1, 5.2]), np.array([-0.2, 0.05, 0.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    o.set_sphere(cen, 3.0, us, mh, 0.03)
    o.set_sphere_width(1.5)
    n.sphere, n.sphere_eps = (cen, 3.0, us, mh, 0.03, 0), 1.5
    F = random_fields(rng, "IDEAL", "D3Q19", shape)
    o.init(F)
    n.init(F)
    for st in range(6):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-14, st
    d, _, _ = n._solid()
    assert ((d > 0) & (d < 1)).sum() > 20 and (d == 0).sum() > 20      # the ramp and the core were both exercised


def test_porosity_limits_and_half_cell():
    """d = 1 everywhere is the fluid run bit for bit; d in {0,1} equals the mask; a d = 1/2 cell in a state at rest takes
    exactly half the solid velocity and the mean of the fields (Eq.13-14)."""
    rng = np.random.default_rng(606)
    shape = (8, 7, 6)
    s = zyx(shape)
    F = random_fields(rng, "IDEAL", "D3Q19", shape)
    par = orc.make_params(orc.IDEAL, orc.D3Q19, shape, gamma=5 / 3, tau=0.7, powell=1.0)
    a, b, c = orc.Oracle(par), orc.Oracle(par), orc.Oracle(par)
    us, Bs = np.array([0.02, -0.01, 0.03]), 0.1 * (rng.random((3,) + s) - 0.5)
    mask = (rng.random(s) < 0.1).astype(np.uint8) * 2
    b.set_obstacle(np.zeros(s, dtype=np.uint8), us, Bs)
    b.set_porosity(np.ones(s))
    for o in (a, b):
        o.init(F)
        o.step(4)
    assert np.array_equal(a.populations(), b.populations())
    b.set_obstacle(mask, us, Bs)
    b.set_porosity(None)
    c.set_obstacle(np.zeros(s, dtype=np.uint8), us, Bs)
    c.set_porosity(np.where(mask == 2, 0.0, 1.0))
    b.init(F)
    c.init(F)
    b.step(4)
    c.step(4)
    assert np.array_equal(b.populations(), c.populations())
    # half cell
    B0 = np.array([0.05, -0.02, 0.03])
    one = np.ones(s)
    Fu = ideal_fields(1.3 * one, np.zeros((3,) + s), B0.reshape(3, 1, 1, 1) * one, 0.03 * one, 5 / 3)
    d = np.ones(s)
    d[2, 3, 4] = 0.5
    h = orc.Oracle(par)
    h.set_obstacle(np.zeros(s, dtype=np.uint8), us, np.zeros((3,) + s))
    h.set_porosity(d)
    h.init(Fu)
    h.step(1)
    Q = h.moments(diag=False)
    assert np.allclose(Q[1:4, 2, 3, 4], 1.3 * 0.5 * us, rtol=0, atol=1e-16)
    assert np.allclose(Q[5:8, 2, 3, 4], 0.5 * B0, rtol=0, atol=1e-16)
    assert abs(Q[0, 2, 3, 4] - 1.3) < 1e-15


def test_P6_numpy_bruteforce_rotating_smooth_sphere():
    """rigid rotation: u^B = u_s + Omega x r, dipole axis co-rotating; against the array writing"""
    rng = np.random.default_rng(707)
    shape = (14, 12, 10)
    o, n = make_pair("IDEAL", "D3Q19", shape, 0.7, bc=(2, 1, 0, 0, 0, 0))
    cen, us = np.array([7.3, 6.1, 5.2]), np.array([-0.2, 0.05, 0.0])
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    om = np.array([0.02, 0.0, 0.02])
    o.set_sphere(cen, 3.0, us, mh, 0.03)
    o.set_sphere_width(1.0)
    o.set_sphere_rotation(om)
    n.sphere, n.sphere_eps, n.sphere_omega = (cen, 3.0, us, mh, 0.03, 0), 1.0, om
    F = random_fields(rng, "IDEAL", "D3Q19", shape)
    o.init(F)
    n.init(F)
    for st in range(6):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-14, st
    # a fully solid cell moves with u_s + Omega x r exactly (post-collision momentum = rho u^B)
    Q = o.moments(diag=False)
    d, uB, BB = n._solid.__func__(_at(n, n.t - 1))
    core = d == 0
    assert core.sum() > 10 and np.abs(uB[:, core] - us.reshape(3, 1)).max() > 1e-3
    for b in range(3):
        assert np.abs(Q[1 + b][core] - Q[0][core] * uB[b][core]).max() < 1e-15
