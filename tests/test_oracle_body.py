"""Pin P12 of the CPU oracle: body integrals (A21).

What fixes them other than the oracle's own code:
  * closed forms at the first step from a uniform state (every dQh is then one algebraic expression per cell,
    the sums over cells are brute-force enumerations of the body in numpy);
  * the conservation law: in a periodic box with kappa = 0 the only thing that changes sum_x Q_k is the blend, so
    the step-to-step difference of the oracle's own moment sums (a different code path) must equal -F, -W, +I_B;
  * the independent numpy restatement (np.cross for the torque) over several steps, moving / rotating / ramped body.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from np_vlbm import NpVLBM
from test_oracle_pins import LATS, zyx, ideal_fields, random_fields

G = 5 / 3


def uniform_state(shape, rho, u, B, p):
    s = zyx(shape)
    one = np.ones(s)
    return ideal_fields(rho * one, np.array(u).reshape(3, 1, 1, 1) * one, np.array(B).reshape(3, 1, 1, 1) * one, p * one, G)


def test_P12_closed_form_first_step_uniform_flow_masked_body():
    """sharp masked body (d = 0) at rest with field B_s in a uniform stream: per solid cell dQh_m = -rho u,
    dQh_B = B_s - B, dQh_E = -rho |u|^2 / 2 + (|B_s|^2 - |B|^2) / 2."""
    shape = (12, 10, 9)
    rho, u, B, p = 1.3, np.array([0.08, -0.05, 0.03]), np.array([0.02, 0.05, -0.04]), 0.02
    Bs = np.array([0.01, -0.03, 0.06])
    ref = np.array([4.25, 5.5, 3.75])
    rng = np.random.default_rng(3)
    s = zyx(shape)
    mask = np.where(rng.random(s) < 0.2, 2, 0).astype(np.uint8)
    o = orc.Oracle(orc.make_params(orc.IDEAL, LATS["D3Q19"], shape, gamma=G, tau=0.6, powell=1.0))
    o.set_obstacle(mask, (0, 0, 0), Bs.reshape(3, 1, 1, 1) * np.ones(s))
    o.set_body_reference(ref)
    o.init(uniform_state(shape, rho, u, B, p))
    o.step(1)
    got = o.body_read()
    zz, yy, xx = np.nonzero(mask == 2)
    n = len(xx)
    sum_r = np.array([xx.sum(), yy.sum(), zz.sum()]) - n * ref
    F = n * rho * u
    want = np.concatenate([F, np.cross(sum_r, rho * u), [n * (0.5 * rho * u @ u - 0.5 * (Bs @ Bs - B @ B))],
                           n * (Bs - B), n * B, [n]])
    assert np.abs(got - want).max() < 1e-12 * n
    # read-and-reset
    o.body_read(reset=True)
    assert np.all(o.body_read() == 0.0)


def test_P12_closed_form_first_step_moving_rotating_sphere():
    """fluid at rest, B = 0; sphere moving with u_s and spinning with Omega, no dipole (B_s = 0):
    dQh_m = rho (u_s + Omega x r), dQh_E = rho |u_s + Omega x r|^2 / 2 at the cells with |r| <= R."""
    shape = (16, 15, 14)
    rho, p = 0.9, 0.05
    c = np.array([7.3, 7.6, 6.2])
    R, us, om = 4.2, np.array([0.02, -0.01, 0.015]), np.array([0.004, -0.002, 0.003])
    o = orc.Oracle(orc.make_params(orc.IDEAL, LATS["D3Q19"], shape, gamma=G, tau=0.6, powell=1.0))
    o.set_sphere(c, R, us, (0, 0, 1), 0.0)
    o.set_sphere_rotation(om)
    o.init(uniform_state(shape, rho, (0, 0, 0), (0, 0, 0), p))
    o.step(1)
    got = o.body_read()
    zz, yy, xx = np.meshgrid(*[np.arange(n) for n in zyx(shape)], indexing="ij")
    r = np.stack([xx - c[0], yy - c[1], zz - c[2]], -1).reshape(-1, 3)
    r = r[(r * r).sum(1) <= R * R]
    v = us + np.cross(om, r)
    F = -(rho * v).sum(0)
    T = -np.cross(r, rho * v).sum(0)
    W = -(0.5 * rho * (v * v).sum(1)).sum()
    want = np.concatenate([F, T, [W], np.zeros(3), np.zeros(3), [len(r)]])
    assert np.abs(got - want).max() < 1e-13 * len(r)
    assert abs(T).max() > 1e-3          # the spin part is really there


@pytest.mark.parametrize("scheme,lat,shape", [("IDEAL", "D3Q19", (10, 9, 8)), ("IDEAL", "D2Q9", (14, 12)), ("INCRES", "D2Q9", (14, 12)),
                                              ("IDEAL", "D3Q7", (10, 9, 8))])
def test_P12_balance_against_moment_sums(scheme, lat, shape):
    """periodic, kappa = 0: sum_x Q_k(t+1) - sum_x Q_k(t) = sum_x dQh_k(t), so the moment sums (oracle_moments, another
    code path) pin F, W and I_B step by step"""
    rng = np.random.default_rng(17)
    D = len(shape)
    sc = orc.IDEAL if scheme == "IDEAL" else orc.INCRES
    o = orc.Oracle(orc.make_params(sc, LATS[lat], shape, gamma=G, tau=0.7, powell=0.0))
    F0 = random_fields(rng, scheme, lat, shape, gamma=G)
    c = np.array([s / 2 + 0.3 for s in shape] + [0.0] * (3 - D))
    o.set_sphere(c, 2.6, (0.01, -0.02, 0.0), (0.3, 0.5, 0.8), 0.02)
    o.set_sphere_width(1.5)
    o.init(F0)
    K = o.K
    iB = 5 if scheme == "IDEAL" else 1 + D
    nvec = 3 if scheme == "IDEAL" else D
    for _ in range(6):
        _, d0 = o.moments()
        o.body_read(reset=True)
        o.step(1)
        _, d1 = o.moments()
        b = o.body_read()
        dS = d1[:K] - d0[:K]
        scale = d0[K:2 * K].max()
        assert np.abs(dS[1:1 + nvec] + b[0:nvec]).max() < 1e-12 * scale
        assert np.abs(dS[iB:iB + nvec] - b[7:7 + nvec]).max() < 1e-12 * scale
        if scheme == "IDEAL":
            assert abs(dS[4] + b[6]) < 1e-12 * scale
            assert abs(dS[0]) < 1e-12 * scale                 # the blend keeps rho
        assert np.abs(b[0:nvec]).max() > 1e-6                 # not trivially zero


@pytest.mark.parametrize("scheme,lat,shape,bc", [
    ("IDEAL", "D3Q19", (9, 8, 7), (0,) * 6), ("IDEAL", "D2Q9", (13, 11), (2, 1, 0, 0, 0, 0)), ("INCRES", "D3Q19", (9, 8, 7), (0,) * 6),
    ("IDEAL_DIVB", "D2Q9", (13, 11), (0,) * 6)])
def test_P12_numpy_restatement(scheme, lat, shape, bc):
    rng = np.random.default_rng(23)
    D = len(shape)
    sc = {"IDEAL": orc.IDEAL, "INCRES": orc.INCRES, "IDEAL_DIVB": orc.IDEAL_DIVB}[scheme]
    base = "IDEAL" if scheme != "INCRES" else "INCRES"
    F0 = random_fields(rng, base, lat, shape, gamma=G)
    if scheme == "IDEAL_DIVB":
        F0 = np.concatenate([F0, 1e-3 * rng.standard_normal((1,) + F0.shape[1:])])
    kw = dict(tau_relax=5.0) if scheme == "IDEAL_DIVB" else {}
    o = orc.Oracle(orc.make_params(sc, LATS[lat], shape, gamma=G, tau=0.7, powell=1.0, bc=bc, **kw))
    m = NpVLBM(scheme, lat, zyx(shape), 0.7, gamma=G, powell=1.0, bc=bc, **kw)
    s = zyx(shape)
    c = np.array([sh / 2 - 0.4 for sh in shape] + [0.0] * (3 - D))
    us, mh, om = np.array([0.015, -0.01, 0.02 if D == 3 else 0.0]), np.array([0.6, 0.0, 0.8]), np.array([0.0, 0.0, 0.01])
    if D == 3:
        om = np.array([0.004, 0.006, -0.008])
    # a masked body with porosity next to the sphere
    mask = np.zeros(s, dtype=np.uint8)
    mask[..., 1:3] = 2
    dfield = np.ones(s)
    dfield[..., 1:3] = rng.random(s)[..., 1:3]
    Bsol = 0.02 * rng.standard_normal((3,) + s)
    for side in (o, m):
        if side is o:
            side.set_obstacle(mask, (0.01, 0.0, -0.01), Bsol)
            side.set_porosity(dfield)
            side.set_sphere(c, 2.4, us, mh, 0.03)
            side.set_sphere_width(1.0)
            side.set_sphere_rotation(om)
        else:
            side.mask, side.u_solid, side.B_solid, side.d_field = mask, np.array([0.01, 0.0, -0.01]), Bsol, dfield
            side.sphere = (c, 2.4, us, mh, 0.03, 0)
            side.sphere_eps, side.sphere_omega = 1.0, om
        side.init(F0)
        side.step(5)
    got, want = o.body_read(), m.body
    assert np.abs(got - want).max() < 1e-12 * max(1.0, np.abs(want).max())
    assert np.abs(want[3:6]).max() > 0


# ---------------------------------------------------------------- dipole ensemble, rotating masked bodies
def dipole_field(x, centre, R, offsets, axes, strengths, cores):
    """sum_j 1/2 Bs_j (R / max(|r_j|, core_j))^3 [3 (m_j.r^_j) r^_j - m_j] written with scipy-free plain numpy on point lists"""
    B = np.zeros_like(x)
    for off, m, bs, core in zip(offsets, axes, strengths, cores):
        rj = x - centre - off
        rn = np.linalg.norm(rj, axis=1)
        rh = rj / rn[:, None]
        B += (0.5 * bs * (R / np.maximum(rn, core)) ** 3)[:, None] * (3.0 * (rh @ m)[:, None] * rh - m)
    return B


def rotation_matrix(omega, angle_steps):
    """matrix exponential of the cross-product matrix: an independent route to the Rodrigues rotation"""
    from scipy.linalg import expm
    wx = np.array([[0, -omega[2], omega[1]], [omega[2], 0, -omega[0]], [-omega[1], omega[0], 0]])
    return expm(wx * angle_steps)


def test_P12_dipole_ensemble_imposed_field():
    """sharp sphere, d = 0: after a step the stored B at the body cells is B^B of that step; four shifted capped dipoles
    co-rotating with the body (axes and offsets rotated by exp([Omega]x t))"""
    shape = (20, 18, 16)
    c, R = np.array([9.3, 8.6, 7.7]), 5.2
    offs = np.array([[1.5, 0.0, 0.5], [-1.0, 2.0, 0.0], [0.0, -1.5, -2.0], [0.5, 0.5, 2.5]])
    axes = np.array([[0.0, 0.0, 1.0], [0.6, 0.0, 0.8], [1.0, 0.0, 0.0], [0.0, -0.8, 0.6]])
    bs, cores = np.array([0.03, -0.02, 0.015, 0.025]), np.array([1.5, 2.0, 1.0, 2.5])
    om = np.array([0.03, -0.02, 0.05])
    o = orc.Oracle(orc.make_params(orc.IDEAL, LATS["D3Q19"], shape, gamma=G, tau=0.6, powell=1.0))
    o.set_sphere(c, R, (0, 0, 0), (0, 0, 1), 0.0)
    o.set_sphere_rotation(om)
    o.set_sphere_dipoles(offs, axes, bs, cores)
    o.init(uniform_state(shape, 1.0, (0, 0, 0), (0.01, 0.0, 0.0), 0.05))
    zz, yy, xx = np.meshgrid(*[np.arange(n) for n in zyx(shape)], indexing="ij")
    pts = np.stack([xx, yy, zz], -1).reshape(-1, 3).astype(float)
    inside = ((pts - c) ** 2).sum(1) <= R * R
    for t in range(4):
        o.step(1)                                   # step t uses the body at angle |Omega| t
        Rm = rotation_matrix(om, t)
        want = dipole_field(pts[inside], c, R, offs @ Rm.T, axes @ Rm.T, bs, cores)
        Q, _ = o.moments()
        got = np.stack([Q[5 + b].reshape(-1)[inside] for b in range(3)], 1)
        assert np.abs(got - want).max() < 1e-13
    assert np.abs(want).max() > 0.01


def test_P12_single_dipole_is_the_ensemble_of_one():
    shape = (16, 14, 12)
    rng = np.random.default_rng(4)
    F0 = random_fields(rng, "IDEAL", "D3Q19", shape, gamma=G)
    c, R, mh = np.array([7.4, 6.6, 5.9]), 4.0, np.array([0.3, -0.5, 0.8])
    out = []
    for ens in (False, True):
        o = orc.Oracle(orc.make_params(orc.IDEAL, LATS["D3Q19"], shape, gamma=G, tau=0.7, powell=1.0))
        o.set_sphere(c, R, (0.01, 0, 0), mh, 0.03)
        o.set_sphere_rotation((0.0, 0.02, 0.01))
        if ens:
            o.set_sphere_dipoles(np.zeros((1, 3)), mh.reshape(1, 3), [0.03], [0.5 * R])
        o.init(F0)
        o.step(5)
        out.append(o.populations())
    assert np.array_equal(out[0], out[1])


def test_P12_rotating_masked_body_closed_form_and_numpy():
    """masked body spinning about a point in fluid at rest: first-step integrals in closed form; then the numpy
    restatement over several steps with the ensemble on a sphere beside it"""
    shape = (14, 12, 10)
    s = zyx(shape)
    rho, p = 1.1, 0.04
    mask = np.zeros(s, dtype=np.uint8)
    mask[2:7, 3:9, 4:10] = 2
    us, om, cen = np.array([0.01, 0.0, -0.02]), np.array([0.003, 0.004, -0.002]), np.array([6.5, 5.5, 4.0])
    o = orc.Oracle(orc.make_params(orc.IDEAL, LATS["D3Q19"], shape, gamma=G, tau=0.6, powell=1.0))
    o.set_obstacle(mask, us, None)
    o.set_obstacle_rotation(om, cen)
    o.set_body_reference(cen)
    o.init(uniform_state(shape, rho, (0, 0, 0), (0, 0, 0), p))
    o.step(1)
    got = o.body_read()
    zz, yy, xx = np.nonzero(mask == 2)
    r = np.stack([xx, yy, zz], 1) - cen
    v = us + np.cross(om, r)
    want = np.concatenate([-(rho * v).sum(0), -np.cross(r, rho * v).sum(0), [-(0.5 * rho * (v * v).sum(1)).sum()], np.zeros(6), [len(r)]])
    assert np.abs(got - want).max() < 1e-13 * len(r)
    # several steps against numpy, rough state, ensemble sphere + rotating masked body
    rng = np.random.default_rng(29)
    F0 = random_fields(rng, "IDEAL", "D3Q19", shape, gamma=G)
    offs, axes = np.array([[0.8, 0.0, 0.3], [-0.5, 0.6, 0.0]]), np.array([[0.0, 0.6, 0.8], [1.0, 0.0, 0.0]])
    bs, cores = np.array([0.02, -0.03]), np.array([0.8, 1.2])
    c2, som = np.array([10.2, 4.1, 3.3]), np.array([0.01, 0.02, -0.015])
    o = orc.Oracle(orc.make_params(orc.IDEAL, LATS["D3Q19"], shape, gamma=G, tau=0.7, powell=1.0))
    m = NpVLBM("IDEAL", "D3Q19", s, 0.7, gamma=G, powell=1.0)
    o.set_obstacle(mask, us, None)
    o.set_obstacle_rotation(om, cen)
    o.set_sphere(c2, 2.2, (0.0, 0.01, 0.0), (0, 0, 1), 0.0)
    o.set_sphere_rotation(som)
    o.set_sphere_dipoles(offs, axes, bs, cores)
    m.mask, m.u_solid, m.obst_omega, m.obst_centre = mask, us, om, cen
    m.sphere, m.sphere_omega = (c2, 2.2, np.array([0.0, 0.01, 0.0]), np.array([0.0, 0.0, 1.0]), 0.0, 0), som
    m.dipoles = list(zip(offs, axes, bs, cores))
    for side in (o, m):
        side.init(F0)
        side.step(4)
    Q, _ = o.moments()
    assert np.abs(Q - m.moments()).max() < 1e-13
    assert np.abs(o.body_read() - m.body).max() < 1e-12
