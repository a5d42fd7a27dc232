"""Pins P2, P3, P4, P7, P9, P10 of the CPU oracle: invariants and symmetries."""
import numpy as np
import pytest

from oracle import oracle as orc
from np_vlbm import lattice_np
from test_oracle_pins import LATS, zyx, admissible_ideal, ideal_fields, incres_fields, random_fields

G = 5 / 3


def uniform_ideal(shape_xyz, rho=1.3, u=(0.11, -0.07, 0.05), B=(0.09, 0.13, -0.04), p=0.03, gamma=G):
    s = zyx(shape_xyz)
    one = np.ones(s)
    uu = np.array(u).reshape(3, 1, 1, 1) * one
    BB = np.array(B).reshape(3, 1, 1, 1) * one
    return ideal_fields(rho * one, uu, BB, p * one, gamma)


# ---------------------------------------------------------------- P2 uniform state invariant
@pytest.mark.parametrize("lat,shape,bc", [
    ("D1Q3", (16,), (0,) * 6), ("D1Q3", (16,), (1, 1, 0, 0, 0, 0)), ("D1Q3", (16,), (2, 1, 0, 0, 0, 0)),
    ("D2Q9", (8, 7), (0,) * 6), ("D2Q9", (8, 7), (1, 1, 1, 1, 0, 0)), ("D2Q9", (8, 7), (2, 1, 0, 0, 0, 0)),
    ("D3Q19", (6, 5, 4), (0,) * 6), ("D3Q19", (6, 5, 4), (2, 1, 0, 0, 0, 0)), ("D3Q19", (6, 5, 4), (1, 1, 1, 1, 1, 1)),
    ("D2Q5", (8, 7), (1, 1, 0, 0, 0, 0)), ("D3Q7", (6, 5, 4), (2, 1, 1, 1, 0, 0)),
])
@pytest.mark.parametrize("scheme", ["IDEAL", "INCRES"])
def test_P2_uniform_invariant(lat, shape, bc, scheme):
    D = lattice_np(lat)[0]
    slow = lat in ("D2Q5", "D3Q7")      # axis-only lattices need |u| + c_f well below w_1-limited speeds
    if scheme == "IDEAL":
        F = uniform_ideal(shape, u=(0.03, -0.02, 0.015), B=(0.03, 0.04, -0.01), p=0.003) if slow else uniform_ideal(shape)
        p = orc.make_params(orc.IDEAL, LATS[lat], shape, gamma=G, tau=0.51, powell=1.0, bc=bc)
    else:
        s = zyx(shape)
        vals = [0.01] + [0.05, -0.03, 0.02][:D] + [0.04, 0.02, -0.05][:D]
        F = np.array(vals).reshape(-1, 1, 1, 1) * np.ones(s)
        p = orc.make_params(orc.INCRES, LATS[lat], shape, tau=0.51, powell=1.0, bc=bc)
    o = orc.Oracle(p)
    o.init(F)
    o.step(100)
    Q, dg = o.moments()
    scale = np.abs(F).reshape(F.shape[0], -1).max(1).reshape(-1, 1, 1, 1)
    scale = np.where(scale > 0, scale, 1.0)
    assert (np.abs(Q - F) / scale).max() < 1e-12      # round-off random walk over 100 steps; any wrong term is O(1e-3)
    assert dg[3 * o.K] < 1e-15          # div_h B of a uniform field
    assert dg[3 * o.K + 3] == 0


# ---------------------------------------------------------------- P3 conservation
@pytest.mark.parametrize("lat,shape", [("D1Q3", (32,)), ("D2Q9", (12, 10)), ("D3Q19", (8, 6, 5)), ("D2Q5", (12, 10)), ("D3Q7", (8, 6, 5))])
@pytest.mark.parametrize("scheme", ["IDEAL", "INCRES"])
@pytest.mark.parametrize("kappa", [0.0, 1.0])
def test_P3_conservation_periodic(lat, shape, scheme, kappa):
    rng = np.random.default_rng(5)
    p = orc.make_params(orc.IDEAL if scheme == "IDEAL" else orc.INCRES, LATS[lat], shape, gamma=G, tau=0.7, powell=kappa)
    o = orc.Oracle(p)
    F = random_fields(rng, scheme, lat, shape, gamma=G)
    o.init(F)
    _, d0 = o.moments()
    o.step(40)
    _, d1 = o.moments()
    K = o.K
    drift = d1[:K] - d0[:K]
    tol = 1e-13 * np.maximum(d0[K:2 * K], 1.0)
    if kappa == 0.0:
        assert (np.abs(drift) <= tol).all()                 # mass, momentum, energy, magnetic flux
        assert np.abs(o.source_log()).max() == 0
    else:
        assert abs(drift[0]) <= tol[0]                      # first variable never gets a source
        # Powell's source is non-conservative by construction: the drift IS the injected source
        assert (np.abs(drift - o.source_log()) <= tol).all()
        if lattice_np(lat)[0] > 1:
            assert np.abs(drift[1:]).max() > 1e-9


# ---------------------------------------------------------------- P4 div B
def test_P4a_1d_Bx_constant():
    """1D: Phi_{Bx},x = 0 and tr Pi_B = first moment of the B_x set = 0 -> B_x never changes."""
    rng = np.random.default_rng(3)
    nx = 64
    s = (1, 1, nx)
    rho, u, B, p = admissible_ideal(rng, s)
    B[0] = 0.0375
    F = ideal_fields(rho, u, B, p, 2.0)
    par = orc.make_params(orc.IDEAL, orc.D1Q3, (nx,), gamma=2.0, tau=0.6, powell=1.0)
    o = orc.Oracle(par)
    o.init(F)
    o.step(200)
    Q = o.moments(diag=False)
    assert np.abs(Q[5] - 0.0375).max() < 2e-16 * 200


def div_h(Bx, By, lat="D2Q9"):
    """lattice divergence sum_i w_i c_i . B(x + c_i) / cs2 on [y, x] arrays, periodic"""
    D, c, w, cs2 = lattice_np(lat)
    out = np.zeros_like(Bx)
    for i in range(len(w)):
        sh = lambda a: np.roll(np.roll(a, -c[i][0], axis=1), -c[i][1], axis=0)
        out += w[i] * (c[i][0] * sh(Bx) + c[i][1] * sh(By))
    return out / cs2


def curl_h(A, lat="D2Q9"):
    """B = (D_y A, -D_x A) with the same lattice operator -> div_h B = 0 identically"""
    D, c, w, cs2 = lattice_np(lat)
    Dx = np.zeros_like(A)
    Dy = np.zeros_like(A)
    for i in range(len(w)):
        sh = np.roll(np.roll(A, -c[i][0], axis=1), -c[i][1], axis=0)
        Dx += w[i] * c[i][0] * sh / cs2
        Dy += w[i] * c[i][1] * sh / cs2
    return Dy, -Dx


def smooth_potential(rng, ny, nx, nmodes=4):
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    A = np.zeros((ny, nx))
    for _ in range(nmodes):
        kx, ky = rng.integers(-2, 3, size=2)
        A += rng.normal() * np.cos(2 * np.pi * (kx * x / nx + ky * y / ny) + rng.uniform(0, 2 * np.pi))
    return A


@pytest.mark.parametrize("scheme", ["IDEAL", "INCRES"])
def test_P4b_divh_free_stays_free_tauB_one(scheme):
    """tau_B = 1, kappa = 0, periodic: div_h B(t+1) = A[div_h B(t)] because Phi_B is antisymmetric."""
    rng = np.random.default_rng(17)
    nx, ny = 32, 24
    Bx, By = curl_h(smooth_potential(rng, ny, nx))
    ux, uy = curl_h(smooth_potential(rng, ny, nx))
    sc = 0.08 / max(np.abs(Bx).max(), np.abs(By).max())
    Bx, By = sc * Bx, sc * By
    sc = 0.08 / max(np.abs(ux).max(), np.abs(uy).max())
    ux, uy = sc * ux, sc * uy
    assert np.abs(div_h(Bx, By)).max() < 1e-16
    if scheme == "IDEAL":
        tau = [0.6] * 5 + [1.0] * 3
        rho = 1.0 + 0.1 * np.cos(2 * np.pi * np.arange(nx) / nx)[None, :] * np.ones((ny, 1))
        u = np.stack([ux, uy, 0 * ux])[:, None]
        B = np.stack([Bx, By, 0 * Bx])[:, None]
        F = ideal_fields(rho[None], u, B, 0.05 * np.ones((1, ny, nx)), G)
        par = orc.make_params(orc.IDEAL, orc.D2Q9, (nx, ny), gamma=G, tau=tau, powell=0.0)
        iB = 5
    else:
        tau = [0.6] * 3 + [1.0] * 2
        F = np.stack([0 * ux, ux, uy, Bx, By])[:, None]
        par = orc.make_params(orc.INCRES, orc.D2Q9, (nx, ny), tau=tau, powell=0.0)
        iB = 3
    o = orc.Oracle(par)
    o.init(F)
    o.step(100)
    Q, dg = o.moments()
    d = div_h(Q[iB][0], Q[iB + 1][0])
    assert np.abs(d).max() < 1e-15
    assert abs(dg[3 * o.K] - np.abs(d).max()) < 1e-17        # the oracle's own diagnostic is this operator
    assert np.abs(Q[iB][0] - Bx).max() > 1e-4                 # the field did evolve


def test_P4b_divh_obeys_smoothing_recursion():
    """same setting but div_h B != 0 initially: div_h B(t+1) = sum_i w_i div_h B(t)(x - c_i)"""
    rng = np.random.default_rng(19)
    nx, ny = 16, 12
    D, c, w, cs2 = lattice_np("D2Q9")
    s = (1, ny, nx)
    rho, u, B, p = admissible_ideal(rng, s)
    F = ideal_fields(rho, u, B, p, G)
    par = orc.make_params(orc.IDEAL, orc.D2Q9, (nx, ny), gamma=G, tau=[0.8] * 5 + [1.0] * 3, powell=0.0)
    o = orc.Oracle(par)
    o.init(F)
    Q = o.moments(diag=False)
    d = div_h(Q[5][0], Q[6][0])
    for _ in range(5):
        o.step(1)
        Q = o.moments(diag=False)
        dn = div_h(Q[5][0], Q[6][0])
        pred = sum(w[i] * np.roll(np.roll(d, c[i][0], axis=1), c[i][1], axis=0) for i in range(9))
        assert np.abs(dn - pred).max() < 1e-15
        d = dn


def test_A6_local_divB_estimator_tracks_divergence():
    """reading A6: delta = -tr Pi_B/(tau_B cs2) approximates div B.  Direct injection adds exactly S_k to
    Q_k at the cell (A5), so one step from identical populations with kappa = 1 and kappa = 0 differs by
    S(x) in the moments; S_{B_x} = -delta u_x gives delta(x), compared with a central difference."""
    nx, ny = 128, 4
    x = np.arange(nx)
    k = 2 * np.pi * 2 / nx
    one = np.ones((1, ny, nx))
    Bx = 0.05 * np.sin(k * x)[None, None, :] * one          # div B = dBx/dx != 0
    u = np.stack([0.02 * one, 0 * one, 0 * one])
    B = np.stack([Bx, 0 * one, 0 * one])
    F = ideal_fields(one, u, B, 0.05 * one, G)
    for tau in (0.55, 0.8, 1.0):
        p0 = orc.make_params(orc.IDEAL, orc.D2Q9, (nx, ny), gamma=G, tau=tau, powell=0.0)
        p1 = orc.make_params(orc.IDEAL, orc.D2Q9, (nx, ny), gamma=G, tau=tau, powell=1.0)
        o0, o1 = orc.Oracle(p0), orc.Oracle(p1)
        o0.init(F)
        o0.step(20)                                         # let the non-equilibrium part establish itself
        g = o0.populations()
        o1.init(F)
        o1.set_populations(g)
        o0.step(1)
        o1.step(1)
        Q0, Q1 = o0.moments(diag=False), o1.moments(diag=False)
        # pre-collision state of that step = streamed populations; its B_x and u_x
        D, c, w, cs2 = lattice_np("D2Q9")
        f = np.stack([np.roll(np.roll(g[:, i, 0], c[i][0], axis=2), c[i][1], axis=1) for i in range(9)], axis=1)
        Qpre = f.sum(1)
        ux = Qpre[1] / Qpre[0]
        delta = -(Q1[5][0] - Q0[5][0]) / ux
        dBdx = (np.roll(Qpre[5], -1, axis=1) - np.roll(Qpre[5], 1, axis=1)) / 2
        assert np.abs(dBdx).max() > 1e-3
        assert np.abs(delta - dBdx).max() < 0.02 * np.abs(dBdx).max(), tau
        # and the other rows of Eq.12: S_m = -delta B, S_E = -delta u.B, S_rho = 0
        assert np.abs((Q1[1][0] - Q0[1][0]) + delta * Qpre[5]).max() < 1e-16
        uB = (Qpre[1:4] / Qpre[0] * Qpre[5:8]).sum(0)
        assert np.abs((Q1[4][0] - Q0[4][0]) + delta * uB).max() < 1e-16
        assert np.array_equal(Q1[0], Q0[0])


# ---------------------------------------------------------------- P7 symmetries
@pytest.mark.parametrize("lat,shape", [("D2Q9", (16, 12)), ("D3Q19", (10, 8, 6))])
def test_P7_mirror_symmetry(lat, shape):
    """x -> L - x with u_x -> -u_x and B reflected as a polar vector stays a symmetry of the run."""
    rng = np.random.default_rng(23)
    s = zyx(shape)
    rho, u, B, p = admissible_ideal(rng, s)

    def sym(a, odd):
        m = a[..., ::-1]
        return 0.5 * (a - m) if odd else 0.5 * (a + m)
    rho, p = sym(rho, False), sym(p, False)
    u = np.stack([sym(u[0], True), sym(u[1], False), sym(u[2], False)])
    B = np.stack([sym(B[0], True), sym(B[1], False), sym(B[2], False)])
    F = ideal_fields(rho, u, B, p, G)
    par = orc.make_params(orc.IDEAL, LATS[lat], shape, gamma=G, tau=0.6, powell=1.0)
    o = orc.Oracle(par)
    o.init(F)
    o.step(30)
    Q = o.moments(diag=False)
    for k in range(8):
        odd = k in (1, 5)
        m = Q[k][..., ::-1]
        assert np.abs(Q[k] - (-m if odd else m)).max() < 1e-13
    assert np.abs(Q[1]).max() > 1e-3


def test_P7_rotation_90():
    """a 90-degree rotated initial state gives the rotated result (square grid, D2Q9)."""
    rng = np.random.default_rng(29)
    n = 12
    rho, u, B, p = admissible_ideal(rng, (1, n, n))
    F = ideal_fields(rho, u, B, p, G)

    def rot(Fin):
        # rotate the picture by +90 degrees: new(x, y) = old(y, n-1-x); vectors (vx, vy) -> (-vy, vx)
        r = lambda a: np.rot90(a[0], k=1, axes=(1, 0))[None] if False else np.transpose(a[0])[:, ::-1][None]
        out = np.empty_like(Fin)
        out[0], out[4] = r(Fin[0]), r(Fin[4])
        out[1], out[2], out[3] = -r(Fin[2]), r(Fin[1]), r(Fin[3])
        out[5], out[6], out[7] = -r(Fin[6]), r(Fin[5]), r(Fin[7])
        return out
    par = orc.make_params(orc.IDEAL, orc.D2Q9, (n, n), gamma=G, tau=0.65, powell=1.0)
    o1, o2 = orc.Oracle(par), orc.Oracle(par)
    o1.init(F)
    o2.init(rot(F))
    o1.step(20)
    o2.step(20)
    assert np.abs(rot(o1.moments(diag=False)) - o2.moments(diag=False)).max() < 1e-13


# ---------------------------------------------------------------- P9 obstacle
def test_P9_no_solid_is_bit_identical_and_solid_imposes_state():
    rng = np.random.default_rng(31)
    shape = (10, 8, 6)
    s = zyx(shape)
    F = random_fields(rng, "IDEAL", "D3Q19", shape, gamma=G)
    par = orc.make_params(orc.IDEAL, orc.D3Q19, shape, gamma=G, tau=0.7, powell=1.0)
    a, b = orc.Oracle(par), orc.Oracle(par)
    b.set_obstacle(np.zeros(s, dtype=np.uint8), (0.1, 0.2, 0.3), 0.5 * np.ones((3,) + s))   # d = 1 everywhere
    a.init(F)
    b.init(F)
    a.step(5)
    b.step(5)
    assert np.array_equal(a.populations(), b.populations())
    mask = np.zeros(s, dtype=np.uint8)
    mask[2:4, 3:5, 4:7] = 2
    Bs = 0.1 * (rng.random((3,) + s) - 0.5)
    us = np.array([0.02, -0.01, 0.03])
    b.set_obstacle(mask, us, Bs)
    b.step(3)
    Q = b.moments(diag=False)
    sol = mask == 2
    for c in range(3):
        assert np.abs(Q[1 + c][sol] - Q[0][sol] * us[c]).max() < 1e-16       # m = rho u^B exactly
        assert np.abs(Q[5 + c][sol] - Bs[c][sol]).max() < 1e-16              # B = B^B exactly


def test_P9_stationary_solid_in_matching_uniform_state_is_invisible():
    shape = (8, 6, 5)
    s = zyx(shape)
    B0 = (0.05, -0.02, 0.03)
    F = uniform_ideal(shape, u=(0, 0, 0), B=B0)
    mask = np.zeros(s, dtype=np.uint8)
    mask[1:3, 2:4, 3:6] = 2
    par = orc.make_params(orc.IDEAL, orc.D3Q19, shape, gamma=G, tau=0.55, powell=1.0)
    o = orc.Oracle(par)
    o.set_obstacle(mask, (0, 0, 0), np.array(B0).reshape(3, 1, 1, 1) * np.ones(s))
    o.init(F)
    o.step(50)
    Q = o.moments(diag=False)
    assert np.abs(Q - F).max() < 1e-13          # round-off only; a visible solid would give O(1e-2)


# ---------------------------------------------------------------- P10 boundaries
def test_P10_frozen_cells_never_change_and_outflow_reflects_little():
    nx = 200
    x = np.arange(nx)
    one = np.ones((1, 1, nx))
    bump = 1e-3 * np.exp(-((x - 150.0) / 6.0) ** 2)[None, None, :]
    rho = one + bump
    p0 = 0.02
    p = p0 * (1 + G * bump)                       # acoustic pulse (both directions)
    F = ideal_fields(rho, np.zeros((3, 1, 1, nx)), np.zeros((3, 1, 1, nx)), p, G)
    par = orc.make_params(orc.IDEAL, orc.D1Q3, (nx,), gamma=G, tau=0.55, powell=1.0, bc=(2, 1, 0, 0, 0, 0))
    o = orc.Oracle(par)
    o.init(F)
    g0 = o.populations()
    a = np.sqrt(G * p0)                           # 0.18 cells / step
    o.step(int(80 / a))                           # right-going half has left through x = nx-1, left-going is mid-domain
    g1 = o.populations()
    assert np.array_equal(g0[..., 0], g1[..., 0])                   # INFLOW face cell is frozen (A10)
    Q = o.moments(diag=False)
    dev = np.abs(Q[0][0, 0] - 1.0)
    left_going = dev[:120].max()
    reflected = dev[125:].max()
    assert left_going > 2e-4                      # half-amplitude pulse still travelling
    assert reflected < 0.05 * 1e-3                # < 5 % of the incident amplitude came back
