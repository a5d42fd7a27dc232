"""Pins P5, P5b, P8 of the CPU oracle: linear waves and hydrodynamic limits.

P5b builds the exact Fourier symbol of the linearised update in numpy, independent of the oracle's
update code; P5 is the closed-form long-wave limit (Eq.5 PAPER.md:98 reduced by 1 - a^2/c_s^2);
P8 compares the B = 0 scheme with the exact Riemann solution of the Euler equations and the
Taylor-Green decay law.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from np_vlbm import lattice_np
from test_oracle_pins import LATS, zyx, ideal_fields

G = 5 / 3


def jacobians(params, Q0, D, h=1e-6):
    """A[alpha][k][l] = d Phi_{k,alpha} / d Q_l by central differences of the flux."""
    K = len(Q0)
    A = np.zeros((D, K, K))
    for l in range(K):
        e = np.zeros(K)
        e[l] = h * max(1.0, abs(Q0[l]))
        Fp, Fm = orc.flux(params, Q0 + e), orc.flux(params, Q0 - e)
        for a in range(D):
            A[a][:, l] = (Fp[:, a] - Fm[:, a]) / (2 * e[l])
    return A


def symbol(lat, scheme, params, Q0, tau, kvec, kappa):
    """M(k) acting on the stored (post-collision) populations, index (k, i) -> k*Qn + i:
    one step = pull (factor exp(-i k.c_i)) then linearised collide + Powell injection."""
    D, c, w, cs2 = lattice_np(lat)
    Qn, K = len(w), len(Q0)
    A = jacobians(params, Q0, D)
    iB = 5 if scheme == "IDEAL" else 1 + D
    if scheme == "IDEAL":
        u0, B0 = Q0[1:4] / Q0[0], Q0[5:8]
        svec = np.concatenate([[0.0], B0, [u0 @ B0], u0])
    else:
        svec = np.concatenate([[0.0], Q0[1 + D:], Q0[1:1 + D]])
    n = K * Qn
    Cm = np.zeros((n, n))
    for k in range(K):
        om = 1.0 / tau[k]
        for i in range(Qn):
            r = k * Qn + i
            Cm[r, r] += 1.0 - om
            for j in range(Qn):
                Cm[r, k * Qn + j] += om * w[i]                                   # w_i dQ_k
                for l in range(K):
                    cA = sum(c[i][a] * A[a][k, l] for a in range(D))
                    Cm[r, l * Qn + j] += om * w[i] * cA / cs2                    # w_i c_i.(A dQ)_k / cs2
            # source: w_i * s_k * (-kappa) * delta,  delta = -sum_b sum_j c_jb f_{B_b,j} / (tau_B cs2)
            for b in range(D):
                for j in range(Qn):
                    Cm[r, (iB + b) * Qn + j] += w[i] * svec[k] * kappa * c[j][b] / (tau[iB] * cs2)
    shift = np.array([np.exp(-1j * (kvec[:D] @ c[i][:D])) for i in range(Qn)])
    return Cm @ np.diag(np.tile(shift, K)), A


CASES = [
    ("D1Q3", "IDEAL", (64,), np.array([1.0, 0.06, 0.03, -0.02, 0.0, 0.09, 0.05, 0.02]), 0.03, (1, 0, 0), 1.0),
    ("D2Q9", "IDEAL", (32, 16), np.array([1.2, 0.05, -0.04, 0.02, 0.0, 0.06, 0.08, -0.03]), 0.04, (1, 2, 0), 1.0),
    ("D3Q19", "IDEAL", (16, 8, 8), np.array([0.9, 0.03, 0.05, -0.04, 0.0, 0.07, -0.05, 0.04]), 0.03, (1, 1, 1), 1.0),
    ("D2Q9", "INCRES", (32, 16), np.array([0.01, 0.04, -0.03, 0.05, 0.06]), None, (2, 1, 0), 1.0),
    ("D2Q9", "IDEAL", (32, 16), np.array([1.2, 0.05, -0.04, 0.02, 0.0, 0.06, 0.08, -0.03]), 0.04, (1, 2, 0), 0.0),
]


@pytest.mark.parametrize("lat,scheme,shape,Q0,p0,kint,kappa", CASES)
def test_P5b_exact_symbol(lat, scheme, shape, Q0, p0, kint, kappa):
    D = lattice_np(lat)[0]
    Q0 = Q0.copy()
    if scheme == "IDEAL":
        rho, m, B = Q0[0], Q0[1:4], Q0[5:8]
        Q0[4] = p0 / (G - 1) + 0.5 * (m @ m) / rho + 0.5 * (B @ B)
        K = 8
        tau = np.array([0.6, 0.7, 0.7, 0.7, 0.55, 0.8, 0.8, 0.8])
    else:
        K = 1 + 2 * D
        tau = np.array([0.6] + [0.7] * D + [0.9] * D)
    params = orc.make_params(orc.IDEAL if scheme == "IDEAL" else orc.INCRES, LATS[lat], shape, gamma=G, tau=tau, powell=kappa)
    s = zyx(shape)
    n_axis = np.array(list(shape) + [1] * (3 - len(shape)), dtype=float)
    kvec = 2 * np.pi * np.array(kint, dtype=float) / n_axis
    M, _ = symbol(lat, scheme, params, Q0, tau, kvec, kappa)
    lam, V = np.linalg.eig(M)
    order = np.argsort(-np.abs(lam))
    zz, yy, xx = np.meshgrid(*[np.arange(n) for n in s], indexing="ij")
    phase = np.exp(1j * (kvec[0] * xx + kvec[1] * yy + kvec[2] * zz))
    Qn = lattice_np(lat)[2].size
    f0 = orc.equilibrium(params, Q0)                          # [K, Qn]
    eps, nsteps = 1e-7, 40
    tested = 0
    for idx in order[:K]:                                     # the K physical (slow) modes
        v = V[:, idx] / np.abs(V[:, idx]).max()
        o = orc.Oracle(params)
        o.init(np.broadcast_to(Q0.reshape(K, 1, 1, 1), (K,) + s).copy())
        g0 = f0.reshape(K, Qn, 1, 1, 1) + eps * np.real(v.reshape(K, Qn, 1, 1, 1) * phase)
        o.set_populations(g0)
        o.step(nsteps)
        g = o.populations()
        want = f0.reshape(K, Qn, 1, 1, 1) + eps * np.real((lam[idx] ** nsteps) * v.reshape(K, Qn, 1, 1, 1) * phase)
        err = np.abs(g - want).max() / eps
        assert err < 1e-6, (idx, lam[idx], err)
        tested += 1
    assert tested == K
    assert np.abs(lam[order[K - 1]]) > 0.5 and np.abs(lam).max() < 1 + 1e-12     # stable; K slow (physical) modes


@pytest.mark.parametrize("tau", [0.51, 0.6, 0.8])
def test_P5_closed_form_long_wave(tau):
    """equal tau: |lambda| = exp(-(tau - 1/2)(cs2 - a^2) k^2), arg lambda = -a k, to O(k^2) relative,
    for every characteristic speed a of the flux Jacobian (sound, Alfven, slow/fast, entropy)."""
    lat, shape = "D1Q3", (256,)
    Q0 = np.array([1.0, 0.05, 0.02, -0.01, 0.0, 0.12, 0.07, 0.03])
    Q0[4] = 0.03 / (G - 1) + 0.5 * (Q0[1:4] @ Q0[1:4]) / Q0[0] + 0.5 * (Q0[5:8] @ Q0[5:8])
    taus = np.full(8, tau)
    params = orc.make_params(orc.IDEAL, LATS[lat], shape, gamma=G, tau=taus, powell=0.0)
    k = 2 * np.pi * 2 / 256
    M, A = symbol(lat, "IDEAL", params, Q0, taus, np.array([k, 0, 0]), 0.0)
    lam = np.linalg.eigvals(M)
    lam = lam[np.argsort(-np.abs(lam))][:8]
    speeds = np.sort(np.linalg.eigvals(A[0]).real)
    # textbook ideal-MHD speeds for this state (independent of the Jacobian): u, u +- c_A, u +- c_f, u +- c_s, (u: div-B mode -> 0 flux row: speed 0)
    rho, ux, Bx = Q0[0], Q0[1] / Q0[0], Q0[5]
    a2, b2 = G * 0.03 / rho, (Q0[5:8] @ Q0[5:8]) / rho
    ca = abs(Bx) / np.sqrt(rho)
    disc = np.sqrt((a2 + b2) ** 2 - 4 * a2 * ca ** 2)
    cf, csl = np.sqrt(0.5 * (a2 + b2 + disc)), np.sqrt(0.5 * (a2 + b2 - disc))
    textbook = np.sort([0.0, ux, ux - ca, ux + ca, ux - cf, ux + cf, ux - csl, ux + csl])
    assert np.allclose(speeds, textbook, atol=2e-7)
    got_phase = np.sort(-np.angle(lam) / k)
    assert np.allclose(got_phase, speeds, atol=5e-4)
    for a in speeds:
        j = np.argmin(np.abs(-np.angle(lam) / k - a))
        rate = -np.log(np.abs(lam[j]))
        want = (tau - 0.5) * (1.0 / 3.0 - a * a) * k * k
        assert abs(rate - want) <= 0.01 * want, (a, rate, want)


# ---------------------------------------------------------------- P8 hydrodynamic limits
def sod_exact(x, t, g=1.4, L=(1.0, 0.0, 1.0), R=(0.125, 0.0, 0.1), x0=0.5):
    """exact Riemann solution of the 1D Euler equations for the Sod data (textbook construction:
    left rarefaction, contact, right shock; p* by Newton iteration on the pressure function)."""
    rl, ul, pl = L
    rr, ur, pr = R
    al, ar = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)

    def fk(p, rk, pk, ak):
        if p > pk:
            Ak, Bk = 2 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * np.sqrt(Ak / (p + Bk)), np.sqrt(Ak / (p + Bk)) * (1 - (p - pk) / (2 * (Bk + p)))
        return 2 * ak / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), 1 / (rk * ak) * (p / pk) ** (-(g + 1) / (2 * g))
    p = 0.5 * (pl + pr)
    for _ in range(50):
        f1, d1 = fk(p, rl, pl, al)
        f2, d2 = fk(p, rr, pr, ar)
        dp = (f1 + f2 + ur - ul) / (d1 + d2)
        p -= dp
        if abs(dp) < 1e-14:
            break
    us = 0.5 * (ul + ur) + 0.5 * (fk(p, rr, pr, ar)[0] - fk(p, rl, pl, al)[0])
    rsl = rl * (p / pl) ** (1 / g)
    asl = al * (p / pl) ** ((g - 1) / (2 * g))
    rsr = rr * ((p / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pr + 1))
    S = ur + ar * np.sqrt((g + 1) / (2 * g) * p / pr + (g - 1) / (2 * g))
    xi = (x - x0) / t
    rho, u, pp = np.empty_like(x), np.empty_like(x), np.empty_like(x)
    for j, s in enumerate(xi):
        if s < ul - al:
            rho[j], u[j], pp[j] = rl, ul, pl
        elif s < us - asl:
            uu = 2 / (g + 1) * (al + (g - 1) / 2 * ul + s)
            aa = al - (g - 1) / 2 * (uu - ul)
            rho[j], u[j], pp[j] = rl * (aa / al) ** (2 / (g - 1)), uu, pl * (aa / al) ** (2 * g / (g - 1))
        elif s < us:
            rho[j], u[j], pp[j] = rsl, us, p
        elif s < S:
            rho[j], u[j], pp[j] = rsr, us, p
        else:
            rho[j], u[j], pp[j] = rr, ur, pr
    return rho, u, pp


def test_P8_euler_limit_sod_tube():
    """B = 0 stays 0 and the scheme solves the Euler equations: L1 distance to the exact Sod solution."""
    g, nx, s = 1.4, 800, 0.1
    x = (np.arange(nx) + 0.5) / nx
    left = x < 0.5
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1) * s * s                       # A1: (u, B, p, E) -> (s u, s B, s^2 p, s^2 E)
    z = np.zeros((3, 1, 1, nx))
    F = ideal_fields(rho[None, None], z, z, p[None, None], g)
    par = orc.make_params(orc.IDEAL, orc.D1Q3, (nx,), gamma=g, tau=0.6, powell=1.0, bc=(1, 1, 0, 0, 0, 0))
    o = orc.Oracle(par)
    o.init(F)
    nsteps = 1600                                              # t = nsteps * s / nx = 0.2
    o.step(nsteps)
    Q, dg = o.moments()
    assert np.abs(Q[5:8]).max() == 0.0 and np.abs(Q[2:4]).max() == 0.0
    assert dg[3 * 8 + 1] > 0 and dg[3 * 8 + 2] > 0 and dg[3 * 8 + 3] == 0
    rho_n = Q[0][0, 0]
    u_n = Q[1][0, 0] / rho_n / s
    p_n = (g - 1) * (Q[4][0, 0] - 0.5 * Q[1][0, 0] ** 2 / rho_n) / (s * s)
    re, ue, pe = sod_exact(x, nsteps * s / nx, g)
    assert np.abs(rho_n - re).mean() < 0.01
    assert np.abs(u_n - ue).mean() < 0.015
    assert np.abs(p_n - pe).mean() < 0.01
    # wave ordering: rarefaction head < contact < shock positions found from the numerical profile
    i_shock = np.max(np.where(p_n > 0.2)[0])
    i_contact = np.max(np.where(rho_n > 0.5 * (0.42632 + 0.26557))[0])
    assert 0.5 < x[i_contact] < x[i_shock] < 0.9
    assert abs(x[i_shock] - (0.5 + 1.75216 * 0.2)) < 0.01      # textbook shock speed for Sod data


def test_P8_incres_taylor_green_decay():
    """INCRES, B = 0: a Taylor-Green vortex decays like exp(-2 nu k^2 t), nu from Eq.5 (tau = 1/2 + nu/cs2)."""
    n, U, nu = 64, 0.02, 0.02
    k = 2 * np.pi / n
    y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    ux = U * np.sin(k * x) * np.cos(k * y)
    uy = -U * np.cos(k * x) * np.sin(k * y)
    P = 0.25 * U * U * (np.cos(2 * k * x) + np.cos(2 * k * y))
    F = np.stack([P, ux, uy, 0 * ux, 0 * ux])[:, None]
    par = orc.make_params(orc.INCRES, orc.D2Q9, (n, n), nu=nu, tau=0.9, eta=0.01, powell=1.0)
    o = orc.Oracle(par)
    o.init(F)
    amps = []
    for _ in range(5):
        Q = o.moments(diag=False)
        amps.append(2 * (Q[1][0] * np.sin(k * x) * np.cos(k * y)).mean() * 2)
        o.step(100)
    amps = np.array(amps)
    rate = -np.log(amps[1:] / amps[:-1]) / 100
    assert np.abs(Q[3:5]).max() == 0.0
    # first interval carries the start-up transient of the non-equilibrium part
    assert np.allclose(rate[1:], 2 * nu * k * k, rtol=0.01, atol=0)
    assert abs(rate[0] - 2 * nu * k * k) < 0.06 * 2 * nu * k * k
