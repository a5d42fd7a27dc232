"""Pins of the full dissipative scheme ORC_FULL (PAPER.md:122 with Eq.9: the viscous stress and
the magnetic gradients transported as independent variables; A23): Q = (rho, m, E, B, G_ab, H_ab),
G ~ tau_M d_a B_b, H ~ tau_M d_a u_b, sigma = mu (h + h^T - 2/3 tr h I) with h = H / tau_M.

What fixes the oracle here other than its own code:
  * the flux against a tensor-form numpy writing (einsum for sigma and u . sigma), and against hand values for one state;
  * the exact Fourier symbol of the linearised update, built in numpy from numerical Jacobians of THAT numpy flux,
    against eigenmode runs of the oracle (1e-6), 1D / 2D / 3D, with the Powell term;
  * physics: a transverse velocity shear mode decays at (mu / rho + (tau_u - 1/2) c_s^2) k^2 (the compressive part of
    sigma is covered by the symbol and the hand values), and the stored H equals (tau_M - 1) grad u (pre-collision
    tau_M grad u, Eq.7);
  * exact balances: rho, m, E, B conserved (kappa = 0), sum G and sum H contract by (1 - 1/tau_M) per step;
  * mu = 0: the first 8 + 3 D variables are bit-identical to the RESIST scheme;
  * the array-at-a-time numpy restatement (tests/np_vlbm.py) with boundaries and a moving body.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from np_vlbm import NpVLBM, flux_full, lattice_np
from test_oracle_pins import LATS, zyx, ideal_fields, random_fields

G = 5 / 3


def full_fields(rng, lat, shape, amp=1e-3):
    D = len(shape)
    F8 = random_fields(rng, "IDEAL", lat, shape, gamma=G)
    return np.concatenate([F8, amp * rng.standard_normal((6 * D,) + F8.shape[1:])])


@pytest.mark.parametrize("lat", ["D1Q3", "D2Q9", "D3Q19", "D3Q7"])
def test_flux_matches_tensor_form(lat):
    rng = np.random.default_rng(2)
    D = lattice_np(lat)[0]
    p = orc.make_params(orc.FULL, LATS[lat], (4,) * D, gamma=G, tau=0.6, eta=0.013, nu=0.021, tau_relax=2.5)
    for _ in range(20):
        rho, p0 = 0.5 + rng.random(), 0.1 + rng.random()
        m, B = rng.standard_normal(3), rng.standard_normal(3)
        E = p0 / (G - 1) + 0.5 * m @ m / rho + 0.5 * B @ B
        Q = np.concatenate([[rho], m, [E], B, rng.standard_normal(6 * D)])
        got = orc.flux(p, Q)
        want = flux_full(Q, G, D, 0.013, 0.021, 2.5)
        assert np.abs(got - want).max() < 1e-13 * max(1.0, np.abs(want).max())
    Q2 = Q.copy()
    Q2[8 + 3 * D:] = 0.0
    assert np.abs(orc.flux(p, Q)[1:5] - orc.flux(p, Q2)[1:5]).max() > 1e-4       # the viscous terms are really there


def test_flux_hand_values_3d():
    """rho = 2, u = (1, 2, 3), B = 0, G = 0, H/tau_M = h with h_xy = 0.5, h_yx = 0.1, h_zz = 0.3, mu = 0.2, tau_M = 2:
    tr h = 0.3; sigma_xy = sigma_yx = 0.2 * 0.6 = 0.12; sigma_xx = sigma_yy = -0.2 * 0.2 = -0.04; sigma_zz = 0.2 (0.6 - 0.2) = 0.08."""
    mu, tm = 0.2, 2.0
    p = orc.make_params(orc.FULL, LATS["D3Q19"], (4, 4, 4), gamma=G, tau=0.6, eta=0.0, nu=mu, tau_relax=tm)
    rho, u = 2.0, np.array([1.0, 2.0, 3.0])
    E = 1.0 / (G - 1) + 0.5 * rho * u @ u
    H = np.zeros((3, 3))
    H[0, 1], H[1, 0], H[2, 2] = 0.5 * tm, 0.1 * tm, 0.3 * tm
    Q = np.concatenate([[rho], rho * u, [E], np.zeros(3), np.zeros(9), H.reshape(-1)])
    Q0 = Q.copy()
    Q0[17:] = 0.0
    d = orc.flux(p, Q) - orc.flux(p, Q0)           # [K, 3]: the viscous contribution (plus Phi_H itself)
    sig = np.array([[-0.04, 0.12, 0.0], [0.12, -0.04, 0.0], [0.0, 0.0, 0.08]])
    for a in range(3):
        for b in range(3):
            assert abs(d[1 + b, a] + sig[a, b]) < 1e-13
        assert abs(d[4, a] + u @ sig[a]) < 1e-13
    assert np.abs(d[5:17]).max() == 0.0
    # Phi_{H_cb},a = H_cb u_a - delta_ca u_b
    F = orc.flux(p, Q)
    for c in range(3):
        for b in range(3):
            for a in range(3):
                assert abs(F[17 + 3 * c + b, a] - (H[c, b] * u[a] - (u[b] if c == a else 0.0))) < 1e-15


def np_jacobians(Q0, D, eta, mu, tau_m, h=1e-6):
    K = len(Q0)
    A = np.zeros((D, K, K))
    for l in range(K):
        e = np.zeros(K)
        e[l] = h * max(1.0, abs(Q0[l]))
        Fp, Fm = flux_full(Q0 + e, G, D, eta, mu, tau_m), flux_full(Q0 - e, G, D, eta, mu, tau_m)
        for a in range(D):
            A[a][:, l] = (Fp[:, a] - Fm[:, a]) / (2 * e[l])
    return A


def symbol(lat, Q0, tau, kvec, kappa, eta, mu, tau_m):
    """one step on the stored populations: pull (phase exp(-i k.c_i)), then collide with the linearised flux, the Powell
    source fed by tr G / tau_M and the relaxation sources -G / tau_M, -H / tau_M, all injected with weight w_i"""
    D, c, w, cs2 = lattice_np(lat)
    Qn, K = len(w), len(Q0)
    A = np_jacobians(Q0, D, eta, mu, tau_m)
    u0, B0 = Q0[1:4] / Q0[0], Q0[5:8]
    svec = np.concatenate([[0.0], B0, [u0 @ B0], u0, np.zeros(6 * D)])
    n = K * Qn
    Cm = np.zeros((n, n))
    for k in range(K):
        om = 1.0 / tau[k]
        for i in range(Qn):
            r = k * Qn + i
            Cm[r, r] += 1.0 - om
            for j in range(Qn):
                Cm[r, k * Qn + j] += om * w[i]
                for l in range(K):
                    Cm[r, l * Qn + j] += om * w[i] * sum(c[i][a] * A[a][k, l] for a in range(D)) / cs2
                for a in range(D):
                    Cm[r, (8 + 3 * a + a) * Qn + j] += -kappa * w[i] * svec[k] / tau_m
                if k >= 8:
                    Cm[r, k * Qn + j] += -w[i] / tau_m
    shift = np.array([np.exp(-1j * (kvec[:D] @ c[i][:D])) for i in range(Qn)])
    return Cm @ np.diag(np.tile(shift, K))


@pytest.mark.parametrize("lat,shape,kint,kappa", [("D1Q3", (64,), (1, 0, 0), 1.0), ("D2Q9", (32, 16), (1, 2, 0), 1.0),
                                                  ("D3Q7", (16, 8, 8), (1, 1, 1), 0.0)])
def test_exact_symbol_eigenmodes(lat, shape, kint, kappa):
    D = lattice_np(lat)[0]
    K = 8 + 6 * D
    slow = lat == "D3Q7"
    sc = 0.4 if slow else 1.0
    rho, m, B, p0 = 1.1, sc * np.array([0.05, -0.04, 0.02]), sc * np.array([0.06, 0.08, -0.03]), sc * sc * 0.04
    Q0 = np.concatenate([[rho], m, [p0 / (G - 1) + 0.5 * m @ m / rho + 0.5 * B @ B], B, np.zeros(6 * D)])
    tau = np.array([0.6, 0.7, 0.7, 0.7, 0.55, 0.8, 0.8, 0.8] + [0.65] * (3 * D) + [0.75] * (3 * D))
    eta, mu, tau_m = 0.02, 0.03, 3.0
    params = orc.make_params(orc.FULL, LATS[lat], shape, gamma=G, tau=tau, powell=kappa, eta=eta, nu=mu, tau_relax=tau_m)
    s = zyx(shape)
    n_axis = np.array(list(shape) + [1] * (3 - len(shape)), dtype=float)
    kvec = 2 * np.pi * np.array(kint, dtype=float) / n_axis
    M = symbol(lat, Q0, tau, kvec, kappa, eta, mu, tau_m)
    lam, V = np.linalg.eig(M)
    order = np.argsort(-np.abs(lam))
    zz, yy, xx = np.meshgrid(*[np.arange(n) for n in s], indexing="ij")
    phase = np.exp(1j * (kvec[0] * xx + kvec[1] * yy + kvec[2] * zz))
    Qn = lattice_np(lat)[2].size
    f0 = orc.equilibrium(params, Q0)
    eps, nsteps = 1e-7, 30
    gb = f0.reshape(K, Qn, 1, 1, 1)
    for idx in order[:K]:
        v = V[:, idx] / np.abs(V[:, idx]).max()
        o = orc.Oracle(params)
        o.init(np.broadcast_to(Q0.reshape(K, 1, 1, 1), (K,) + s).copy())
        o.set_populations(f0.reshape(K, Qn, 1, 1, 1) + eps * np.real(v.reshape(K, Qn, 1, 1, 1) * phase))
        o.step(nsteps)
        got = (o.populations() - gb) / eps
        want = np.real((lam[idx] ** nsteps) * v.reshape(K, Qn, 1, 1, 1) * phase)
        assert np.abs(got - want).max() < 2e-6, (idx, lam[idx])
    assert np.abs(lam).max() < 1 + 1e-12


@pytest.mark.parametrize("mu,tau_m", [(0.01, 2.0), (0.03, 4.0), (0.0, 2.0)])
def test_viscous_shear_decay_and_recovered_gradient(mu, tau_m):
    """fluid at rest, B = 0, u_y = eps sin(k x): the shear mode decays at (mu / rho + (tau_u - 1/2) c_s^2) k^2 and the stored
    H_xy is (tau_M - 1) d_x u_y"""
    nx, tauU, rho0 = 128, 0.6, 1.3
    k = 2 * np.pi / nx
    x = np.arange(nx)
    eps = 1e-4
    rho = rho0 * np.ones((1, 1, nx))
    u = np.zeros((3, 1, 1, nx))
    u[1, 0, 0] = eps * np.sin(k * x)
    F8 = ideal_fields(rho, u, np.zeros((3, 1, 1, nx)), 0.02 * np.ones((1, 1, nx)), G)
    F = np.concatenate([F8, np.zeros((6, 1, 1, nx))])
    tau = [0.6] + [tauU] * 3 + [0.6] * 4 + [0.6] * 6
    o = orc.Oracle(orc.make_params(orc.FULL, LATS["D1Q3"], (nx,), gamma=G, tau=tau, powell=1.0, eta=0.0, nu=mu, tau_relax=tau_m))
    o.init(F)
    o.step(200)
    Q1, _ = o.moments()
    a1 = 2 * (Q1[2].reshape(-1) @ np.sin(k * x)) / nx / rho0
    o.step(400)
    Q2, _ = o.moments()
    a2 = 2 * (Q2[2].reshape(-1) @ np.sin(k * x)) / nx / rho0
    rate = -np.log(a2 / a1) / 400
    want = (mu / rho0 + (tauU - 0.5) / 3.0) * k * k
    assert abs(rate / want - 1) < 0.02, (rate, want)
    # H_xy (index 8 + 3 + 3*0 + 1 = 12): stored (post-collision) moment = (tau_M - 1) d_x u_y
    hxy = 2 * (Q2[12].reshape(-1) @ np.cos(k * x)) / nx
    assert abs(hxy / ((tau_m - 1.0) * a2 * k) - 1) < 0.01, (hxy, (tau_m - 1.0) * a2 * k)
    assert np.abs(Q2[13]).max() < 1e-12          # H_xz stays 0


@pytest.mark.parametrize("lat,shape", [("D1Q3", (32,)), ("D2Q9", (12, 10)), ("D3Q19", (8, 6, 5)), ("D3Q7", (8, 6, 5))])
def test_balances_periodic(lat, shape):
    rng = np.random.default_rng(5)
    tau_m = 2.5
    o = orc.Oracle(orc.make_params(orc.FULL, LATS[lat], shape, gamma=G, tau=0.7, powell=0.0, eta=0.02, nu=0.015, tau_relax=tau_m))
    o.init(full_fields(rng, lat, shape))
    _, d0 = o.moments()
    K = o.K
    for _ in range(5):
        o.step(1)
        _, d1 = o.moments()
        scale = d0[K:2 * K][:8].max()
        assert np.abs(d1[:8] - d0[:8]).max() < 1e-13 * scale * np.prod(shape)
        assert np.abs(d1[8:K] - (1 - 1 / tau_m) * d0[8:K]).max() < 1e-13 * max(d0[K + 8:2 * K].max(), 1e-30) * np.prod(shape)
        d0 = d1


def test_mu_zero_is_resist_bit_for_bit():
    rng = np.random.default_rng(8)
    shape = (10, 9, 8)
    F = full_fields(rng, "D3Q19", shape)
    a = orc.Oracle(orc.make_params(orc.FULL, LATS["D3Q19"], shape, gamma=G, tau=0.7, powell=1.0, eta=0.02, nu=0.0, tau_relax=3.0,
                                   bc=(1, 1, 0, 0, 0, 0)))
    b = orc.Oracle(orc.make_params(orc.RESIST, LATS["D3Q19"], shape, gamma=G, tau=0.7, powell=1.0, eta=0.02, tau_relax=3.0,
                                   bc=(1, 1, 0, 0, 0, 0)))
    a.init(F)
    b.init(F[:17])
    a.step(10)
    b.step(10)
    assert np.array_equal(a.moments()[0][:17], b.moments()[0])


@pytest.mark.parametrize("lat,shape,bc", [("D1Q3", (24,), (1, 1, 0, 0, 0, 0)), ("D2Q9", (13, 11), (2, 1, 0, 0, 0, 0)), ("D3Q19", (9, 8, 7), (0,) * 6),
                                          ("D3Q19", (9, 8, 7), (1, 1, 1, 1, 1, 1)), ("D2Q5", (13, 11), (0,) * 6)])
def test_numpy_restatement(lat, shape, bc):
    rng = np.random.default_rng(31)
    D = len(shape)
    F0 = full_fields(rng, lat, shape)
    tau = 0.7
    o = orc.Oracle(orc.make_params(orc.FULL, LATS[lat], shape, gamma=G, tau=tau, powell=1.0, bc=bc, eta=0.015, nu=0.012, tau_relax=2.0))
    m = NpVLBM("FULL", lat, zyx(shape), tau, gamma=G, powell=1.0, bc=bc, tau_relax=2.0)
    m.eta, m.mu = 0.015, 0.012
    if D > 1:
        c = np.array([sh / 2 - 0.4 for sh in shape] + [0.0] * (3 - D))
        us, mh = np.array([0.015, -0.01, 0.02 if D == 3 else 0.0]), np.array([0.6, 0.0, 0.8])
        o.set_sphere(c, 2.4, us, mh, 0.03)
        o.set_sphere_width(1.0)
        m.sphere, m.sphere_eps = (c, 2.4, us, mh, 0.03, 0), 1.0
    o.init(F0)
    m.init(F0)
    o.step(6)
    m.step(6)
    Q, _ = o.moments()
    assert np.abs(Q - m.moments()).max() < 1e-13
    assert np.abs(o.source_log() - m.src_acc).max() < 1e-12
    assert np.abs(o.body_read() - m.body).max() < 1e-12
