"""Pins of the current-dependent resistivity eta(j) = eta0 (1 + (j/j_c)^2) (reading A20)
in the INCRES scheme: cell-local tau_B from the antisymmetric non-equilibrium first moment of the B sets."""
import numpy as np
import pytest

from oracle import oracle as orc
from np_vlbm import NpVLBM, lattice_np
from test_oracle_pins import LATS, zyx, incres_fields
from test_oracle_invariants import curl_h, smooth_potential


def test_cubic_root_against_numpy_roots():
    rng = np.random.default_rng(1)
    for _ in range(200):
        e0 = 10 ** rng.uniform(-4, 0)
        tau0 = 0.5 + e0
        a2 = 10 ** rng.uniform(-8, 2)
        jc = 10 ** rng.uniform(-3, 1)
        t = orc.tau_of_current(tau0, e0, a2, jc)
        roots = np.roots([1.0, -tau0, 0.0, -e0 * a2 / jc ** 2])
        real = roots[np.abs(roots.imag) < 1e-9].real
        want = real[real >= tau0 - 1e-12].max()
        assert abs(t - want) <= 1e-9 * want, (tau0, a2, jc, t, want)
        assert abs(t - (0.5 + e0 * (1 + a2 / (t * t * jc * jc)))) < 1e-9 * t          # tau = 1/2 + eta(j)/cs2 with j = a/tau
    assert orc.tau_of_current(0.53, 0.03, 0.0, 0.1) == 0.53                         # no current: eta0


@pytest.mark.parametrize("lat,shape", [("D2Q9", (9, 8)), ("D3Q19", (7, 6, 5)), ("D2Q5", (9, 8))])
def test_numpy_bruteforce_with_eta_j(lat, shape):
    rng = np.random.default_rng(2)
    D = lattice_np(lat)[0]
    s = zyx(shape)
    tau = [0.7] + [0.6] * D + [0.55] * D
    p = orc.make_params(orc.INCRES, LATS[lat], shape, c0sq=1 / 36, tau=tau, powell=1.0, eta_jc=0.02)
    o = orc.Oracle(p)
    n = NpVLBM("INCRES", lat, s, tau, c0sq=1 / 36, powell=1.0, eta_jc=0.02)
    F = incres_fields(rng, D, s)
    o.init(F)
    n.init(F)
    for st in range(6):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-13, st
    # the feature was live: same run with constant eta differs
    o2 = orc.Oracle(orc.make_params(orc.INCRES, LATS[lat], shape, c0sq=1 / 36, tau=tau, powell=1.0))
    o2.init(F)
    o2.step(6)
    assert np.abs(o2.populations() - o.populations()).max() > 1e-6


def test_local_current_estimator_and_small_current_limit():
    """a / tau_B ~ |curl B| (central differences) on a smooth field; for j << j_c the run equals the constant-eta run"""
    rng = np.random.default_rng(3)
    nx, ny = 64, 48
    Bx, By = curl_h(smooth_potential(rng, ny, nx))
    sc = 0.05 / max(np.abs(Bx).max(), np.abs(By).max())
    Bx, By = sc * Bx, sc * By
    F = np.stack([0 * Bx, 0 * Bx, 0 * Bx, Bx, By])[:, None]
    tau = [0.6, 0.6, 0.6, 0.8, 0.8]
    big = orc.Oracle(orc.make_params(orc.INCRES, orc.D2Q9, (nx, ny), c0sq=1 / 36, tau=tau, powell=0.0, eta_jc=1e3))
    ref = orc.Oracle(orc.make_params(orc.INCRES, orc.D2Q9, (nx, ny), c0sq=1 / 36, tau=tau, powell=0.0))
    for o in (big, ref):
        o.init(F)
        o.step(10)
    assert np.abs(big.populations() - ref.populations()).max() < 1e-9          # (j/jc)^2 ~ 1e-11
    # estimator: rebuild a2 from the oracle's populations in numpy and compare a/tau with the curl
    g = ref.populations()
    D, c, w, cs2 = lattice_np("D2Q9")
    f = np.stack([np.roll(np.roll(g[:, i, 0], c[i][0], axis=2), c[i][1], axis=1) for i in range(9)], axis=1)   # pulled
    Q = f.sum(1)
    Pxy = np.tensordot(c[:, 0].astype(float), f[4], axes=([0], [0])) - (Q[1] * Q[4] - Q[3] * Q[2])   # N_{x,By}
    Pyx = np.tensordot(c[:, 1].astype(float), f[3], axes=([0], [0])) - (Q[2] * Q[3] - Q[4] * Q[1])   # N_{y,Bx}
    j_est = -(Pxy - Pyx) / (0.8 * cs2)
    j_cd = (np.roll(Q[4], -1, 1) - np.roll(Q[4], 1, 1)) / 2 - (np.roll(Q[3], -1, 0) - np.roll(Q[3], 1, 0)) / 2
    assert np.abs(j_cd).max() > 1e-3
    assert np.abs(j_est - j_cd).max() < 0.03 * np.abs(j_cd).max()
