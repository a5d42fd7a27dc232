"""Pins of the IDEAL_DIVB scheme (reading A19): the paper's local gradient evolution
in its traced form — one extra set D = tr G with flux D u - B and source -D/tau_M, so that D ~ tau_M div B (Eq.7) —
feeding the Powell source (Eq.12) instead of the tr Pi_B estimator."""
import numpy as np
import pytest

from oracle import oracle as orc
from np_vlbm import NpVLBM, lattice_np
from test_oracle_pins import LATS, zyx, admissible_ideal, ideal_fields

G = 5 / 3


def divb_fields(rng, s, amp=0.2):
    rho, u, B, p = admissible_ideal(rng, s, amp=amp)
    F = ideal_fields(rho, u, B, p, G)
    return np.concatenate([F, 0.05 * (rng.random((1,) + s) - 0.5)])


def test_flux_row_and_equilibrium_moments():
    rng = np.random.default_rng(1)
    for lat in ("D1Q3", "D2Q9", "D3Q19", "D3Q7"):
        D, Q, c, w, cs2 = orc.lattice(LATS[lat])
        p = orc.make_params(orc.IDEAL_DIVB, LATS[lat], (4,) * D, gamma=G, tau_relax=20.0)
        Qv = divb_fields(rng, (1, 1, 1), amp=1.0).reshape(9)
        Phi = orc.flux(p, Qv)
        u = Qv[1:4] / Qv[0]
        want = Qv[8] * u - Qv[5:8]
        want[D:] = 0
        assert np.allclose(Phi[8], want, rtol=0, atol=1e-15)            # Eq.10 traced: D u - B
        p8 = orc.make_params(orc.IDEAL, LATS[lat], (4,) * D, gamma=G)
        assert np.array_equal(Phi[:8], orc.flux(p8, Qv[:8]))            # the ideal rows are untouched
        feq = orc.equilibrium(p, Qv)
        assert np.abs(feq.sum(1) - Qv).max() < 1e-15 and np.abs(feq @ c.astype(float) - Phi).max() < 1e-15


@pytest.mark.parametrize("lat,shape,bc", [("D2Q9", (7, 6), (0,) * 6), ("D3Q19", (6, 5, 4), (2, 1, 1, 1, 0, 0)), ("D1Q3", (9,), (1, 1, 0, 0, 0, 0))])
def test_numpy_bruteforce(lat, shape, bc):
    rng = np.random.default_rng(2)
    s = zyx(shape)
    tau = [0.7] * 5 + [0.8] * 3 + [0.9]
    p = orc.make_params(orc.IDEAL_DIVB, LATS[lat], shape, gamma=G, tau=tau, powell=1.0, bc=bc, tau_relax=7.5)
    mask = np.zeros(s, dtype=np.uint8)
    mask.reshape(-1)[rng.choice(mask.size, 2, replace=False)] = 2
    o = orc.Oracle(p, mask=mask)
    n = NpVLBM("IDEAL_DIVB", lat, s, tau, gamma=G, powell=1.0, bc=bc, mask=mask, tau_relax=7.5)
    us, Bs = np.array([0.03, -0.02, 0.01]), 0.1 * (rng.random((3,) + s) - 0.5)
    o.set_obstacle(mask, us, Bs)
    n.u_solid, n.B_solid = us, Bs
    F = divb_fields(rng, s)
    o.init(F)
    n.init(F)
    for st in range(6):
        o.step(1)
        n.step(1)
        assert np.abs(o.populations() - n.g).max() < 1e-14, st
    assert np.abs(o.source_log() - n.src_acc).max() < 1e-13
    assert abs(n.src_acc[8]) > 1e-6 and np.abs(n.src_acc[1:4]).max() > 1e-9       # relaxation and Powell rows were live


def test_D_relaxes_to_tauM_divB():
    """Eq.7: with a weak, frozen-in non-solenoidal B_x(x) (1D: B_x never changes), D -> tau_M dB_x/dx."""
    nx, tauM, b, m = 256, 15.0, 1e-4, 2
    k = 2 * np.pi * m / nx
    x = np.arange(nx)
    one = np.ones((1, 1, nx))
    B = np.stack([b * np.sin(k * x)[None, None, :] * one, 0 * one, 0 * one])
    F = np.concatenate([ideal_fields(one, np.zeros((3, 1, 1, nx)), B, 0.03 * one, G), 0 * one[None]])
    p = orc.make_params(orc.IDEAL_DIVB, orc.D1Q3, (nx,), gamma=G, tau=0.6, powell=0.0, tau_relax=tauM)
    o = orc.Oracle(p)
    o.init(F)
    o.step(int(12 * tauM))
    Q = o.moments(diag=False)
    # B_x has no flux in 1D: the mode only decays slowly by the stabilising diffusion; D follows the CURRENT gradient
    amp = 2 * (Q[5][0, 0] * np.sin(k * x)).mean()
    assert 0.97 * b < amp < b and np.abs(Q[5][0, 0] - amp * np.sin(k * x)).max() < 1e-3 * b
    # lbmhd/oracle moments are POST-collision: D_post = D_pre (1 - 1/tau_M) with D_pre = tau_M dB_x/dx, the value the
    # Powell source divides by tau_M.  So the stored D is (tau_M - 1) dB_x/dx.
    want = (tauM - 1.0) * amp * k * np.cos(k * x)
    assert np.abs(Q[8][0, 0] - want).max() < 0.003 * np.abs(want).max()


def test_uniform_state_invariant_and_D_decays():
    shape = (8, 7)
    s = zyx(shape)
    one = np.ones(s)
    F8 = ideal_fields(1.3 * one, np.array([0.05, -0.03, 0.02]).reshape(3, 1, 1, 1) * one,
                      np.array([0.04, 0.06, -0.02]).reshape(3, 1, 1, 1) * one, 0.03 * one, G)
    F = np.concatenate([F8, 0.01 * one[None]])
    p = orc.make_params(orc.IDEAL_DIVB, orc.D2Q9, shape, gamma=G, tau=0.6, powell=0.0, tau_relax=10.0)
    o = orc.Oracle(p)
    o.init(F)
    o.step(30)
    Q = o.moments(diag=False)
    assert np.abs(Q[:8] - F8).max() < 1e-13
    assert np.allclose(Q[8], 0.01 * (1 - 1 / 10.0) ** 30, rtol=1e-12)        # explicit injection: D <- D (1 - 1/tau_M) per step
