"""Seeded synthetic inputs for the five BASELINE.json configs.

This module only PREPARES INPUT ARRAYS (numpy, fp64); it holds none of the update's arithmetic and is
imported by neither the CUDA library nor the oracle: tests and bench.py hand the same arrays to both.
The inputs take the shapes, sizes and value distributions of the paper's cases (Brio-Wu PAPER.md:187,
resistive Orszag-Tang :215, compressible Orszag-Tang :231-233, MHD rotor :193, 16-Psyche showcase
:281-302) and stand in for them.  All randomness: numpy Generator(PCG64(20260641 + c)).

A workload is a dict:
  scheme 'IDEAL'|'INCRES'|'IDEAL_DIVB'|'RESIST'|'FULL', lattice 'D1Q3'|'D2Q9'|'D3Q19', shape (nx[,ny[,nz]]), gamma, c0sq, nu, eta,
  tau (scalar), powell, bc (6 ints: 0 periodic, 1 zero-gradient, 2 inflow), steps,
  fields  float64 [K, nz, ny, nx] in LATTICE units (reading A1),
  sphere  None or dict(centre, radius, u_solid, dipole_dir, B_surface).
"""
import numpy as np

SEED0 = 20260641
PERIODIC, ZEROGRAD, INFLOW = 0, 1, 2


def _rng(c):
    return np.random.Generator(np.random.PCG64(SEED0 + c))


def _ideal_Q(rho, u, B, p, gamma):
    """conserved variables from primitives (initial data only): E = p/(gamma-1) + rho|u|^2/2 + |B|^2/2"""
    E = p / (gamma - 1.0) + 0.5 * rho * (u * u).sum(0) + 0.5 * (B * B).sum(0)
    return np.concatenate([rho[None], rho[None] * u, E[None], B]).astype(np.float64)


def _fast_speed_bound(rho, u, B, p, gamma):
    a2 = gamma * p / rho
    b2 = (B * B).sum(0) / rho
    return float((np.sqrt((u * u).sum(0)) + np.sqrt(a2 + b2)).max())


def _to_lattice(rho, u, B, p, gamma, cfl):
    """A1: ideal MHD is invariant under (u, B, p, E) -> (s u, s B, s^2 p, s^2 E); s = CFL / max(|u| + c_f)."""
    s = cfl / _fast_speed_bound(rho, u, B, p, gamma)
    return rho, s * u, s * B, s * s * p, s


def config1(nx=800, steps=500, cfl=0.25, tau=0.55):
    """C1: 1D Riemann problem (Brio-Wu type), D1Q3, gamma = 2, seeded right state."""
    rng = _rng(1)
    gamma = 2.0
    rho_R, p_R = rng.uniform(0.1, 0.2), rng.uniform(0.08, 0.12)
    x = (np.arange(nx) + 0.5) / nx
    left = (x < 0.5)[None, None, :]
    rho = np.where(left, 1.0, rho_R)
    p = np.where(left, 1.0, p_R)
    B = np.stack([0.75 * np.ones_like(rho), np.where(left, 1.0, -1.0), np.zeros_like(rho)])
    u = np.zeros_like(B)
    rho, u, B, p, s = _to_lattice(rho, u, B, p, gamma, cfl)
    return dict(name="C1", scheme="IDEAL", lattice="D1Q3", shape=(nx,), gamma=gamma, c0sq=0.0, nu=0.0, eta=0.0,
                tau=tau, powell=1.0, bc=(ZEROGRAD, ZEROGRAD, 0, 0, 0, 0), steps=steps,
                fields=_ideal_Q(rho, u, B, p, gamma), sphere=None, scale=s)


def _curl_h(psi):
    """(D_y psi, -D_x psi) with the D2Q9 lattice difference D_a = sum_i w_i c_ia shift(c_i) / c_s^2
    on [y, x] arrays: its lattice divergence vanishes identically."""
    c = [(1, 0), (-1, 0), (0, 1), (0, -1), (1, 1), (-1, -1), (1, -1), (-1, 1)]
    w = [1 / 9] * 4 + [1 / 36] * 4
    Dx, Dy = np.zeros_like(psi), np.zeros_like(psi)
    for (cx, cy), wi in zip(c, w):
        sh = np.roll(np.roll(psi, -cx, axis=1), -cy, axis=0)
        Dx += 3.0 * wi * cx * sh
        Dy += 3.0 * wi * cy * sh
    return Dy, -Dx


def _fourier_potential(rng, n, nmodes=8, kmax=4):
    y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    psi = np.zeros((n, n))
    got = 0
    while got < nmodes:
        kx, ky = rng.integers(-kmax, kmax + 1, size=2)
        if 0 < kx * kx + ky * ky <= kmax * kmax:
            psi += rng.normal() * np.cos(2 * np.pi * (kx * x + ky * y) / n + rng.uniform(0, 2 * np.pi))
            got += 1
    return psi


def _config2_uB(n, rms):
    """divergence-free (in the lattice sense) u and B from 8 random Fourier modes each, |k| <= 4, rms amplitude `rms`"""
    rng = _rng(2)
    ux, uy = _curl_h(_fourier_potential(rng, n))
    Bx, By = _curl_h(_fourier_potential(rng, n))
    su = rms / np.sqrt((ux * ux + uy * uy).mean())
    sb = rms / np.sqrt((Bx * Bx + By * By).mean())
    return su * ux, su * uy, sb * Bx, sb * By


def config2(n=512, steps=1000, rms=0.05, nu=1e-3, eta=1e-3, sound=0.13, tau=0.5015, tau_relax=4.0):
    """C2 as BASELINE states it: 2D resistive MHD, D2Q9, periodic, 8 random Fourier modes |k| <= 4 with rms amplitude 0.05 in
    lattice units, nu = eta = 1e-3, 1000 steps — on the system the paper itself runs this case with: the
    full dissipative equations (scheme FULL: viscous stress and resistive terms in the FLUX, from the transported gradients)
    at low Mach number.  rho = 1, p = sound^2 rho / gamma (rms Mach 0.38), gamma = 5/3; tau = 0.5015 is the stabilisation
    (0.5e-3, half the physical diffusivity; A17 records the stability boundary found in the oracle)."""
    gamma = 5.0 / 3.0
    ux, uy, Bx, By = _config2_uB(n, rms)
    z = np.zeros((n, n))
    rho = np.ones((1, n, n))
    u = np.stack([ux, uy, z])[:, None]
    B = np.stack([Bx, By, z])[:, None]
    p = (sound * sound / gamma) * np.ones((1, n, n))
    F8 = _ideal_Q(rho, u, B, p, gamma)
    F = np.concatenate([F8, np.zeros((12,) + F8.shape[1:])])        # G and H start at 0 and relax to tau_M grad B, tau_M grad u
    return dict(name="C2", scheme="FULL", lattice="D2Q9", shape=(n, n), gamma=gamma, c0sq=0.0, nu=nu, eta=eta, tau=tau,
                powell=1.0, bc=(0,) * 6, steps=steps, fields=np.ascontiguousarray(F), sphere=None, scale=1.0, tau_relax=tau_relax)


def config2_incres(n=512, steps=1000, rms=0.02, nu=1e-3, eta=1e-3, c0sq=1.0 / 36.0, eta_jc=0.0):
    """C2 on the artificial-compressibility reading A3 (scheme INCRES: P, u, B sets; nu and eta through tau): the same recipe at
    rms 0.02 — at BASELINE's 0.05 this closure is unstable at tau = 0.503 whatever c0^2 (A17)."""
    ux, uy, Bx, By = _config2_uB(n, rms)
    F = np.stack([np.zeros_like(ux), ux, uy, Bx, By])[:, None]
    return dict(name="C2i", scheme="INCRES", lattice="D2Q9", shape=(n, n), gamma=0.0, c0sq=c0sq, nu=nu, eta=eta,
                tau=0.5 + 3.0 * nu, powell=1.0, bc=(0,) * 6, steps=steps, fields=np.ascontiguousarray(F), sphere=None,
                scale=1.0, eta_jc=eta_jc)      # eta_jc > 0: the paper's eta(j) = eta0 (1 + (j/j_c)^2), lattice units


def config3(n=1024, steps=2000, cfl=0.1, tau=0.505):
    """C3: 2D ideal compressible MHD vortex field (Orszag-Tang type), D2Q9, periodic, gamma = 5/3."""
    rng = _rng(3)
    gamma = 5.0 / 3.0
    ph = rng.uniform(0, 2 * np.pi, size=(4, 2))
    t = 2 * np.pi * (np.arange(n) + 0.5) / n
    y, x = np.meshgrid(t, t, indexing="ij")
    ux = -0.5 * sum(np.sin((k + 1) * y + ph[0, k]) for k in range(2))
    uy = +0.5 * sum(np.sin((k + 1) * x + ph[1, k]) for k in range(2))
    Bx = -0.5 * sum(np.sin((k + 1) * y + ph[2, k]) for k in range(2))
    By = +0.5 * sum(np.sin((k + 1) * x + ph[3, k]) for k in range(2))
    z = np.zeros_like(ux)
    rho = gamma * gamma * np.ones((1, n, n))
    p = gamma * np.ones((1, n, n))
    u = np.stack([ux, uy, z])[:, None]
    B = np.stack([Bx, By, z])[:, None]
    rho, u, B, p, s = _to_lattice(rho, u, B, p, gamma, cfl)
    return dict(name="C3", scheme="IDEAL", lattice="D2Q9", shape=(n, n), gamma=gamma, c0sq=0.0, nu=0.0, eta=0.0,
                tau=tau, powell=1.0, bc=(0,) * 6, steps=steps, fields=_ideal_Q(rho, u, B, p, gamma), sphere=None, scale=s)


def config4(n=2048, steps=1000, cfl=0.1, tau=0.51):
    """C4: 2D MHD rotor type, D2Q9, zero-gradient sides, gamma = 1.4, +-1 % seeded density noise."""
    rng = _rng(4)
    gamma = 1.4
    t = (np.arange(n) + 0.5) / n
    y, x = np.meshgrid(t, t, indexing="ij")
    dx, dy = x - 0.5, y - 0.5
    r = np.sqrt(dx * dx + dy * dy)
    r0, r1 = 0.1, 0.115
    taper = np.clip((r1 - r) / (r1 - r0), 0.0, 1.0)
    rho = (1.0 + 9.0 * taper) * (1.0 + 0.01 * rng.uniform(-1.0, 1.0, size=(n, n)))
    # rigid rotation (angular speed 20) inside r0, continued as taper * 20 * r0 * phi^ across the taper
    rr = np.where(r > 0, r, 1.0)
    speed = np.where(r < r0, 20.0 * r, taper * 20.0 * r0)
    ux, uy = -speed * dy / rr, speed * dx / rr
    z = np.zeros((n, n))
    u = np.stack([ux, uy, z])[:, None]
    B = np.stack([5.0 / np.sqrt(4 * np.pi) * np.ones((n, n)), z, z])[:, None]
    p = np.ones((1, n, n))
    rho, u, B, p, s = _to_lattice(rho[None], u, B, p, gamma, cfl)
    return dict(name="C4", scheme="IDEAL", lattice="D2Q9", shape=(n, n), gamma=gamma, c0sq=0.0, nu=0.0, eta=0.0,
                tau=tau, powell=1.0, bc=(ZEROGRAD,) * 4 + (0, 0), steps=steps,
                fields=_ideal_Q(rho, u, B, p, gamma), sphere=None, scale=s)


def dipole_field(shape_zyx, centre, R, mhat, Bs, dtype=np.float64, planes=None):
    """input data only: capped dipole 1/2 Bs (R / max(|r|, R/2))^3 [3 (m.r^) r^ - m] on integer cell coordinates;
    planes = global z indices to build (default: all nz)"""
    nz, ny, nx = shape_zyx
    zs = np.arange(nz) if planes is None else np.asarray(planes)
    out = np.zeros((3, len(zs), ny, nx), dtype=dtype)
    xs = np.arange(nx, dtype=np.float64) - centre[0]
    ys = np.arange(ny, dtype=np.float64) - centre[1]
    for iz, z in enumerate(zs):                           # plane by plane: bounded temporaries at full size
        rz = float(z) - centre[2]
        X, Y = np.meshgrid(xs, ys, indexing="xy")
        r2 = X * X + Y * Y + rz * rz
        rn = np.sqrt(r2)
        rc = np.maximum(rn, 0.5 * R)
        inv = np.where(rn > 0, 1.0 / np.where(rn > 0, rn, 1.0), 0.0)
        hx, hy, hz = X * inv, Y * inv, rz * inv
        mr = mhat[0] * hx + mhat[1] * hy + mhat[2] * hz
        amp = 0.5 * Bs * (R / rc) ** 3
        out[0, iz] = amp * (3 * mr * hx - mhat[0])
        out[1, iz] = amp * (3 * mr * hy - mhat[1])
        out[2, iz] = amp * (3 * mr * hz - mhat[2])
    return out


def config5(shape=(384, 256, 256), steps=500, tau=0.7, radius=None, planes=None):
    """C5: 3D supersonic flow (Mach 4) past a moving magnetised sphere, D3Q19, lattice units directly.
    planes: build the fields of these global z planes only (slab decomposition: each rank makes its own slab)."""
    rng = _rng(5)
    gamma = 5.0 / 3.0
    nx, ny, nz = shape
    a = 0.04
    p0 = a * a * 1.0 / gamma
    R = float(radius) if radius is not None else 24.0 * ny / 256.0
    centre = np.array([nx / 3.0, ny / 2.0, nz / 2.0])
    m = rng.normal(size=3)
    mhat = m / np.linalg.norm(m)
    Bs = 0.03
    F = np.empty((8, nz if planes is None else len(planes), ny, nx), dtype=np.float64)
    B = dipole_field((nz, ny, nx), centre, R, mhat, Bs, planes=planes)
    B[2] += 0.1 * a / np.sqrt(gamma)
    ux = 4.0 * a
    F[0] = 1.0
    F[1] = ux
    F[2] = 0.0
    F[3] = 0.0
    F[5:8] = B
    F[4] = p0 / (gamma - 1.0) + 0.5 * ux * ux + 0.5 * (B * B).sum(0)
    sphere = dict(centre=centre, radius=R, u_solid=np.array([-0.02, 0.0, 0.0]), dipole_dir=mhat, B_surface=Bs)
    return dict(name="C5", scheme="IDEAL", lattice="D3Q19", shape=tuple(shape), gamma=gamma, c0sq=0.0, nu=0.0, eta=0.0,
                tau=tau, powell=1.0, bc=(INFLOW, ZEROGRAD, 0, 0, 0, 0), steps=steps, fields=F, sphere=sphere, scale=1.0)


def variant(w, scheme=None, lattice=None, tau_relax=8.0, eta=1e-3, mu=1e-3):
    """the same input on another scheme of the IDEAL family or on the paper's own lattice (DESIGN.md §0 NEXT rows):
    IDEAL_DIVB adds D = tr G (1 set), RESIST adds G_ab (3 D sets), FULL adds G_ab and H_ab (6 D sets), all started at 0 (they relax to tau_M grad B in
    ~tau_M steps, Eq.7); D2Q5 / D3Q7 replace D2Q9 / D3Q19."""
    w = dict(w)
    if scheme is not None and scheme != w["scheme"]:
        if w["scheme"] != "IDEAL" or scheme not in ("IDEAL_DIVB", "RESIST", "FULL"):
            raise ValueError("variant: %s -> %s" % (w["scheme"], scheme))
        D = len(w["shape"])
        extra = 1 if scheme == "IDEAL_DIVB" else (3 * D if scheme == "RESIST" else 6 * D)
        w["fields"] = np.concatenate([w["fields"], np.zeros((extra,) + w["fields"].shape[1:])])
        w["scheme"], w["tau_relax"] = scheme, tau_relax
        if scheme in ("RESIST", "FULL"):
            w["eta"] = eta
        if scheme == "FULL":
            w["nu"] = mu
    if lattice is not None and lattice != w["lattice"]:
        if lattice[:2] != w["lattice"][:2]:
            raise ValueError("variant: %s -> %s" % (w["lattice"], lattice))
        w["lattice"] = lattice
    return w


def get(name, small=False):
    """the five configs (and C2i, config 2 on the INCRES reading); small=True gives the reduced sizes the oracle finishes in seconds."""
    if name == "C1":
        return config1()
    if name == "C2":
        return config2(n=128 if small else 512)
    if name == "C2i":
        return config2_incres(n=128 if small else 512)
    if name == "C3":
        return config3(n=160 if small else 1024)
    if name == "C4":
        return config4(n=200 if small else 2048)
    if name == "C5":
        return config5(shape=(96, 64, 64) if small else (384, 256, 256))
    raise KeyError(name)
