"""A second, independent writing of the VLBM step (Eq.2-4, 8, 11-14):
array-at-a-time numpy with np.roll streaming, no per-cell loop.  It exists only to pin the C oracle
(pin P6) — two writings of the same equations by different routes must agree to round-off.
Everything here is typed from the paper's formulas in tensor form (outer products, traces), not
from oracle/vlbm_oracle.c.
"""
import numpy as np

PERIODIC, ZEROGRAD, INFLOW = 0, 1, 2
FLUID, FROZEN, SOLID = 0, 1, 2


def lattice_np(name):
    """velocities [Q, 3] and weights [Q] built from shells, then ordered as reading A2."""
    if name == "D1Q3":
        c = [(0, 0, 0), (1, 0, 0), (-1, 0, 0)]
        w = [2 / 3, 1 / 6, 1 / 6]
        D = 1
    elif name == "D2Q9":
        c = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0),
             (1, 1, 0), (-1, -1, 0), (1, -1, 0), (-1, 1, 0)]
        w = [4 / 9] + [1 / 9] * 4 + [1 / 36] * 4
        D = 2
    elif name == "D3Q19":
        c = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
        for (a, b) in ((0, 1), (0, 2), (1, 2)):
            for (sa, sb) in ((1, 1), (-1, -1), (1, -1), (-1, 1)):
                v = [0, 0, 0]
                v[a], v[b] = sa, sb
                c.append(tuple(v))
        w = [1 / 3] + [1 / 18] * 6 + [1 / 36] * 12
        D = 3
    elif name == "D2Q5":
        c = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0)]
        w = [1 / 3] + [1 / 6] * 4
        D = 2
    elif name == "D3Q7":
        c = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
        w = [1 / 4] + [1 / 8] * 6
        D = 3
    else:
        raise ValueError(name)
    c = np.array(c, dtype=int)
    w = np.array(w, dtype=float)
    cs2 = float((w * c[:, 0] ** 2).sum())
    return D, c, w, cs2


def flux_ideal(Q, gamma, D):
    """Eq.11 in tensor form. Q: [8, ...] -> Phi [8, 3, ...] (axes >= D are zero)."""
    rho, m, E, B = Q[0], Q[1:4], Q[4], Q[5:8]
    u = m / rho
    B2 = (B * B).sum(0)
    p = (gamma - 1.0) * (E - 0.5 * (m * u).sum(0) - 0.5 * B2)     # Eq.8
    pt = p + 0.5 * B2
    uB = (u * B).sum(0)
    Phi = np.zeros((8, 3) + Q.shape[1:])
    eye = np.eye(3).reshape((3, 3) + (1,) * (Q.ndim - 1))
    Phi[0] = m
    Phi[1:4] = m[:, None] * u[None, :] + pt[None, None] * eye - B[:, None] * B[None, :]   # [beta, alpha]
    Phi[4] = (E + pt)[None] * u - B * uB[None]
    Phi[5:8] = u[None, :] * B[:, None] - B[None, :] * u[:, None]                           # [beta, alpha]
    Phi[:, D:] = 0.0
    return Phi


def flux_ideal_divb(Q, gamma, D):
    """IDEAL plus the traced gradient variable D = tr G of PAPER.md:104-138: flux D u - B (Eq.10 traced)."""
    Phi = np.zeros((9, 3) + Q.shape[1:])
    Phi[:8] = flux_ideal(Q[:8], gamma, D)
    u = Q[1:4] / Q[0]
    Phi[8] = Q[8][None] * u - Q[5:8]
    Phi[8, D:] = 0.0
    return Phi


LEVI = np.zeros((3, 3, 3))
for _a, _b, _c in ((0, 1, 2), (1, 2, 0), (2, 0, 1)):
    LEVI[_a, _b, _c], LEVI[_a, _c, _b] = 1.0, -1.0


def flux_resist(Q, gamma, D, eta, tau_m):
    """dissipative system with transported gradients G (Eq.9-10): Q = (rho, m, E, B, G[a<D][b<3]).
    Tensor form: g = G / tau_M ~ grad B; j = curl B = eps : g; Phi_B -= eta g; Phi_E += eta j x B; Phi_G = G (x) u - I (x) B."""
    K = 8 + 3 * D
    tail = Q.shape[1:]
    Phi = np.zeros((K, 3) + tail)
    Phi[:8] = flux_ideal(Q[:8], gamma, D)
    u, B = Q[1:4] / Q[0], Q[5:8]
    G = np.zeros((3, 3) + tail)
    G[:D] = Q[8:].reshape((D, 3) + tail)
    g = G / tau_m
    j = np.einsum("ecb,cb...->e...", LEVI, g)
    jxB = np.einsum("aef,e...,f...->a...", LEVI, j, B)
    Phi[4] += eta * jxB
    Phi[5:8] -= eta * np.swapaxes(g, 0, 1)                      # Phi[5+b, a] -= eta g[a, b]
    PhiG = G[:, :, None] * u[None, None] - np.einsum("ca,b...->cba...", np.eye(3), B)     # [c, b, a]
    Phi[8:] = PhiG[:D].reshape((3 * D, 3) + tail)
    Phi[:, D:] = 0.0
    return Phi


def flux_full(Q, gamma, D, eta, mu, tau_m):
    """full dissipative system of PAPER.md:122 with transported gradients of B and of u (Eq.9; reading A23):
    Q = (rho, m, E, B, G[a<D][b<3], H[a<D][b<3]), h = H / tau_M ~ grad u, sigma = mu (h + h^T - 2/3 tr h I);
    Phi_m -= sigma; Phi_E -= u . sigma; Phi_H = H (x) u - I (x) u."""
    K = 8 + 6 * D
    tail = Q.shape[1:]
    Phi = np.zeros((K, 3) + tail)
    Phi[:8 + 3 * D] = flux_resist(Q[:8 + 3 * D], gamma, D, eta, tau_m)
    u = Q[1:4] / Q[0]
    H = np.zeros((3, 3) + tail)
    H[:D] = Q[8 + 3 * D:].reshape((D, 3) + tail)
    h = H / tau_m
    eye = np.eye(3).reshape((3, 3) + (1,) * len(tail))
    sigma = mu * (h + np.swapaxes(h, 0, 1) - (2.0 / 3.0) * np.einsum("cc...->...", h)[None, None] * eye)      # [a, b]
    Phi[1:4] -= np.swapaxes(sigma, 0, 1)                         # Phi[1+b, a] -= sigma[a, b]
    Phi[4] -= np.einsum("b...,ab...->a...", u, sigma)
    PhiH = H[:, :, None] * u[None, None] - np.einsum("ca,b...->cba...", np.eye(3), u)     # [c, b, a]
    Phi[8 + 3 * D:] = PhiH[:D].reshape((3 * D, 3) + tail)
    Phi[:, D:] = 0.0
    return Phi


def flux_incres(Q, c0sq, D):
    """A3. Q: [1+2D, ...] = (P, u, B)."""
    P, u, B = Q[0], Q[1:1 + D], Q[1 + D:1 + 2 * D]
    B2 = (B * B).sum(0)
    Phi = np.zeros((1 + 2 * D, 3) + Q.shape[1:])
    eye = np.eye(D).reshape((D, D) + (1,) * (Q.ndim - 1))
    Phi[0, :D] = c0sq * u
    Phi[1:1 + D, :D] = u[:, None] * u[None, :] + (P + 0.5 * B2)[None, None] * eye - B[:, None] * B[None, :]
    Phi[1 + D:, :D] = u[None, :] * B[:, None] - B[None, :] * u[:, None]
    return Phi


class NpVLBM:
    """fields / populations are indexed [k, (i,) z, y, x]."""

    def __init__(self, scheme, lat, shape_zyx, tau, gamma=5 / 3, c0sq=1 / 12, powell=1.0,
                 bc=(0,) * 6, mask=None, tau_relax=0.0, eta_jc=0.0):
        self.scheme = scheme
        self.D, self.c, self.w, self.cs2 = lattice_np(lat)
        self.Qn = len(self.w)
        self.shape = tuple(shape_zyx)
        self.K = {"IDEAL": 8, "IDEAL_DIVB": 9, "RESIST": 8 + 3 * self.D, "FULL": 8 + 6 * self.D, "INCRES": 1 + 2 * self.D}[scheme]
        self.ideal = scheme in ("IDEAL", "IDEAL_DIVB", "RESIST", "FULL")
        self.eta = 0.0                 # RESIST, FULL: magnetic diffusivity of the flux terms
        self.mu = 0.0                  # FULL: shear viscosity of the flux terms
        self.tau_relax = tau_relax
        self.eta_jc = eta_jc
        self.tau = np.broadcast_to(np.asarray(tau, dtype=float), (self.K,)).copy()
        self.gamma, self.c0sq, self.kappa = gamma, c0sq, powell
        self.bc = tuple(bc)
        self.iB = 5 if self.ideal else 1 + self.D
        self.mask = np.zeros(self.shape, dtype=np.uint8) if mask is None else np.asarray(mask, dtype=np.uint8).reshape(self.shape)
        self.u_solid = np.zeros(3)
        self.B_solid = None
        self.sphere = None
        self.sphere_eps = 0.0
        self.sphere_omega = np.zeros(3)
        self.d_field = None
        self.dipoles = None            # [(offset[3], axis[3], B_surface, core)] in the body frame, replaces the sphere's own dipole
        self.obst_omega, self.obst_centre = np.zeros(3), np.zeros(3)
        self.t = 0
        self.src_acc = np.zeros(self.K)
        self.body = np.zeros(14)
        self.body_ref = np.zeros(3)
        zz, yy, xx = np.meshgrid(*[np.arange(n) for n in self.shape], indexing="ij")
        self.coord = (xx, yy, zz)
        self.n_axis = (self.shape[2], self.shape[1], self.shape[0])

    def flux(self, Q):
        if self.scheme == "IDEAL":
            return flux_ideal(Q, self.gamma, self.D)
        if self.scheme == "IDEAL_DIVB":
            return flux_ideal_divb(Q, self.gamma, self.D)
        if self.scheme == "RESIST":
            return flux_resist(Q, self.gamma, self.D, self.eta, self.tau_relax)
        if self.scheme == "FULL":
            return flux_full(Q, self.gamma, self.D, self.eta, self.mu, self.tau_relax)
        return flux_incres(Q, self.c0sq, self.D)

    def feq(self, Q, Phi):
        # Eq.3: w_i (Q_k + c_i.Phi_k / cs2) -> [K, Qn, ...]
        cPhi = np.tensordot(self.c.astype(float), Phi, axes=([1], [1]))     # [Qn, K, ...]
        cPhi = np.moveaxis(cPhi, 0, 1)
        wv = self.w.reshape((1, self.Qn) + (1,) * (Q.ndim - 1))
        return wv * (Q[:, None] + cPhi / self.cs2)

    def init(self, fields):
        Q = np.asarray(fields, dtype=float).reshape((self.K,) + self.shape)
        self.g = self.feq(Q, self.flux(Q))
        self.t = 0

    def moments(self):
        return self.g.sum(1)

    # -- helpers for boundaries
    def _frozen(self):
        fr = self.mask == FROZEN
        for a in range(self.D):
            if self.bc[2 * a] == INFLOW:
                fr = fr | (self.coord[a] == 0)
            if self.bc[2 * a + 1] == INFLOW:
                fr = fr | (self.coord[a] == self.n_axis[a] - 1)
        return fr

    def _shift(self, arr, cvec):
        """arr(x - c): np.roll by +c along each axis (array axes are ..., z, y, x)."""
        out = arr
        for a in range(self.D):
            if cvec[a]:
                out = np.roll(out, int(cvec[a]), axis=arr.ndim - 1 - a)
        return out

    def _solid(self):
        """porosity d [z,y,x], uB [3,...], BB [3,...]"""
        d = np.ones(self.shape)
        uB = np.zeros((3,) + self.shape)
        BB = np.zeros((3,) + self.shape)
        if self.d_field is not None:
            d = np.asarray(self.d_field, dtype=float).reshape(self.shape).copy()
        else:
            d[self.mask == SOLID] = 0.0
        sol = d < 1.0
        if sol.any():
            rr = np.zeros(self.shape + (3,))
            for a in range(self.D):
                rr[..., a] = self.coord[a] - self.obst_centre[a]
            urot = np.cross(np.asarray(self.obst_omega, dtype=float), rr)
            for a in range(3):
                uB[a][sol] = self.u_solid[a] + urot[..., a][sol]
                if self.B_solid is not None:
                    BB[a][sol] = self.B_solid[a][sol]
        if self.sphere is not None:
            c0, R, us, mh, Bs, t0 = self.sphere
            cen = c0 + (self.t - t0) * us
            r = np.zeros((3,) + self.shape)
            for a in range(self.D):
                r[a] = self.coord[a] - cen[a]
            r2 = (r * r).sum(0)
            rn = np.sqrt(r2)
            if self.sphere_eps > 0:
                ds = np.clip((rn - R) / self.sphere_eps + 0.5, 0.0, 1.0)
            else:
                ds = np.where(r2 <= R * R, 0.0, 1.0)
            ins = ds < 1.0
            om = np.asarray(self.sphere_omega, dtype=float)
            omn = np.linalg.norm(om)

            def rot(v):                                  # Rodrigues rotation about Omega by |Omega| (t - t0)
                v = np.asarray(v, dtype=float)
                if omn == 0:
                    return v
                e, th = om / omn, omn * (self.t - t0)
                return v * np.cos(th) + np.cross(e, v) * np.sin(th) + e * (e @ v) * (1 - np.cos(th))
            urot = np.cross(om.reshape(1, 1, 1, 3), np.moveaxis(r, 0, -1))     # Omega x r
            urot = np.moveaxis(urot, -1, 0)
            ensemble = self.dipoles if self.dipoles is not None else [(np.zeros(3), mh, Bs, 0.5 * R)]
            dip = np.zeros((3,) + self.shape)
            for off, axis, bsj, core in ensemble:
                oj, mj = rot(off), rot(axis)
                rj = np.zeros((3,) + self.shape)
                for a in range(self.D):
                    rj[a] = r[a] - oj[a]
                rjn = np.sqrt((rj * rj).sum(0))
                with np.errstate(invalid="ignore", divide="ignore"):
                    rh = np.where(rjn > 0, rj / np.where(rjn > 0, rjn, 1.0), 0.0)
                mr = (mj.reshape(3, 1, 1, 1) * rh).sum(0)
                dip += 0.5 * bsj * (R / np.maximum(rjn, core)) ** 3 * (3.0 * mr * rh - mj.reshape(3, 1, 1, 1))
            d[ins] = ds[ins]
            for a in range(3):
                uB[a][ins] = us[a] + urot[a][ins]
                BB[a][ins] = dip[a][ins]
        return d, uB, BB

    def step(self, n=1):
        for _ in range(n):
            self._one()

    def _one(self):
        g = self.g
        K, Qn, D = self.K, self.Qn, self.D
        # 1. pull with periodic roll
        f = np.empty_like(g)
        for i in range(Qn):
            f[:, i] = self._shift(g[:, i], self.c[i])
        # A9: outside sources -> equilibrium of the inward neighbour's state
        nonper = [a for a in range(D) if self.bc[2 * a] != PERIODIC]
        if nonper:
            Qst = g.sum(1)
            idx = [self.coord[2], self.coord[1], self.coord[0]]      # z, y, x index arrays
            for a in nonper:
                na = self.n_axis[a]
                ia = idx[2 - a].copy()
                ia[self.coord[a] == 0] = 1
                ia[self.coord[a] == na - 1] = na - 2
                idx[2 - a] = ia
            Qnb = Qst[:, idx[0], idx[1], idx[2]]
            fnb = self.feq(Qnb, self.flux(Qnb))
            for i in range(Qn):
                out = np.zeros(self.shape, dtype=bool)
                for a in nonper:
                    s = self.coord[a] - self.c[i][a]
                    out |= (s < 0) | (s >= self.n_axis[a])
                f[:, i] = np.where(out[None], fnb[:, i], f[:, i])
        # 2. moments
        Q = f.sum(1)
        # 3. delta = -tr(Pi_B) / (tau_B cs2)
        tr = np.zeros(self.shape)
        for b in range(D):
            tr += np.tensordot(self.c[:, b].astype(float), f[self.iB + b], axes=([0], [0]))
        tauB = self.tau[self.iB] * np.ones(self.shape)
        if self.scheme == "INCRES" and self.eta_jc > 0:
            # PAPER.md:215 eta(j) = eta0 (1 + (j/jc)^2): local tau_B from the antisymmetric non-equilibrium moment (A20)
            Pieq = self.flux(Q)
            cf = self.c.astype(float)
            Nab = np.zeros((D, D) + self.shape)
            for a_ in range(D):
                for b in range(D):
                    Nab[a_, b] = np.tensordot(cf[:, a_], f[self.iB + b], axes=([0], [0])) - Pieq[self.iB + b, a_]
            a2 = np.zeros(self.shape)
            for a_ in range(D):
                for b in range(a_ + 1, D):
                    a2 += (Nab[a_, b] - Nab[b, a_]) ** 2
            a2 /= self.cs2 ** 2
            tau0 = self.tau[self.iB]
            cc = (tau0 - 0.5) * a2 / self.eta_jc ** 2
            t = tau0 + np.cbrt(cc)
            for _ in range(60):                       # converged root of t^3 - tau0 t^2 - c (the oracle does 6 Newton steps)
                t = t - ((t - tau0) * t * t - cc) / (t * (3 * t - 2 * tau0))
            tauB = t
        delta = -tr / (tauB * self.cs2)
        if self.scheme in ("RESIST", "FULL"):
            delta = sum(Q[8 + 3 * a + a] for a in range(D)) / self.tau_relax        # div B = tr G / tau_M
        if self.scheme == "IDEAL_DIVB":
            delta = Q[8] / self.tau_relax            # Eq.7: D ~ tau_M div B
        # 4. Powell source
        S = np.zeros_like(Q)
        if self.ideal:
            u = Q[1:4] / Q[0]
            B = Q[5:8]
            S[1:4] = -self.kappa * delta * B
            S[4] = -self.kappa * delta * (u * B).sum(0)
            S[5:8] = -self.kappa * delta * u
            if self.scheme in ("IDEAL_DIVB", "RESIST", "FULL"):
                S[8:] = -Q[8:] / self.tau_relax      # relaxation source of Eq.6
        else:
            u, B = Q[1:1 + D], Q[1 + D:]
            S[1:1 + D] = -self.kappa * delta * B
            S[1 + D:] = -self.kappa * delta * u
        # 5. homogenised solid
        d, uB, BB = self._solid()
        Qh = Q.copy()
        if self.ideal:
            rho = Q[0]
            u = Q[1:4] / rho
            B = Q[5:8]
            p = (self.gamma - 1.0) * (Q[4] - 0.5 * (Q[1:4] * u).sum(0) - 0.5 * (B * B).sum(0))
            uh = d * u + (1.0 - d) * uB
            Bh = d * B + (1.0 - d) * BB
            Eh = p / (self.gamma - 1.0) + 0.5 * rho * (uh * uh).sum(0) + 0.5 * (Bh * Bh).sum(0)
            sol = d < 1.0
            for b in range(3):
                Qh[1 + b] = np.where(sol, rho * uh[b], Q[1 + b])
                Qh[5 + b] = np.where(sol, Bh[b], Q[5 + b])
            Qh[4] = np.where(sol, Eh, Q[4])
        else:
            sol = d < 1.0
            for b in range(D):
                Qh[1 + b] = np.where(sol, d * Q[1 + b] + (1 - d) * uB[b], Q[1 + b])
                Qh[1 + D + b] = np.where(sol, d * Q[1 + D + b] + (1 - d) * BB[b], Q[1 + D + b])
        dQh = Qh - Q
        if self.scheme in ("IDEAL_DIVB", "RESIST", "FULL"):
            S[:8] = S[:8] * d
        else:
            S = S * d
        # 6./7. flux, BGK, injection
        feq = self.feq(Q, self.flux(Qh))
        om = (1.0 / self.tau).reshape((K, 1) + (1,) * len(self.shape)) * np.ones((K, 1) + self.shape)
        if self.scheme == "INCRES" and self.eta_jc > 0:
            om[self.iB:self.iB + D, 0] = 1.0 / tauB
        wv = self.w.reshape((1, Qn) + (1,) * len(self.shape))
        gnew = f + om * (feq - f) + wv * (dQh + S)[:, None]
        fr = self._frozen()
        if fr.any():
            gnew = np.where(fr[None, None], g, gnew)
            S = np.where(fr[None], 0.0, S)
        self.src_acc += S.reshape(K, -1).sum(1)
        # body integrals (A21): what the blend hands over at the cells with d < 1
        body_cells = (d < 1.0) & ~fr
        if body_cells.any():
            nvec = 3 if self.ideal else D
            ref = self.body_ref if self.sphere is None else self.sphere[0] + (self.t - self.sphere[5]) * self.sphere[2]
            r = np.zeros((3,) + self.shape)
            Fm = np.zeros((3,) + self.shape)
            for a in range(D):
                r[a] = self.coord[a] - ref[a]
            Fm[:nvec] = -dQh[1:1 + nvec]
            Tq = np.cross(np.moveaxis(r, 0, -1), np.moveaxis(Fm, 0, -1))
            sel = body_cells
            self.body[0:3] += Fm[:, sel].sum(1)
            self.body[3:6] += Tq[sel].sum(0)
            if self.ideal:
                self.body[6] += -dQh[4][sel].sum()
            self.body[7:7 + nvec] += dQh[self.iB:self.iB + nvec][:, sel].sum(1)
            self.body[10:10 + nvec] += ((1.0 - d) * Q[self.iB:self.iB + nvec])[:, sel].sum(1)
            self.body[13] += (1.0 - d)[sel].sum()
        self.g = gnew
        self.t += 1
