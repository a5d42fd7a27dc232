"""ctypes front end of oracle/vlbm_oracle.c (argument marshalling only; the arithmetic is in the C file).

TEST INFRASTRUCTURE ONLY — see oracle/vlbm_oracle.h.  Cites: PAPER.md Eq.2-5, 8, 11-14; SURVEY.md §8c.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "vlbm_oracle.c")
_HDR = os.path.join(_HERE, "vlbm_oracle.h")

D1Q3, D2Q9, D3Q19, D2Q5, D3Q7 = 1, 2, 3, 4, 5
IDEAL, INCRES, IDEAL_DIVB, RESIST, FULL = 0, 1, 2, 3, 4
BC_PERIODIC, BC_ZEROGRAD, BC_INFLOW = 0, 1, 2
CELL_FLUID, CELL_FROZEN, CELL_SOLID = 0, 1, 2


def build(force=False):
    """gcc -O2 -ffp-contract=off -fopenmp: no FMA contraction, plain evaluation order."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _SO
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-Wall", "-shared", "-fPIC", _SRC, "-o", _SO, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class OracleParams(C.Structure):
    _fields_ = [("scheme", C.c_int), ("lattice", C.c_int),
                ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("gamma", C.c_double), ("c0sq", C.c_double),
                ("nu", C.c_double), ("eta", C.c_double),
                ("tau", C.c_double * 32), ("tau_relax", C.c_double), ("eta_jc", C.c_double), ("powell", C.c_double), ("bc", C.c_int * 6)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_SO)
        dp, ip, up = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_ubyte)
        pp = C.POINTER(OracleParams)
        lib.oracle_create.argtypes = [pp, up, C.POINTER(C.c_void_p)]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_destroy.restype = None
        lib.oracle_init.argtypes = [C.c_void_p, dp]
        lib.oracle_step.argtypes = [C.c_void_p, C.c_int]
        lib.oracle_moments.argtypes = [C.c_void_p, dp, dp]
        lib.oracle_set_obstacle.argtypes = [C.c_void_p, up, dp, dp]
        lib.oracle_set_sphere.argtypes = [C.c_void_p, dp, C.c_double, dp, dp, C.c_double]
        lib.oracle_set_porosity.argtypes = [C.c_void_p, dp]
        lib.oracle_set_sphere_width.argtypes = [C.c_void_p, C.c_double]
        lib.oracle_set_sphere_rotation.argtypes = [C.c_void_p, dp]
        lib.oracle_get_populations.argtypes = [C.c_void_p, dp]
        lib.oracle_set_populations.argtypes = [C.c_void_p, dp]
        lib.oracle_source_log.argtypes = [C.c_void_p, dp]
        lib.oracle_set_sphere_dipoles.argtypes = [C.c_void_p, C.c_int, dp, dp, dp, dp]
        lib.oracle_set_obstacle_rotation.argtypes = [C.c_void_p, dp, dp]
        lib.oracle_body_read.argtypes = [C.c_void_p, dp, C.c_int]
        lib.oracle_set_body_reference.argtypes = [C.c_void_p, dp]
        lib.oracle_lattice.argtypes = [C.c_int, ip, ip, ip, dp, dp]
        lib.oracle_flux.argtypes = [pp, dp, dp]
        lib.oracle_equilibrium.argtypes = [pp, dp, dp]
        lib.oracle_num_vars.argtypes = [pp]
        lib.oracle_num_dirs.argtypes = [pp]
        lib.oracle_tau_of_current.argtypes = [C.c_double] * 4
        lib.oracle_tau_of_current.restype = C.c_double
        lib.oracle_set_threads.argtypes = [C.c_int]
        lib.oracle_set_threads.restype = None
        lib.oracle_get_threads.restype = C.c_int
        _lib = lib
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def make_params(scheme, lattice, shape, gamma=5.0 / 3.0, c0sq=1.0 / 12.0, nu=0.0, eta=0.0, tau=0.6,
                powell=1.0, bc=(0, 0, 0, 0, 0, 0), tau_relax=0.0, eta_jc=0.0):
    """shape = (nx,), (nx, ny) or (nx, ny, nz)."""
    p = OracleParams()
    p.scheme, p.lattice = scheme, lattice
    dims = list(shape) + [1] * (3 - len(shape))
    p.nx, p.ny, p.nz = dims
    p.gamma, p.c0sq, p.nu, p.eta, p.powell = gamma, c0sq, nu, eta, powell
    taus = [tau] * 32 if np.isscalar(tau) else list(tau) + [0.0] * (32 - len(tau))
    for k in range(32):
        p.tau[k] = taus[k]
    p.tau_relax = tau_relax
    p.eta_jc = eta_jc
    for j in range(6):
        p.bc[j] = bc[j]
    return p


def lattice(lat):
    """-> (D, Q, c[Q,3] int, w[Q], cs2)"""
    lib = _load()
    D, Q = C.c_int(), C.c_int()
    c = np.zeros((19, 3), dtype=np.int32)
    w = np.zeros(19)
    cs2 = C.c_double()
    if lib.oracle_lattice(lat, C.byref(D), C.byref(Q), c.ctypes.data_as(C.POINTER(C.c_int)), _dptr(w), C.byref(cs2)):
        raise ValueError("bad lattice")
    return D.value, Q.value, c[:Q.value].copy(), w[:Q.value].copy(), cs2.value


def flux(params, Qv):
    lib = _load()
    K = lib.oracle_num_vars(C.byref(params))
    Qv = _f64(Qv)
    out = np.zeros((K, 3))
    lib.oracle_flux(C.byref(params), _dptr(Qv), _dptr(out))
    return out


def equilibrium(params, Qv):
    lib = _load()
    K, Q = lib.oracle_num_vars(C.byref(params)), lib.oracle_num_dirs(C.byref(params))
    Qv = _f64(Qv)
    out = np.zeros((K, Q))
    lib.oracle_equilibrium(C.byref(params), _dptr(Qv), _dptr(out))
    return out


def tau_of_current(tau0, e0, a2, jc):
    return float(_load().oracle_tau_of_current(tau0, e0, a2, jc))


def set_threads(n):
    _load().oracle_set_threads(int(n))


def get_threads():
    return int(_load().oracle_get_threads())


class Oracle:
    """Thin handle wrapper.  Fields are numpy [K, nz, ny, nx] float64."""

    def __init__(self, params, mask=None):
        self.lib = _load()
        self.params = params
        self.K = self.lib.oracle_num_vars(C.byref(params))
        self.Q = self.lib.oracle_num_dirs(C.byref(params))
        self.shape = (params.nz, params.ny, params.nx)
        self.N = params.nx * params.ny * params.nz
        h = C.c_void_p()
        m = None
        if mask is not None:
            self._mask = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
            assert self._mask.size == self.N
            m = self._mask.ctypes.data_as(C.POINTER(C.c_ubyte))
        rc = self.lib.oracle_create(C.byref(params), m, C.byref(h))
        if rc:
            raise ValueError("oracle_create failed: %d" % rc)
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.oracle_destroy(self.h)
            self.h = None

    __del__ = close

    def init(self, fields):
        f = _f64(fields).reshape(self.K, -1)
        assert f.shape[1] == self.N
        if self.lib.oracle_init(self.h, _dptr(f)):
            raise RuntimeError("oracle_init")

    def step(self, n=1):
        if self.lib.oracle_step(self.h, int(n)):
            raise RuntimeError("oracle_step")

    def moments(self, diag=True):
        out = np.zeros((self.K,) + self.shape)
        dg = np.zeros(3 * self.K + 4)
        if self.lib.oracle_moments(self.h, _dptr(out), _dptr(dg) if diag else None):
            raise RuntimeError("oracle_moments")
        return (out, dg) if diag else out

    def set_obstacle(self, mask, u_solid=(0.0, 0.0, 0.0), B_solid=None):
        m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
        u = _f64(u_solid)
        b = None if B_solid is None else _f64(B_solid).reshape(3, -1)
        rc = self.lib.oracle_set_obstacle(self.h, m.ctypes.data_as(C.POINTER(C.c_ubyte)), _dptr(u),
                                          None if b is None else _dptr(b))
        if rc:
            raise RuntimeError("oracle_set_obstacle")

    def set_sphere(self, centre, radius, u_solid, dipole_dir, B_surface):
        c, u, m = _f64(centre), _f64(u_solid), _f64(dipole_dir)
        if self.lib.oracle_set_sphere(self.h, _dptr(c), float(radius), _dptr(u), _dptr(m), float(B_surface)):
            raise RuntimeError("oracle_set_sphere")

    def set_porosity(self, d_field):
        d = None if d_field is None else _f64(d_field).reshape(-1)
        if self.lib.oracle_set_porosity(self.h, None if d is None else _dptr(d)):
            raise RuntimeError("oracle_set_porosity")

    def set_sphere_width(self, eps):
        if self.lib.oracle_set_sphere_width(self.h, float(eps)):
            raise RuntimeError("oracle_set_sphere_width")

    def set_sphere_rotation(self, omega):
        om = _f64(omega)
        if self.lib.oracle_set_sphere_rotation(self.h, _dptr(om)):
            raise RuntimeError("oracle_set_sphere_rotation")

    def set_sphere_dipoles(self, offsets, dirs, B_surface, cores):
        off, m, bs, co = _f64(offsets).reshape(-1, 3), _f64(dirs).reshape(-1, 3), _f64(B_surface).reshape(-1), _f64(cores).reshape(-1)
        if self.lib.oracle_set_sphere_dipoles(self.h, len(bs), _dptr(off), _dptr(m), _dptr(bs), _dptr(co)):
            raise RuntimeError("oracle_set_sphere_dipoles")

    def set_obstacle_rotation(self, omega, centre):
        om, c = _f64(omega), _f64(centre)
        if self.lib.oracle_set_obstacle_rotation(self.h, _dptr(om), _dptr(c)):
            raise RuntimeError("oracle_set_obstacle_rotation")

    def populations(self):
        g = np.zeros((self.K, self.Q) + self.shape)
        self.lib.oracle_get_populations(self.h, _dptr(g))
        return g

    def set_populations(self, g):
        g = _f64(g)
        assert g.size == self.K * self.Q * self.N
        self.lib.oracle_set_populations(self.h, _dptr(g))

    def source_log(self):
        acc = np.zeros(self.K)
        self.lib.oracle_source_log(self.h, _dptr(acc))
        return acc

    def body_read(self, reset=False):
        """body integrals accumulated since init / the last reset: F[3] | T[3] | W | I_B[3] | sum (1-d) B [3] | sum (1-d)"""
        out = np.zeros(14)
        assert self.lib.oracle_body_read(self.h, _dptr(out), int(reset)) == 0
        return out

    def set_body_reference(self, ref):
        ref = np.ascontiguousarray(ref, dtype=np.float64)
        assert self.lib.oracle_set_body_reference(self.h, _dptr(ref)) == 0


LATTICES = {"D1Q3": D1Q3, "D2Q9": D2Q9, "D3Q19": D3Q19, "D2Q5": D2Q5, "D3Q7": D3Q7}
SCHEMES = {"IDEAL": IDEAL, "INCRES": INCRES, "IDEAL_DIVB": IDEAL_DIVB, "RESIST": RESIST, "FULL": FULL}


def from_workload(w, mask=None):
    """Oracle handle configured (boundaries, tau, sphere) for an input-recipe dict (keys: scheme, lattice, shape, gamma,
    c0sq, nu, eta, tau, powell, bc, optional tau_relax, eta_jc, sphere); fields not yet initialised.  Marshalling only."""
    p = make_params(SCHEMES[w["scheme"]], LATTICES[w["lattice"]], w["shape"],
                    gamma=w["gamma"] or 1.4, c0sq=w["c0sq"], nu=w["nu"], eta=w["eta"], tau=w["tau"],
                    powell=w["powell"], bc=w["bc"], tau_relax=w.get("tau_relax", 0.0), eta_jc=w.get("eta_jc", 0.0))
    o = Oracle(p, mask=mask)
    if w.get("sphere"):
        s = w["sphere"]
        o.set_sphere(s["centre"], s["radius"], s["u_solid"], s["dipole_dir"], s["B_surface"])
        if s.get("width"):
            o.set_sphere_width(s["width"])
        if s.get("omega") is not None:
            o.set_sphere_rotation(s["omega"])
        if s.get("dipoles"):
            dp = s["dipoles"]
            o.set_sphere_dipoles(dp["offsets"], dp["dirs"], dp["B_surface"], dp["cores"])
    return o
