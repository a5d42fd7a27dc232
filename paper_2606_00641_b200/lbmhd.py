"""ctypes binding of the C-ABI CUDA library (include/lbmhd.h): same names, argument marshalling only.

Every step of the path runs in the library's kernels.  torch is used for device memory (the workspace
tensor), the current stream and pinned host buffers; numpy arrays are accepted for host-side fields.
There is no CPU fallback: if the shared library is missing, cannot be loaded, or no CUDA device is
present, construction raises.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

D1Q3, D2Q9, D3Q19, D2Q5, D3Q7 = 1, 2, 3, 4, 5
IDEAL, INCRES, IDEAL_DIVB, RESIST, FULL = 0, 1, 2, 3, 4
BC_PERIODIC, BC_ZEROGRAD, BC_INFLOW, BC_HALO = 0, 1, 2, 3
CELL_FLUID, CELL_FROZEN, CELL_SOLID = 0, 1, 2
STREAM_AB, STREAM_INPLACE = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ENUMERIC = 0, -1, -2, -3, -4
HALO_CROSSING, HALO_FULL, HALO_RETURN = 0, 1, 2
LATTICES = {"D1Q3": D1Q3, "D2Q9": D2Q9, "D3Q19": D3Q19, "D2Q5": D2Q5, "D3Q7": D3Q7}
SCHEMES = {"IDEAL": IDEAL, "INCRES": INCRES, "IDEAL_DIVB": IDEAL_DIVB, "RESIST": RESIST, "FULL": FULL}


class LbmhdParams(C.Structure):
    _fields_ = [("scheme", C.c_int), ("lattice", C.c_int), ("precision", C.c_int),
                ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("gamma", C.c_double), ("c0sq", C.c_double), ("nu", C.c_double), ("eta", C.c_double),
                ("tau", C.c_double * 32), ("tau_relax", C.c_double), ("eta_jc", C.c_double), ("powell", C.c_double), ("bc", C.c_int * 6),
                ("halo_offset", C.c_int), ("streaming", C.c_int), ("device", C.c_int), ("stream", C.c_void_p),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class LbmhdError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("lbmhd error %d: %s" % (code, text))
        self.code = code


_lib = None


def load_library():
    """dlopen the in-tree liblbmhd.so (it must have been built: __graft_entry__.build())."""
    global _lib
    if _lib is not None:
        return _lib
    so = os.environ.get("LBMHD_LIBRARY", _build.SO)      # another build of this library (same ABI), e.g. with other compile flags
    if not os.path.exists(so):
        raise ImportError("CUDA extension %s is missing; run __graft_entry__.build() (nvcc, sm_100a)" % so)
    lib = C.CDLL(so)
    dp, up, pp = C.c_void_p, C.c_void_p, C.POINTER(LbmhdParams)
    lib.lbmhd_num_vars.argtypes = [pp]
    lib.lbmhd_num_dirs.argtypes = [pp]
    lib.lbmhd_workspace_bytes.argtypes = [pp]
    lib.lbmhd_workspace_bytes.restype = C.c_size_t
    lib.lbmhd_create.argtypes = [pp, up, C.POINTER(C.c_void_p)]
    lib.lbmhd_destroy.argtypes = [C.c_void_p]
    lib.lbmhd_destroy.restype = None
    lib.lbmhd_init.argtypes = [C.c_void_p, dp, C.c_int]
    lib.lbmhd_step.argtypes = [C.c_void_p, C.c_int]
    lib.lbmhd_moments.argtypes = [C.c_void_p, dp, dp, C.c_int]
    lib.lbmhd_set_obstacle.argtypes = [C.c_void_p, up, dp, dp, C.c_int]
    lib.lbmhd_set_sphere.argtypes = [C.c_void_p, dp, C.c_double, dp, dp, C.c_double]
    lib.lbmhd_set_porosity.argtypes = [C.c_void_p, dp, C.c_int]
    lib.lbmhd_set_sphere_width.argtypes = [C.c_void_p, C.c_double]
    lib.lbmhd_set_sphere_rotation.argtypes = [C.c_void_p, dp]
    lib.lbmhd_halo_bytes.argtypes = [C.c_void_p, C.c_int]
    lib.lbmhd_halo_bytes.restype = C.c_size_t
    lib.lbmhd_halo_pack.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
    lib.lbmhd_halo_unpack.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
    lib.lbmhd_halo_pack_on.argtypes = [C.c_void_p, C.c_int, C.c_int, dp, C.c_int, C.c_void_p]
    lib.lbmhd_halo_unpack_on.argtypes = [C.c_void_p, C.c_int, C.c_int, dp, C.c_int, C.c_void_p]
    lib.lbmhd_step_part.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
    lib.lbmhd_diagnostics.argtypes = [C.c_void_p, dp, dp, C.c_int]
    lib.lbmhd_workspace_bytes_min.argtypes = [pp]
    lib.lbmhd_workspace_bytes_min.restype = C.c_size_t
    lib.lbmhd_get_populations.argtypes = [C.c_void_p, dp, C.c_int]
    lib.lbmhd_set_populations.argtypes = [C.c_void_p, dp, C.c_int]
    lib.lbmhd_steps_done.argtypes = [C.c_void_p]
    lib.lbmhd_steps_done.restype = C.c_longlong
    lib.lbmhd_launch_count.argtypes = [C.c_void_p]
    lib.lbmhd_launch_count.restype = C.c_longlong
    lib.lbmhd_step_path.argtypes = [C.c_void_p]
    lib.lbmhd_set_sphere_dipoles.argtypes = [C.c_void_p, C.c_int, dp, dp, dp, dp]
    lib.lbmhd_set_obstacle_rotation.argtypes = [C.c_void_p, dp, dp]
    lib.lbmhd_body_enable.argtypes = [C.c_void_p, C.c_int, dp]
    lib.lbmhd_body_read.argtypes = [C.c_void_p, dp, C.c_int, C.c_int]
    lib.lbmhd_copy_probe.argtypes = [dp, dp, C.c_size_t, C.c_int, C.c_void_p]
    lib.lbmhd_triad_probe.argtypes = [dp, dp, dp, C.c_double, C.c_size_t, C.c_int, C.c_void_p]
    lib.lbmhd_diagnostics_static.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.c_double, dp, dp, C.c_int,
                                             C.c_void_p]
    lib.lbmhd_last_error.restype = C.c_char_p
    _lib = lib
    return lib


EXPORTS = ["lbmhd_num_vars", "lbmhd_num_dirs", "lbmhd_workspace_bytes", "lbmhd_create", "lbmhd_destroy",
           "lbmhd_init", "lbmhd_step", "lbmhd_moments", "lbmhd_set_obstacle", "lbmhd_set_sphere",
           "lbmhd_set_porosity", "lbmhd_set_sphere_width", "lbmhd_set_sphere_rotation", "lbmhd_halo_bytes", "lbmhd_halo_pack",
           "lbmhd_halo_unpack", "lbmhd_get_populations", "lbmhd_set_populations", "lbmhd_steps_done", "lbmhd_launch_count",
           "lbmhd_copy_probe", "lbmhd_last_error", "lbmhd_body_enable", "lbmhd_body_read",
           "lbmhd_set_sphere_dipoles", "lbmhd_set_obstacle_rotation", "lbmhd_step_path", "lbmhd_triad_probe",
           "lbmhd_halo_pack_on", "lbmhd_halo_unpack_on", "lbmhd_step_part", "lbmhd_diagnostics", "lbmhd_workspace_bytes_min",
           "lbmhd_diagnostics_static"]


def _check(rc, allow=()):
    if rc != 0 and rc not in allow:
        raise LbmhdError(rc, load_library().lbmhd_last_error().decode())
    return rc


def make_params(scheme, lattice, shape, precision=64, gamma=5.0 / 3.0, c0sq=1.0 / 36.0, nu=0.0, eta=0.0, tau=0.6,
                powell=1.0, bc=(0,) * 6, streaming=STREAM_AB, device=0, tau_relax=0.0, eta_jc=0.0, halo_offset=0):
    p = LbmhdParams()
    p.scheme = SCHEMES.get(scheme, scheme)
    p.lattice = LATTICES.get(lattice, lattice)
    p.precision = precision
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
    p.streaming, p.device, p.halo_offset = streaming, device, halo_offset
    return p


def workspace_bytes(params, solid_fields=True):
    """device bytes a handle needs; solid_fields=False leaves out the per-cell B_solid / porosity storage"""
    lib = load_library()
    return int(lib.lbmhd_workspace_bytes(C.byref(params)) if solid_fields else lib.lbmhd_workspace_bytes_min(C.byref(params)))


def _host_ptr(a):
    return C.c_void_p(a.ctypes.data)


class Lbmhd:
    """Handle wrapper: lbmhd_create / init / step / moments / set_obstacle / set_sphere / destroy."""

    def __init__(self, params, mask=None, stream=None, solid_fields=True):
        import torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise LbmhdError(ECUDA, "no CUDA device: this library has no CPU path")
        self.torch = torch
        self.params = params
        self.K = self.lib.lbmhd_num_vars(C.byref(params))
        self.Q = self.lib.lbmhd_num_dirs(C.byref(params))
        if self.K < 0 or self.Q < 0:
            raise LbmhdError(EINVAL, "unknown scheme or lattice")
        self.shape = (params.nz, params.ny, params.nx)
        self.N = params.nx * params.ny * params.nz
        nbytes = workspace_bytes(params, solid_fields)
        if nbytes == 0:
            raise LbmhdError(EINVAL, "bad dims or precision")
        dev = torch.device("cuda", params.device)
        # LBMHD_GUARD_BYTES=n (debugging aid, tests/test_guard_gpu.py): n bytes of 0xA5 before and after the workspace, checked by
        # close(): a kernel that writes outside the memory it was given trips it (compute-sanitizer is not available everywhere)
        guard = int(os.environ.get("LBMHD_GUARD_BYTES", "0"))
        if guard:
            self.workspace = torch.full((nbytes + 256 + 2 * guard,), 0xA5, dtype=torch.uint8, device=dev)
        else:
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
        base = self.workspace.data_ptr()
        aligned = (base + guard + 255) // 256 * 256
        self._guard = (aligned - base, nbytes) if guard else None
        params.workspace = aligned
        params.workspace_bytes = nbytes
        self.stream = stream if stream is not None else torch.cuda.current_stream(dev)
        params.stream = self.stream.cuda_stream
        h = C.c_void_p()
        m = None
        if mask is not None:
            self._mask = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
            assert self._mask.size == self.N
            m = _host_ptr(self._mask)
        _check(self.lib.lbmhd_create(C.byref(params), m, C.byref(h)))
        self.h = h

    def guards_intact(self):
        """True if the guard bands around the workspace (LBMHD_GUARD_BYTES) still hold their pattern"""
        if self._guard is None or self.workspace is None:
            return True
        lo, n = self._guard
        self.torch.cuda.synchronize(self.workspace.device)
        return bool((self.workspace[:lo] == 0xA5).all().item()) and bool((self.workspace[lo + n:] == 0xA5).all().item())

    def close(self):
        if getattr(self, "h", None):
            ok = self.guards_intact() if getattr(self, "_guard", None) else True
            self.lib.lbmhd_destroy(self.h)
            self.h = None
            self.workspace = None
            if not ok:
                raise LbmhdError(ECUDA, "a kernel wrote outside the workspace (guard band damaged)")

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptr(self, a, nelem, dtype_np, dtype_torch):
        """(pointer, on_device, keepalive) for a numpy array or a torch tensor"""
        torch = self.torch
        if isinstance(a, torch.Tensor):
            assert a.dtype == dtype_torch and a.is_contiguous() and a.numel() == nelem
            return C.c_void_p(a.data_ptr()), int(a.is_cuda), a
        arr = np.ascontiguousarray(a, dtype=dtype_np)
        assert arr.size == nelem
        return _host_ptr(arr), 0, arr

    def init(self, fields):
        ptr, dev, keep = self._ptr(fields, self.K * self.N, np.float64, self.torch.float64)
        _check(self.lib.lbmhd_init(self.h, ptr, dev))

    def step(self, n=1):
        _check(self.lib.lbmhd_step(self.h, int(n)))

    def step_part(self, plane_lo, plane_hi, last):
        """one step in pieces: planes [plane_lo, plane_hi) of the slowest lattice axis; last=True completes the step"""
        _check(self.lib.lbmhd_step_part(self.h, int(plane_lo), int(plane_hi), int(bool(last))))

    def diagnostics(self, fields_dev, diag_out=None):
        """the 3K+4 diagnostics of a device fields tensor [K*N]; -> numpy array (host, synchronises) or the given device tensor"""
        assert fields_dev.is_cuda and fields_dev.dtype == self.torch.float64 and fields_dev.numel() == self.K * self.N
        if diag_out is not None:
            _check(self.lib.lbmhd_diagnostics(self.h, C.c_void_p(fields_dev.data_ptr()), C.c_void_p(diag_out.data_ptr()), 1))
            return diag_out
        dg = np.empty(3 * self.K + 4, dtype=np.float64)
        _check(self.lib.lbmhd_diagnostics(self.h, C.c_void_p(fields_dev.data_ptr()), _host_ptr(dg), 0), allow=(ENUMERIC,))
        return dg

    def moments(self, fields_out=None, diag_out=None, want_fields=True, want_diag=True, check=False):
        """-> (fields [K, nz, ny, nx], diag [3K+4]).  Host numpy by default; pass CUDA tensors to stay on device."""
        torch = self.torch
        nd = 3 * self.K + 4
        on_dev = isinstance(fields_out, torch.Tensor) and fields_out.is_cuda or isinstance(diag_out, torch.Tensor) and diag_out.is_cuda
        if on_dev:
            fp = C.c_void_p(fields_out.data_ptr()) if fields_out is not None else None
            dg = C.c_void_p(diag_out.data_ptr()) if diag_out is not None else None
            _check(self.lib.lbmhd_moments(self.h, fp, dg, 1))
            return fields_out, diag_out
        if fields_out is None and want_fields:
            fields_out = np.empty((self.K,) + self.shape, dtype=np.float64)
        if diag_out is None and want_diag:
            diag_out = np.empty(nd, dtype=np.float64)
        fp = None
        if fields_out is not None:
            fp = C.c_void_p(fields_out.data_ptr()) if isinstance(fields_out, torch.Tensor) else _host_ptr(fields_out)
        dg = None
        if diag_out is not None:
            dg = C.c_void_p(diag_out.data_ptr()) if isinstance(diag_out, torch.Tensor) else _host_ptr(diag_out)
        _check(self.lib.lbmhd_moments(self.h, fp, dg, 0), allow=() if check else (ENUMERIC,))
        return fields_out, diag_out

    def set_obstacle(self, mask, u_solid=(0.0, 0.0, 0.0), B_solid=None):
        mp, dev, k1 = self._ptr(mask, self.N, np.uint8, self.torch.uint8)
        u = np.ascontiguousarray(u_solid, dtype=np.float64)
        bp, k2 = None, None
        if B_solid is not None:
            bp, dev2, k2 = self._ptr(B_solid, 3 * self.N, np.float64, self.torch.float64)
            assert dev2 == dev
        _check(self.lib.lbmhd_set_obstacle(self.h, mp, _host_ptr(u), bp, dev))

    def set_sphere(self, centre, radius, u_solid, dipole_dir, B_surface):
        c = np.ascontiguousarray(centre, dtype=np.float64)
        u = np.ascontiguousarray(u_solid, dtype=np.float64)
        m = np.ascontiguousarray(dipole_dir, dtype=np.float64)
        _check(self.lib.lbmhd_set_sphere(self.h, _host_ptr(c), float(radius), _host_ptr(u), _host_ptr(m), float(B_surface)))

    def set_porosity(self, d_field):
        if d_field is None:
            _check(self.lib.lbmhd_set_porosity(self.h, None, 0))
            return
        dp_, dev, keep = self._ptr(d_field, self.N, np.float64, self.torch.float64)
        _check(self.lib.lbmhd_set_porosity(self.h, dp_, dev))

    def set_sphere_width(self, eps):
        _check(self.lib.lbmhd_set_sphere_width(self.h, float(eps)))

    def set_sphere_rotation(self, omega):
        om = np.ascontiguousarray(omega, dtype=np.float64)
        _check(self.lib.lbmhd_set_sphere_rotation(self.h, _host_ptr(om)))

    def set_sphere_dipoles(self, offsets, dirs, B_surface, cores):
        off = np.ascontiguousarray(offsets, dtype=np.float64).reshape(-1, 3)
        m = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
        bs = np.ascontiguousarray(B_surface, dtype=np.float64).reshape(-1)
        co = np.ascontiguousarray(cores, dtype=np.float64).reshape(-1)
        assert len(off) == len(m) == len(bs) == len(co)
        _check(self.lib.lbmhd_set_sphere_dipoles(self.h, len(bs), _host_ptr(off), _host_ptr(m), _host_ptr(bs), _host_ptr(co)))

    def set_obstacle_rotation(self, omega, centre):
        om = np.ascontiguousarray(omega, dtype=np.float64)
        c = np.ascontiguousarray(centre, dtype=np.float64)
        _check(self.lib.lbmhd_set_obstacle_rotation(self.h, _host_ptr(om), _host_ptr(c)))

    def body_enable(self, enable=True, ref=None):
        """accumulate the body integrals during the steps (lbmhd_body_enable); ref: torque reference of masked bodies"""
        r = None if ref is None else np.ascontiguousarray(ref, dtype=np.float64)
        _check(self.lib.lbmhd_body_enable(self.h, int(bool(enable)), None if r is None else _host_ptr(r)))

    def body_read(self, reset=False, out=None):
        """F[3] | T[3] | W | I_B[3] | sum (1-d) B [3] | sum (1-d) since init / the last reset.  `out`: a device fp64 tensor
        of 14 elements (asynchronous), else a numpy array is returned (synchronises)"""
        if out is not None:
            assert out.is_cuda and out.dtype == self.torch.float64 and out.numel() >= 14 and out.is_contiguous()
            _check(self.lib.lbmhd_body_read(self.h, C.c_void_p(out.data_ptr()), int(reset), 1))
            return out
        res = np.zeros(14)
        _check(self.lib.lbmhd_body_read(self.h, _host_ptr(res), int(reset), 0))
        return res

    def populations(self):
        """canonical fp64 [K, Q, nz, ny, nx] on the host (via a device tensor)"""
        torch = self.torch
        t = torch.empty(self.K * self.Q * self.N, dtype=torch.float64, device=self.workspace.device)
        _check(self.lib.lbmhd_get_populations(self.h, C.c_void_p(t.data_ptr()), 1))
        self.stream.synchronize()
        return t.cpu().numpy().reshape((self.K, self.Q) + self.shape)

    def set_populations(self, g):
        torch = self.torch
        t = torch.as_tensor(np.ascontiguousarray(g, dtype=np.float64).reshape(-1)).to(self.workspace.device)
        _check(self.lib.lbmhd_set_populations(self.h, C.c_void_p(t.data_ptr()), 1))
        self.stream.synchronize()

    def halo_buffer(self, what=HALO_CROSSING):
        """device tensor sized for one packed face (element type = precision)"""
        torch = self.torch
        nbytes = int(self.lib.lbmhd_halo_bytes(self.h, int(what)))
        return torch.empty(nbytes, dtype=torch.uint8, device=self.workspace.device)

    def halo_pack(self, side, buf, what=HALO_CROSSING, next_copy=False, stream=None):
        if stream is None and not next_copy:
            _check(self.lib.lbmhd_halo_pack(self.h, int(side), int(what), C.c_void_p(buf.data_ptr())))
        else:
            st = (stream if stream is not None else self.stream).cuda_stream
            _check(self.lib.lbmhd_halo_pack_on(self.h, int(side), int(what), C.c_void_p(buf.data_ptr()), int(bool(next_copy)), st))

    def halo_unpack(self, side, buf, what=HALO_CROSSING, next_copy=False, stream=None):
        if stream is None and not next_copy:
            _check(self.lib.lbmhd_halo_unpack(self.h, int(side), int(what), C.c_void_p(buf.data_ptr())))
        else:
            st = (stream if stream is not None else self.stream).cuda_stream
            _check(self.lib.lbmhd_halo_unpack_on(self.h, int(side), int(what), C.c_void_p(buf.data_ptr()), int(bool(next_copy)), st))

    @property
    def steps_done(self):
        return int(self.lib.lbmhd_steps_done(self.h))

    @property
    def launch_count(self):
        return int(self.lib.lbmhd_launch_count(self.h))

    @property
    def step_path(self):
        """PATH_ONE / PATH_MULTI / PATH_CLUSTER / PATH_TMA / PATH_PERSIST of the last step launch (-1 before the first)"""
        return int(self.lib.lbmhd_step_path(self.h))


PATH_ONE, PATH_MULTI, PATH_CLUSTER, PATH_TMA, PATH_PERSIST, PATH_CELL, PATH_RESIDENT = 0, 1, 2, 3, 4, 5, 6


def from_workload(w, precision=64, device=0, streaming=STREAM_AB, solid_fields=True):
    """Lbmhd handle configured (boundaries, tau, sphere) for a workloads.py dict; fields not yet initialised."""
    p = make_params(w["scheme"], w["lattice"], w["shape"], precision=precision, gamma=w["gamma"] or 1.4, c0sq=w["c0sq"],
                    nu=w["nu"], eta=w["eta"], tau=w["tau"], powell=w["powell"], bc=w["bc"], streaming=streaming,
                    device=device, tau_relax=w.get("tau_relax", 0.0), eta_jc=w.get("eta_jc", 0.0))
    sim = Lbmhd(p, solid_fields=solid_fields)
    if w.get("sphere"):
        s = w["sphere"]
        sim.set_sphere(s["centre"], s["radius"], s["u_solid"], s["dipole_dir"], s["B_surface"])
        if s.get("width"):
            sim.set_sphere_width(s["width"])
        if s.get("omega") is not None:
            sim.set_sphere_rotation(s["omega"])
        if s.get("dipoles"):
            dp = s["dipoles"]
            sim.set_sphere_dipoles(dp["offsets"], dp["dirs"], dp["B_surface"], dp["cores"])
    return sim


def copy_probe(n_elems=1 << 28, reps=10, device=0):
    """measured fp64 copy bandwidth in GB/s (read + write bytes), BabelStream-style"""
    import torch
    lib = load_library()
    dev = torch.device("cuda", device)
    a = torch.ones(n_elems, dtype=torch.float64, device=dev)
    b = torch.empty_like(a)
    st = torch.cuda.current_stream(dev)
    _check(lib.lbmhd_copy_probe(C.c_void_p(a.data_ptr()), C.c_void_p(b.data_ptr()), n_elems, 3, st.cuda_stream))
    best = 0.0
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        _check(lib.lbmhd_copy_probe(C.c_void_p(a.data_ptr()), C.c_void_p(b.data_ptr()), n_elems, 1, st.cuda_stream))
        e1.record(st)
        e1.synchronize()
        best = max(best, 2 * 8 * n_elems / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return best


def triad_probe(n_elems=1 << 27, reps=10, device=0):
    """measured fp64 triad bandwidth in GB/s (a = b + s c: 24 bytes per element), BabelStream-style"""
    import torch
    lib = load_library()
    dev = torch.device("cuda", device)
    b = torch.ones(n_elems, dtype=torch.float64, device=dev)
    c = torch.ones_like(b)
    a = torch.empty_like(b)
    st = torch.cuda.current_stream(dev)
    args = (C.c_void_p(a.data_ptr()), C.c_void_p(b.data_ptr()), C.c_void_p(c.data_ptr()), 0.5, n_elems)
    _check(lib.lbmhd_triad_probe(*args, 3, st.cuda_stream))
    best = 0.0
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        _check(lib.lbmhd_triad_probe(*args, 1, st.cuda_stream))
        e1.record(st)
        e1.synchronize()
        best = max(best, 3 * 8 * n_elems / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return best


STATIC_DIAG_MAX_CELLS = 1 << 30


def diagnostics_static(scheme, lattice, shape, bc, gamma, fields_dev, diag_dev, device=0, stream=None):
    """lbmhd_diagnostics_static: the 3K+4 diagnostics of a device fields tensor with no allocation, no handle, no workspace
    (scratch in a static device array of the library).  fields_dev [K*N] and diag_dev [3K+4] are CUDA fp64 tensors (both None:
    set-up only); enqueued on `stream` (default: torch's current stream), nothing synchronises."""
    import torch
    lib = load_library()
    dims = list(shape) + [1] * (3 - len(shape))
    bcv = (C.c_int * 6)(*[int(b) for b in bc])
    st = stream if stream is not None else torch.cuda.current_stream(torch.device("cuda", device))
    fp = None if fields_dev is None else C.c_void_p(fields_dev.data_ptr())
    dg = None if diag_dev is None else C.c_void_p(diag_dev.data_ptr())
    if fields_dev is not None:
        assert fields_dev.is_cuda and fields_dev.dtype == torch.float64 and fields_dev.is_contiguous()
        assert diag_dev is not None and diag_dev.is_cuda and diag_dev.dtype == torch.float64 and diag_dev.is_contiguous()
    _check(lib.lbmhd_diagnostics_static(SCHEMES.get(scheme, scheme), LATTICES.get(lattice, lattice), dims[0], dims[1], dims[2], bcv,
                                        float(gamma), fp, dg, int(device), st.cuda_stream))
    return diag_dev
