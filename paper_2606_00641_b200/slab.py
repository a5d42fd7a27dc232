"""Slab decomposition of one lattice over several GPUs.

The step couples cells only through nearest-neighbour pulls (|c_i| <= 1), so the lattice is cut into slabs along
its slowest axis (z in 3D, y in 2D), one slab per rank, each with one ghost plane per cut face
(`LBMHD_BC_HALO`).  Before every step each rank packs the populations that leave through its cut faces
(5 of 19 directions on D3Q19) and the neighbour unpacks them into its ghost plane: one paired send/recv per face
and step, no other collective on the data path.  This module holds only the host-side orchestration; packing,
unpacking and the step run in the CUDA library.

Two drivers of the same exchange schedule:
  * `exchange_local(slabs, ...)`      all slabs in one process (one GPU): device-to-device copies; used by the tests
    to check the sharded run against the unsharded one;
  * `exchange_distributed(slab, ...)` one slab per rank over `torch.distributed` (NCCL on GPUs, gloo in the CPU tests).
"""
import numpy as np

PERIODIC, ZEROGRAD, INFLOW, HALO = 0, 1, 2, 3


def slab_ranges(n, parts):
    """[(start, stop)] of the owned planes of each part; sizes differ by at most one, larger ones first"""
    if parts < 1 or n < parts:
        raise ValueError("cannot cut %d planes into %d slabs" % (n, parts))
    base, extra = divmod(n, parts)
    out, start = [], 0
    for r in range(parts):
        size = base + (1 if r < extra else 0)
        out.append((start, start + size))
        start += size
    return out


def neighbours(rank, parts, periodic):
    """(low, high) neighbour ranks along the cut axis, None where the slab touches a true boundary face"""
    if parts == 1:
        return None, None
    lo = rank - 1 if rank > 0 else (parts - 1 if periodic else None)
    hi = rank + 1 if rank < parts - 1 else (0 if periodic else None)
    return lo, hi


def local_geometry(shape, bc, rank, parts):
    """-> dict(shape, bc, halo_offset, owned=(lo, hi) local plane range, take=global plane indices incl. ghosts)"""
    D = len(shape)
    if D < 2:
        raise ValueError("slab decomposition needs a 2D or 3D lattice")
    nH = shape[D - 1]
    periodic = bc[2 * (D - 1)] == PERIODIC
    start, stop = slab_ranges(nH, parts)[rank]
    lo_nb, hi_nb = neighbours(rank, parts, periodic)
    lbc = list(bc)
    take = list(range(start, stop))
    if lo_nb is not None:
        take = [(start - 1) % nH] + take
        lbc[2 * (D - 1)] = HALO
    if hi_nb is not None:
        take = take + [stop % nH]
        lbc[2 * (D - 1) + 1] = HALO
    lshape = tuple(shape[:D - 1]) + (len(take),)
    g_lo = 1 if lo_nb is not None else 0
    return dict(shape=lshape, bc=tuple(lbc), halo_offset=start - g_lo, owned=(g_lo, g_lo + stop - start), take=np.array(take),
                lo=lo_nb, hi=hi_nb, start=start, stop=stop)


class Slab:
    """one rank's slab of a workloads.py dict, backed by an Lbmhd handle"""

    def __init__(self, w, rank, parts, precision=64, device=0):
        from . import lbmhd
        self.w, self.rank, self.parts = w, rank, parts
        self.D = len(w["shape"])
        self.geo = local_geometry(w["shape"], w["bc"], rank, parts)
        lw = dict(w, shape=self.geo["shape"], bc=self.geo["bc"])
        p = lbmhd.make_params(lw["scheme"], lw["lattice"], lw["shape"], precision=precision, gamma=lw["gamma"] or 1.4,
                              c0sq=lw["c0sq"], nu=lw["nu"], eta=lw["eta"], tau=lw["tau"], powell=lw["powell"], bc=lw["bc"],
                              device=device, tau_relax=lw.get("tau_relax", 0.0), eta_jc=lw.get("eta_jc", 0.0),
                              halo_offset=self.geo["halo_offset"])
        self.sim = lbmhd.Lbmhd(p)
        if w.get("sphere"):
            s = w["sphere"]                      # global coordinates: the kernels add halo_offset to the plane index
            self.sim.set_sphere(s["centre"], s["radius"], s["u_solid"], s["dipole_dir"], s["B_surface"])
            if s.get("width"):
                self.sim.set_sphere_width(s["width"])
            if s.get("omega") is not None:
                self.sim.set_sphere_rotation(s["omega"])
            if s.get("dipoles"):
                dp = s["dipoles"]
                self.sim.set_sphere_dipoles(dp["offsets"], dp["dirs"], dp["B_surface"], dp["cores"])
        self.lo, self.hi = self.geo["lo"], self.geo["hi"]

    def local_fields(self, fields):
        """[K, nz, ny, nx] global -> this slab's planes including ghosts (ghost values only matter until the first exchange)"""
        axis = 1 if self.D == 3 else 2          # fields are [K, z, y, x]; the cut axis is z in 3D, y in 2D
        return np.ascontiguousarray(np.take(fields, self.geo["take"], axis=axis))

    def init(self, fields):
        self.sim.init(self.local_fields(fields))

    def init_local(self, local_fields):
        """fields of this slab's planes only (ghosts included), e.g. generated per rank"""
        self.sim.init(local_fields)

    def owned(self, local_fields):
        lo, hi = self.geo["owned"]
        return local_fields[:, lo:hi] if self.D == 3 else local_fields[:, :, lo:hi]

    # the three calls the exchange drivers need
    def halo_buffer(self, full=False):
        return self.sim.halo_buffer(full)

    def halo_pack(self, side, buf, full=False):
        self.sim.halo_pack(side, buf, full)

    def halo_unpack(self, side, buf, full=False):
        self.sim.halo_unpack(side, buf, full)


def exchange_local(slabs, full=False):
    """refresh every ghost plane; all slabs live in this process and share one stream (ordering is stream order)"""
    for s in slabs:
        for side, nb in ((0, s.lo), (1, s.hi)):
            if nb is None:
                continue
            buf = s.halo_buffer(full)
            s.halo_pack(side, buf, full)                 # our plane next to the ghost on `side` ...
            slabs[nb].halo_unpack(1 - side, buf, full)   # ... is the neighbour's ghost on its opposite side


def exchange_distributed(slab, dist, full=False, via_host=False):
    """one slab per rank: one batch of paired send / recv with the low and the high neighbour, then unpack.
    Sends are posted low face first, receives high face first: when both neighbours are the same rank (two slabs,
    periodic) the k-th send to that rank then meets the k-th receive posted there, which is what an order-matched
    transport (NCCL) needs; the tags say the same to a tag-matched one (gloo).  via_host stages the packed planes
    through host memory (gloo cannot move CUDA tensors point to point): tests only."""
    ops, recv, keep, staged = [], {}, [], []
    for side, nb in ((0, slab.lo), (1, slab.hi)):
        if nb is None:
            continue
        out = slab.halo_buffer(full)
        slab.halo_pack(side, out, full)
        keep.append(out)
        if via_host:
            out = out.cpu()
            keep.append(out)
        ops.append(dist.P2POp(dist.isend, out, nb, tag=side))           # leaves through our `side`
    for side, nb in ((1, slab.hi), (0, slab.lo)):
        if nb is None:
            continue
        inp = slab.halo_buffer(full)
        keep.append(inp)
        recv[side] = inp
        if via_host:
            host = inp.cpu()
            staged.append((inp, host))
            inp = host
        ops.append(dist.P2POp(dist.irecv, inp, nb, tag=1 - side))       # left through the neighbour's opposite side
    if ops:
        for r in dist.batch_isend_irecv(ops):
            r.wait()
    for dev, host in staged:
        dev.copy_(host)
    for side, inp in recv.items():
        slab.halo_unpack(side, inp, full)
    return keep


def combine_diag(diags, K):
    """fold per-slab diagnostics [3K+4]: sums add, maxima max, minima min, flags or"""
    d = np.array(diags, dtype=np.float64)
    out = np.empty(3 * K + 4)
    out[:2 * K] = d[:, :2 * K].sum(0)
    out[2 * K:3 * K + 1] = d[:, 2 * K:3 * K + 1].max(0)
    out[3 * K + 1:3 * K + 3] = d[:, 3 * K + 1:3 * K + 3].min(0)
    flag = 0
    for v in d[:, 3 * K + 3]:
        flag |= int(v)
    out[3 * K + 3] = float(flag)
    return out


class LocalSlabGroup:
    """all slabs of a workload in one process on one GPU: the sharded run used to check the decomposition"""

    def __init__(self, w, parts, precision=64, device=0):
        self.w, self.parts = w, parts
        self.slabs = [Slab(w, r, parts, precision=precision, device=device) for r in range(parts)]
        self.K = self.slabs[0].sim.K

    def init(self, fields):
        for s in self.slabs:
            s.init(fields)

    def step(self, n=1):
        for _ in range(n):
            exchange_local(self.slabs)
            for s in self.slabs:
                s.sim.step(1)

    def moments(self):
        exchange_local(self.slabs, full=True)
        parts, diags = [], []
        for s in self.slabs:
            F, dg = s.sim.moments()
            parts.append(s.owned(F))
            diags.append(dg)
        axis = 1 if len(self.w["shape"]) == 3 else 2
        return np.concatenate(parts, axis=axis), combine_diag(diags, self.K)

    def body_enable(self, enable=True, ref=None):
        for s in self.slabs:
            s.sim.body_enable(enable, ref)

    def body_read(self, reset=False):
        """body integrals of the whole lattice: every slab sums over its owned cells, the sums add"""
        return sum(s.sim.body_read(reset) for s in self.slabs)

    def close(self):
        for s in self.slabs:
            s.sim.close()
