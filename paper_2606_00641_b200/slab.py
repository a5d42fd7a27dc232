"""Slab decomposition of one lattice over several GPUs (the paper's own runs use two GPUs,
PAPER.md:281).

The step couples cells only through nearest-neighbour pulls (|c_i| <= 1), so the lattice is cut into slabs along its slowest
axis (z in 3D, y in 2D), one slab per rank, each with one ghost plane per cut face (`LBMHD_BC_HALO`).  Per step and cut face
one packed plane of crossing populations (5 of 19 directions on D3Q19) goes to the neighbour: a paired send / recv, no other
collective on the data path.  This module holds only the host-side orchestration; packing, unpacking and the step run in the
CUDA library.

Schedule of one step (`overlap=True`, both streaming modes):
  1. main stream: wait for the previous exchange; update the owned planes next to the ghosts (`lbmhd_step_part`);
  2. side stream: pack those planes' crossing populations out of the copy the step writes, send / receive, unpack into the
     ghost planes of that copy (`lbmhd_halo_*_on(next_copy=1)`);
  3. main stream, meanwhile: update the interior planes and complete the step.
`overlap=False` is the plain order (whole step, then exchange); both give bit-identical results.

What is exchanged after a step (the buffers are allocated once per slab):
  A/B streaming       LBMHD_HALO_CROSSING: owned boundary plane -> the neighbour's ghost plane.
  in place (AA)       after a pull-push step LBMHD_HALO_RETURN (the pushed populations sit in OUR ghost plane and belong in the
                      neighbour's boundary plane), after a local step LBMHD_HALO_CROSSING.

Two drivers of that schedule:
  * `LocalSlabGroup`        all slabs in one process on one GPU, device copies: the tests check the sharded run against the
                            unsharded one and the overlapped schedule against the serial one;
  * `DistributedExchange`   one slab per rank over `torch.distributed` (NCCL on GPUs; gloo with host staging in the tests).
"""
import numpy as np

PERIODIC, ZEROGRAD, INFLOW, HALO = 0, 1, 2, 3
CROSSING, FULL, RETURN = 0, 1, 2


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


def step_pieces(owned, has_lo, has_hi):
    """-> (boundary plane ranges, interior plane range) of one step: the owned planes next to a ghost go first"""
    g_lo, g_hi = owned
    b = []
    if has_lo:
        b.append((g_lo, g_lo + 1))
    if has_hi and (not has_lo or g_hi - 1 > g_lo):
        b.append((g_hi - 1, g_hi))
    i_lo = g_lo + (1 if has_lo else 0)
    i_hi = g_hi - (1 if has_hi else 0)
    return b, (i_lo, max(i_lo, i_hi))


def exchange_kind(streaming, parity_before_step):
    """what moves after a step that started from in-place layout `parity_before_step` (A/B: always CROSSING)"""
    if streaming == 0:
        return CROSSING
    return RETURN if parity_before_step == 0 else CROSSING


class Slab:
    """one rank's slab of a workloads.py dict, backed by an Lbmhd handle; halo buffers are allocated once"""

    def __init__(self, w, rank, parts, precision=64, device=0, streaming=0):
        from . import lbmhd
        self.w, self.rank, self.parts, self.streaming = w, rank, parts, streaming
        self.D = len(w["shape"])
        self.geo = local_geometry(w["shape"], w["bc"], rank, parts)
        lw = dict(w, shape=self.geo["shape"], bc=self.geo["bc"])
        p = lbmhd.make_params(lw["scheme"], lw["lattice"], lw["shape"], precision=precision, gamma=lw["gamma"] or 1.4,
                              c0sq=lw["c0sq"], nu=lw["nu"], eta=lw["eta"], tau=lw["tau"], powell=lw["powell"], bc=lw["bc"],
                              device=device, tau_relax=lw.get("tau_relax", 0.0), eta_jc=lw.get("eta_jc", 0.0),
                              halo_offset=self.geo["halo_offset"], streaming=streaming)
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
        self.parity = 0                          # in place: layout of the stored populations (0 after init)
        self.pieces = step_pieces(self.geo["owned"], self.lo is not None, self.hi is not None)
        # one send and one receive buffer per cut face, for the life of the slab (CROSSING and RETURN have the same size)
        self.send = {side: self.sim.halo_buffer(CROSSING) for side, nb in ((0, self.lo), (1, self.hi)) if nb is not None}
        self.recv = {side: self.sim.halo_buffer(CROSSING) for side, nb in ((0, self.lo), (1, self.hi)) if nb is not None}
        self._full = None

    def local_fields(self, fields):
        """[K, nz, ny, nx] global -> this slab's planes including ghosts (ghost values only matter until the first exchange)"""
        axis = 1 if self.D == 3 else 2          # fields are [K, z, y, x]; the cut axis is z in 3D, y in 2D
        return np.ascontiguousarray(np.take(fields, self.geo["take"], axis=axis))

    def init(self, fields):
        self.sim.init(self.local_fields(fields))
        self.parity = 0

    def init_local(self, local_fields):
        """fields of this slab's planes only (ghosts included), e.g. generated per rank"""
        self.sim.init(local_fields)
        self.parity = 0

    def owned(self, local_fields):
        lo, hi = self.geo["owned"]
        return local_fields[:, lo:hi] if self.D == 3 else local_fields[:, :, lo:hi]

    # ---- the calls the exchange drivers need ------------------------------------------------------------------
    def halo_buffer(self, what=CROSSING):
        if what == FULL:
            return self.sim.halo_buffer(FULL)
        raise ValueError("crossing / return buffers are preallocated: slab.send[side], slab.recv[side]")

    def full_buffers(self):
        """(send, recv) buffers of the all-directions exchange (A/B diagnostics route), allocated on first use"""
        if self._full is None:
            self._full = ({s: self.sim.halo_buffer(FULL) for s in self.send}, {s: self.sim.halo_buffer(FULL) for s in self.recv})
        return self._full

    def halo_pack(self, side, buf, what=CROSSING, next_copy=False, stream=None):
        self.sim.halo_pack(side, buf, what, next_copy=next_copy, stream=stream)

    def halo_unpack(self, side, buf, what=CROSSING, next_copy=False, stream=None):
        self.sim.halo_unpack(side, buf, what, next_copy=next_copy, stream=stream)

    def step_boundary(self):
        """the owned planes next to the ghosts (step not completed)"""
        for lo, hi in self.pieces[0]:
            self.sim.step_part(lo, hi, False)

    def step_interior(self):
        """the other owned planes; completes the step"""
        lo, hi = self.pieces[1]
        self.sim.step_part(lo, hi, True)
        self.parity ^= 1

    def step_whole(self):
        self.sim.step(1)
        self.parity ^= 1

    def kind_after_step(self, parity_before):
        return exchange_kind(self.streaming, parity_before)

    # ---- ghost planes of a FIELDS tensor [K, planes...] (diagnostics across the cuts) ------------------------------
    def field_plane(self, F, idx):
        return F[:, idx] if self.D == 3 else F[:, :, idx]


def _moments_device(sl):
    torch = sl.sim.torch
    F = torch.empty((sl.sim.K,) + sl.sim.shape, dtype=torch.float64, device=sl.sim.workspace.device)
    sl.sim.moments(F.view(-1), None)
    return F


def exchange_local(slabs, what=CROSSING, next_copy=False, stream=None):
    """refresh the ghost planes (CROSSING / FULL) or hand the pushed populations back (RETURN); all slabs live in this process"""
    for s in slabs:
        for side, nb in ((0, s.lo), (1, s.hi)):
            if nb is None:
                continue
            buf = s.send[side] if what != FULL else s.sim.halo_buffer(FULL)
            s.halo_pack(side, buf, what, next_copy=next_copy, stream=stream)                 # our plane on `side` ...
            slabs[nb].halo_unpack(1 - side, buf, what, next_copy=next_copy, stream=stream)   # ... lands on the neighbour's opposite side


def exchange_distributed(slab, dist, what=CROSSING, via_host=False, next_copy=False, stream=None):
    """one slab per rank: one batch of paired send / recv with the low and the high neighbour, then unpack.
    Sends are posted low face first, receives high face first: when both neighbours are the same rank (two slabs,
    periodic) the k-th send to that rank then meets the k-th receive posted there, which is what an order-matched
    transport (NCCL) needs; the tags say the same to a tag-matched one (gloo).  via_host stages the packed planes
    through host memory (gloo cannot move CUDA tensors point to point): tests only.  With `stream`, the caller has made it
    the current torch stream: pack, the transfers and unpack are ordered on it."""
    ops, recv, staged = [], {}, []
    send_b, recv_b = slab.full_buffers() if what == FULL else (slab.send, slab.recv)
    keep = []
    for side, nb in ((0, slab.lo), (1, slab.hi)):
        if nb is None:
            continue
        out = send_b[side]
        slab.halo_pack(side, out, what, next_copy=next_copy, stream=stream)
        if via_host:
            out = out.cpu()
            keep.append(out)
        ops.append(dist.P2POp(dist.isend, out, nb, tag=side))           # leaves through our `side`
    for side, nb in ((1, slab.hi), (0, slab.lo)):
        if nb is None:
            continue
        inp = recv_b[side]
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
        slab.halo_unpack(side, inp, what, next_copy=next_copy, stream=stream)
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


class DistributedExchange:
    """one slab per rank: drives steps and exchanges over torch.distributed"""

    def __init__(self, slab, dist, via_host=False, overlap=True):
        self.sl, self.dist, self.via_host, self.overlap = slab, dist, via_host, overlap
        torch = slab.sim.torch
        self.torch = torch
        self.main = slab.sim.stream
        self.side = torch.cuda.Stream(device=slab.sim.workspace.device) if overlap else None
        self.ev_boundary = torch.cuda.Event()
        self.ev_exchanged = torch.cuda.Event()
        self.pending = False

    def prime(self):
        """after init: ghost planes hold the neighbours' boundary populations (layout P0 in place)"""
        exchange_distributed(self.sl, self.dist, CROSSING, via_host=self.via_host)

    def step(self):
        sl, torch = self.sl, self.torch
        kind = sl.kind_after_step(sl.parity)
        if not self.overlap:
            sl.step_whole()
            exchange_distributed(sl, self.dist, kind, via_host=self.via_host)
            return
        if self.pending:
            self.main.wait_event(self.ev_exchanged)          # the ghost planes this step pulls from are in place
        sl.step_boundary()
        self.ev_boundary.record(self.main)
        with torch.cuda.stream(self.side):
            self.side.wait_event(self.ev_boundary)
            exchange_distributed(sl, self.dist, kind, via_host=self.via_host, next_copy=True, stream=self.side)
            self.ev_exchanged.record(self.side)
        self.pending = True
        sl.step_interior()                                   # overlaps the exchange; completes the step

    def join(self):
        """the main stream waits for the last exchange (call before timing stops or before reading the state)"""
        if self.pending:
            self.main.wait_event(self.ev_exchanged)
            self.pending = False

    def fields_with_ghosts(self):
        """moments of this slab on the device with the ghost planes of the FIELDS refreshed from the neighbours"""
        sl, dist = self.sl, self.dist
        self.join()
        F = _moments_device(sl)
        g_lo, g_hi = sl.geo["owned"]
        ops, recv, staged = [], [], []
        for side, nb, src_idx in ((0, sl.lo, g_lo), (1, sl.hi, g_hi - 1)):
            if nb is None:
                continue
            out = sl.field_plane(F, src_idx).contiguous()
            if self.via_host:
                out = out.cpu()
            ops.append(dist.P2POp(dist.isend, out, nb, tag=10 + side))
        for side, nb, dst_idx in ((1, sl.hi, g_hi), (0, sl.lo, g_lo - 1)):
            if nb is None:
                continue
            buf = self.torch.empty_like(sl.field_plane(F, dst_idx).contiguous())
            host = buf.cpu() if self.via_host else buf
            ops.append(dist.P2POp(dist.irecv, host, nb, tag=10 + (1 - side)))
            recv.append((dst_idx, buf, host))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        for dst_idx, buf, host in recv:
            if self.via_host:
                buf.copy_(host)
            sl.field_plane(F, dst_idx).copy_(buf)
        return F

    def diagnostics(self):
        """this slab's share of the diagnostics (owned cells; div_h B sees the neighbours' fields); fold with combine_diag"""
        F = self.fields_with_ghosts()
        return self.sl.sim.diagnostics(F.view(-1))

    def moments(self):
        F = self.fields_with_ghosts()
        dg = self.sl.sim.diagnostics(F.view(-1))
        return F.cpu().numpy(), dg


class LocalSlabGroup:
    """all slabs of a workload in one process on one GPU: the sharded run used to check the decomposition"""

    def __init__(self, w, parts, precision=64, device=0, streaming=0, overlap=False):
        self.w, self.parts, self.overlap = w, parts, overlap
        self.slabs = [Slab(w, r, parts, precision=precision, device=device, streaming=streaming) for r in range(parts)]
        self.K = self.slabs[0].sim.K
        torch = self.slabs[0].sim.torch
        self.torch = torch
        self.main = self.slabs[0].sim.stream
        self.side = torch.cuda.Stream(device=self.slabs[0].sim.workspace.device) if overlap else None
        self.ev_b, self.ev_x, self.pending = torch.cuda.Event(), torch.cuda.Event(), False

    def init(self, fields):
        for s in self.slabs:
            s.init(fields)
        exchange_local(self.slabs, CROSSING)

    def step(self, n=1):
        for _ in range(n):
            kind = self.slabs[0].kind_after_step(self.slabs[0].parity)
            if not self.overlap:
                for s in self.slabs:
                    s.step_whole()
                exchange_local(self.slabs, kind)
                continue
            if self.pending:
                self.main.wait_event(self.ev_x)
            for s in self.slabs:
                s.step_boundary()
            self.ev_b.record(self.main)
            self.side.wait_event(self.ev_b)
            exchange_local(self.slabs, kind, next_copy=True, stream=self.side)      # before any slab completes its step
            self.ev_x.record(self.side)
            self.pending = True
            for s in self.slabs:
                s.step_interior()

    def join(self):
        if self.pending:
            self.main.wait_event(self.ev_x)
            self.pending = False

    def moments(self):
        """fields of the whole lattice and the folded diagnostics; ghost planes of the FIELDS come from the neighbours"""
        self.join()
        Fs = [_moments_device(s) for s in self.slabs]
        for s, F in zip(self.slabs, Fs):
            g_lo, g_hi = s.geo["owned"]
            if s.lo is not None:
                nb = self.slabs[s.lo]
                s.field_plane(F, g_lo - 1).copy_(nb.field_plane(Fs[s.lo], nb.geo["owned"][1] - 1))
            if s.hi is not None:
                nb = self.slabs[s.hi]
                s.field_plane(F, g_hi).copy_(nb.field_plane(Fs[s.hi], nb.geo["owned"][0]))
        parts, diags = [], []
        for s, F in zip(self.slabs, Fs):
            diags.append(s.sim.diagnostics(F.view(-1)))
            parts.append(s.owned(F.cpu().numpy()))
        axis = 1 if len(self.w["shape"]) == 3 else 2
        return np.concatenate(parts, axis=axis), combine_diag(diags, self.K)

    def moments_via_population_exchange(self):
        """A/B only: the older route — all Q directions of the boundary planes into the ghosts (LBMHD_HALO_FULL), then lbmhd_moments"""
        self.join()
        exchange_local(self.slabs, FULL)
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
        self.join()
        return sum(s.sim.body_read(reset) for s in self.slabs)

    def close(self):
        for s in self.slabs:
            s.sim.close()
