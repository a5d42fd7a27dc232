"""Slab decomposition on one GPU: all slabs in one process, ghost planes refreshed by device copies through the same
pack / unpack kernels a multi-GPU run uses.  The sharded run must reproduce the unsharded one (and hence the oracle)."""
import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from parity_util import field_errors, oracle_from_workload, TOL64, TOL32
from test_parity_gpu import random_workload, gpu_from_workload, divb_workload, resist_workload, full_workload

pytestmark = pytest.mark.gpu


def run_both(w, parts, steps, precision=64, streaming=0, overlap=False):
    from paper_2606_00641_b200 import slab
    ref = gpu_from_workload(w, precision=precision, streaming=streaming)
    ref.init(w["fields"])
    ref.step(steps)
    Qr, dr = ref.moments()
    ref.close()
    grp = slab.LocalSlabGroup(w, parts, precision=precision, streaming=streaming, overlap=overlap)
    grp.init(w["fields"])
    grp.step(steps)
    Qs, ds = grp.moments()
    grp.close()
    return Qr, dr, Qs, ds


@pytest.mark.parametrize("parts", [2, 3])
def test_config5_slabs_match_unsharded_and_oracle(parts):
    """periodic z cut through the moving sphere (centre z = 32 of 64)"""
    w = W.get("C5", small=True)
    Qr, dr, Qs, ds = run_both(w, parts, 30)
    assert (field_errors(Qs, Qr) <= 1e-13).all()
    K = 8
    assert np.allclose(ds[:2 * K], dr[:2 * K], rtol=1e-12, atol=1e-14)
    assert np.allclose(ds[2 * K:3 * K + 3], dr[2 * K:3 * K + 3], rtol=1e-12, atol=1e-14) and ds[-1] == dr[-1]
    o = oracle_from_workload(w)
    o.init(w["fields"])
    o.step(30)
    assert (field_errors(Qs, o.moments(diag=False)) <= TOL64).all()


@pytest.mark.parametrize("scheme,lattice,shape,bc,parts", [
    ("IDEAL", "D2Q9", (150, 37), (1, 1, 1, 1, 0, 0), 3),        # non-periodic cut axis: true faces at both ends
    ("IDEAL", "D2Q9", (150, 36), (0,) * 6, 2),                  # periodic, two slabs: both neighbours are the other slab
    ("INCRES", "D3Q19", (70, 9, 12), (1, 1, 0, 0, 2, 1), 4),
    ("IDEAL", "D3Q7", (100, 12, 10), (2, 1, 1, 1, 0, 0), 2),
])
def test_random_state_slabs(scheme, lattice, shape, bc, parts):
    w = random_workload(scheme, lattice, shape, bc, seed=61)
    Qr, dr, Qs, ds = run_both(w, parts, 12)
    assert (field_errors(Qs, Qr) <= 1e-13).all()
    assert abs(ds[3 * (Qr.shape[0])] - dr[3 * (Qr.shape[0])]) <= 1e-12 * max(dr[3 * Qr.shape[0]], 1e-30)    # max|div_h B| across cuts


def test_slabs_fp32_and_divb_scheme():
    w = random_workload("IDEAL", "D3Q19", (200, 12, 12), (2, 1, 0, 0, 0, 0), seed=62)
    Qr, dr, Qs, ds = run_both(w, 3, 10, precision=32)
    assert (field_errors(Qs, Qr) <= 1e-6).all()
    w = divb_workload("D3Q19", (100, 12, 12), (0,) * 6, seed=63)
    Qr, dr, Qs, ds = run_both(w, 2, 10)
    assert (field_errors(Qs, Qr) <= 1e-13).all()
    w = resist_workload("D3Q19", (100, 12, 12), (2, 1, 0, 0, 0, 0), seed=64)      # K = 17 sets across the cuts
    Qr, dr, Qs, ds = run_both(w, 3, 10)
    assert (field_errors(Qs, Qr) <= 1e-13).all()
    w = resist_workload("D2Q9", (100, 24), (0,) * 6, seed=65)
    Qr, dr, Qs, ds = run_both(w, 2, 10)
    assert (field_errors(Qs, Qr) <= 1e-13).all()
    w = full_workload("D3Q19", (64, 12, 12), (2, 1, 0, 0, 0, 0), seed=66)        # K = 26 sets across the cuts
    Qr, dr, Qs, ds = run_both(w, 3, 8)
    assert (field_errors(Qs, Qr) <= 1e-13).all()


@pytest.mark.parametrize("streaming", [0, 1])
@pytest.mark.parametrize("scheme,lattice,shape,bc,parts,steps", [
    ("IDEAL", "D3Q19", (100, 12, 12), (2, 1, 0, 0, 0, 0), 3, 11),       # periodic cut axis, odd step count (in place: layout P1 at the end)
    ("IDEAL", "D3Q19", (70, 9, 12), (1, 1, 1, 1, 1, 1), 4, 8),          # true faces at both ends of the cut axis
    ("IDEAL", "D2Q9", (150, 36), (0,) * 6, 2, 9),                       # two slabs, each the other's both neighbours
    ("INCRES", "D2Q9", (90, 30), (1, 1, 2, 1, 0, 0), 3, 6),
    ("IDEAL", "D3Q7", (100, 12, 10), (2, 1, 1, 1, 0, 0), 5, 7),         # slabs of two owned planes: both are boundary planes
])
def test_overlapped_schedule_is_bit_equal_to_serial(scheme, lattice, shape, bc, parts, steps, streaming):
    """boundary planes first, exchange on a side stream while the interior planes update: the same numbers, bit
    for bit, as whole-step-then-exchange, in both streaming modes; and both equal the unsharded run"""
    from paper_2606_00641_b200 import slab
    w = random_workload(scheme, lattice, shape, bc, seed=67)
    out = []
    for overlap in (False, True):
        grp = slab.LocalSlabGroup(w, parts, streaming=streaming, overlap=overlap)
        grp.init(w["fields"])
        grp.step(steps)
        out.append(grp.moments())
        grp.close()
    assert np.array_equal(out[0][0], out[1][0])
    assert np.array_equal(out[0][1], out[1][1])
    ref = gpu_from_workload(w, streaming=streaming)
    ref.init(w["fields"])
    ref.step(steps)
    Qr, dr = ref.moments()
    ref.close()
    assert (field_errors(out[1][0], Qr) <= 1e-13).all()
    K = Qr.shape[0]
    assert abs(out[1][1][3 * K] - dr[3 * K]) <= 1e-12 * max(dr[3 * K], 1e-30)


@pytest.mark.parametrize("overlap", [False, True])
def test_config5_in_place_slabs_with_the_sphere(overlap):
    """in-place (AA) streaming across cuts through the moving sphere: return exchange after pull-push steps, refresh after local ones"""
    w = W.get("C5", small=True)
    Qr, dr, Qs, ds = run_both(w, 3, 21, streaming=1, overlap=overlap)
    assert (field_errors(Qs, Qr) <= 1e-13).all()
    K = 8
    assert np.allclose(ds[:2 * K], dr[:2 * K], rtol=1e-12, atol=1e-14)
    assert np.allclose(ds[2 * K:3 * K + 3], dr[2 * K:3 * K + 3], rtol=1e-12, atol=1e-14) and ds[-1] == dr[-1]
    o = oracle_from_workload(w)
    o.init(w["fields"])
    o.step(21)
    assert (field_errors(Qs, o.moments(diag=False)) <= TOL64).all()


def test_population_exchange_route_of_the_diagnostics():
    """A/B: ghost planes refreshed with all Q directions (LBMHD_HALO_FULL) and lbmhd_moments give the same as the fields route"""
    from paper_2606_00641_b200 import slab
    w = random_workload("IDEAL", "D3Q19", (64, 10, 12), (0,) * 6, seed=68)
    grp = slab.LocalSlabGroup(w, 3)
    grp.init(w["fields"])
    grp.step(5)
    Qa, da = grp.moments()
    Qb, db = grp.moments_via_population_exchange()
    grp.close()
    assert np.array_equal(Qa, Qb) and np.allclose(da, db, rtol=1e-13, atol=1e-15)


def test_step_in_pieces_equals_whole_step():
    """lbmhd_step_part over any partition of the planes == lbmhd_step(1), both streaming modes, multi-cell kernel included"""
    import os
    for streaming in (0, 1):
        for lattice, shape, bc in (("D3Q19", (292, 6, 9), (2, 1, 0, 0, 0, 0)), ("D2Q9", (150, 37), (1, 1, 1, 1, 0, 0))):
            w = random_workload("IDEAL", lattice, shape, bc, seed=69)
            saved = os.environ.get("LBMHD_MULTI")
            os.environ["LBMHD_MULTI"] = "1"
            try:
                a, b = gpu_from_workload(w, streaming=streaming), gpu_from_workload(w, streaming=streaming)
            finally:
                if saved is None:
                    os.environ.pop("LBMHD_MULTI")
                else:
                    os.environ["LBMHD_MULTI"] = saved
            nH = shape[-1]
            for g in (a, b):
                g.init(w["fields"])
            for _ in range(5):
                a.step(1)
                b.step_part(nH - 2, nH, False)
                b.step_part(0, 1, False)
                b.step_part(3, 3, False)          # empty range: nothing launched
                b.step_part(1, nH - 2, True)
            assert a.steps_done == b.steps_done == 5
            assert np.array_equal(a.moments()[0], b.moments()[0])
            a.close()
            b.close()
