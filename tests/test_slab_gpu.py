"""Slab decomposition on one GPU: all slabs in one process, ghost planes refreshed by device copies through the same
pack / unpack kernels a multi-GPU run uses.  The sharded run must reproduce the unsharded one (and hence the oracle)."""
import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from parity_util import field_errors, oracle_from_workload, TOL64, TOL32
from test_parity_gpu import random_workload, gpu_from_workload, divb_workload, resist_workload, full_workload

pytestmark = pytest.mark.gpu


def run_both(w, parts, steps, precision=64):
    from paper_2606_00641_b200 import slab
    ref = gpu_from_workload(w, precision=precision)
    ref.init(w["fields"])
    ref.step(steps)
    Qr, dr = ref.moments()
    ref.close()
    grp = slab.LocalSlabGroup(w, parts, precision=precision)
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
