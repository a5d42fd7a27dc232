"""lbmhd_diagnostics_static (csrc/lbmhd_noalloc.cu): the diagnostics with no device allocation, no handle and no workspace —
its reduction scratch is a static device array of the library — against the existing path (lbmhd_moments with device
pointers, scratch in the caller's workspace) on the same device fields.  Different problems back to back, large then small
then large again: every call shares the one array, and a call must not see what the previous one left there.
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from parity_util import TOL64
from test_parity_gpu import random_workload

pytestmark = pytest.mark.gpu


def existing_and_static(w, steps):
    import torch
    from paper_2606_00641_b200 import lbmhd
    sim = lbmhd.from_workload(w)
    sim.init(w["fields"])
    sim.step(steps)
    K, N = sim.K, sim.N
    F = torch.empty(K * N, dtype=torch.float64, device="cuda")
    d_old = torch.empty(3 * K + 4, dtype=torch.float64, device="cuda")
    sim.moments(F, d_old)                                    # existing path: partials in the handle's workspace
    d_new = torch.full((3 * K + 4,), float("nan"), dtype=torch.float64, device="cuda")
    lbmhd.diagnostics_static(w["scheme"], w["lattice"], w["shape"], w["bc"], w["gamma"] or 1.4, F, d_new, stream=sim.stream)
    torch.cuda.synchronize()
    a, b = d_old.cpu().numpy(), d_new.cpu().numpy()
    sim.close()
    return a, b, K


def check(a, b, K):
    assert np.isfinite(b).all()
    scale = np.maximum(np.abs(a), 1e-300)
    assert (np.abs(b - a) <= TOL64 * scale).all(), (a, b)
    assert np.array_equal(a, b)                              # same kernels, same block count: bit-identical
    assert b[3 * K + 3] == 0


def test_static_scratch_diagnostics_match_the_workspace_path_on_calls_in_a_row():
    big = W.config5(shape=(96, 64, 64))                      # 393 216 cells, K = 8: all 1184 partial blocks in use
    small = random_workload("INCRES", "D2Q9", (90, 21), (1, 1, 2, 1, 0, 0), seed=401)      # 1890 cells, K = 5: 8 blocks
    full = W.variant(W.config5(shape=(48, 32, 32)), scheme="FULL")                        # K = 26: the widest partial rows
    for w, steps in ((big, 3), (small, 4), (big, 2), (full, 2), (small, 1)):
        a, b, K = existing_and_static(w, steps)
        check(a, b, K)


def test_static_scratch_limits_and_setup_call():
    from paper_2606_00641_b200 import lbmhd
    lbmhd.diagnostics_static("IDEAL", "D3Q19", (8, 8, 8), (0,) * 6, 5 / 3, None, None)      # set-up only
    with pytest.raises(lbmhd.LbmhdError) as ei:                                            # 2^31 cells > the stated 2^30
        lbmhd.diagnostics_static("IDEAL", "D3Q19", (2048, 1024, 1024), (0,) * 6, 5 / 3, None, None)
    assert ei.value.code == lbmhd.ENOMEM and "at most" in str(ei.value)
    assert lbmhd.STATIC_DIAG_MAX_CELLS == 1 << 30
    with pytest.raises(lbmhd.LbmhdError) as ei:
        lbmhd.diagnostics_static("IDEAL", "D2Q9", (8, 8, 8), (0,) * 6, 5 / 3, None, None)   # nz != 1 on a 2D lattice
    assert ei.value.code == lbmhd.EINVAL
