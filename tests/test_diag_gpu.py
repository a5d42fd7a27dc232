"""The moments / diagnostics kernels (S9) on their own: failure detection (NaN, rho <= 0 -> flag bits, LBMHD_ENUMERIC) and the
two-stage reduction checked against numpy sums of the very fields the same lbmhd_moments call returned (no oracle round-off in
the comparison: the fold is deterministic, so agreement is at the level of summation-order rounding, ~eps * sum|.|)."""
import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from parity_util import oracle_from_workload
from test_parity_gpu import gpu_from_workload, random_workload

pytestmark = pytest.mark.gpu


def _poisoned(w, kinds):
    """populations of the initial state with a NaN and / or a rho <= 0 cell far apart (different reduction blocks)"""
    o = oracle_from_workload(w)
    o.init(w["fields"])
    g0 = o.populations()
    K, Q = g0.shape[:2]
    flat = g0.reshape(K, Q, -1)
    N = flat.shape[2]
    if "nan" in kinds:
        flat[6, 1, 17] = np.nan                      # B_y population of cell 17
    if "rho" in kinds:
        flat[0, :, N - 5] = -0.25 / Q                # rho = -0.25 at the far end of the domain
    return o, g0


@pytest.mark.parametrize("kinds,flag", [(("nan",), 1), (("rho",), 2), (("nan", "rho"), 3)])
@pytest.mark.parametrize("streaming", [0, 1])
def test_failure_flag_and_enumeric(kinds, flag, streaming):
    """lbmhd.h: flag = 1*(non-finite seen) + 2*(rho <= 0 seen); LBMHD_ENUMERIC from the host-pointer call"""
    from paper_2606_00641_b200 import lbmhd
    w = random_workload("IDEAL", "D3Q19", (300, 40, 30), (0,) * 6, seed=7)      # 360 000 cells: 1184 reduction blocks
    o, g0 = _poisoned(w, kinds)
    o.set_populations(g0)
    g = gpu_from_workload(w, streaming=streaming)
    g.init(w["fields"])
    g.set_populations(g0)
    K = g.K
    Qo, do = o.moments()
    Qg, dg = g.moments()                             # default: the flag is returned, not raised
    assert do[3 * K + 3] == flag and dg[3 * K + 3] == flag, (do[3 * K + 3], dg[3 * K + 3])
    with pytest.raises(lbmhd.LbmhdError) as ei:
        g.moments(check=True)
    assert ei.value.code == lbmhd.ENUMERIC
    # a device-pointer call stays asynchronous and returns OK; the flag is in the device diag
    import torch
    dd = torch.empty(3 * K + 4, dtype=torch.float64, device="cuda")
    fd = torch.empty(K * g.N, dtype=torch.float64, device="cuda")
    g.moments(fd, dd)
    assert float(dd[-1].cpu()) == flag
    g.close()


def test_clean_state_has_no_flag():
    w = random_workload("IDEAL", "D2Q9", (150, 37), (0,) * 6, seed=8)
    g = gpu_from_workload(w)
    g.init(w["fields"])
    g.step(3)
    _, dg = g.moments(check=True)
    assert dg[-1] == 0
    g.close()


@pytest.mark.parametrize("name,shape", [("C5", (192, 128, 128)), ("C4", None), ("C2", None)])
def test_reduction_against_numpy_of_the_same_fields(name, shape):
    """diag[0:K] = sum, [K:2K] = sum|.|, [2K:3K] = max|.| of fields_out of the SAME call, at ~ sqrt(N) eps sum|.|
    (pairwise-like two-stage fold on the device, pairwise in numpy), and exact for the extrema"""
    w = W.config5(shape=shape) if shape else W.get(name)
    g = gpu_from_workload(w)
    g.init(w["fields"])
    g.step(3)
    Q, dg = g.moments()
    K = g.K
    F = Q.reshape(K, -1)
    N = F.shape[1]
    eps = np.finfo(np.float64).eps
    s_abs = np.abs(F).sum(1)
    bound = 8 * np.sqrt(N) * eps * np.maximum(s_abs, 1e-300)
    assert (np.abs(dg[:K] - F.sum(1)) <= bound).all(), (dg[:K] - F.sum(1), bound)
    assert (np.abs(dg[K:2 * K] - s_abs) <= bound).all()
    assert (dg[2 * K:3 * K] == np.abs(F).max(1)).all()
    if w["scheme"] != "INCRES":
        assert dg[3 * K + 1] == F[0].min()
    g.close()
