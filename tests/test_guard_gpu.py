"""Memory-safety and race evidence without compute-sanitizer (the tool is closed on this GPU pool: profiles/r2_sanitizer.md).

* Guard bands: every handle the cases of tests/sanitizer_cases.py create gets 1 MiB of 0xA5 before and after its workspace
  (LBMHD_GUARD_BYTES); closing the handle checks them.  The cases cover every step-kernel family (one cell per thread, several
  cells per thread with vector accesses and shuffled stores, cell per thread, 2-CTA cluster, cooperative many-step launch, the
  register-resident cluster kernel of the 1D lattices), both
  in-place step types, x-edge / general / sphere tiles and the slab halo kernels, each also compared with the oracle: an
  out-of-bounds WRITE trips a guard, an out-of-bounds or misplaced READ changes a result.
* Races: the in-place (AA) kernels and the cluster exchange are the places where a mis-indexed slot would be a silent race.
  A race shows as run-to-run differences: the same in-place run, repeated, must give bit-identical populations."""
import os

import numpy as np
import pytest

from test_parity_gpu import random_workload, resist_workload, gpu_from_workload

pytestmark = pytest.mark.gpu


@pytest.fixture
def env():
    saved = dict(os.environ)
    yield os.environ
    os.environ.clear()
    os.environ.update(saved)


def test_guard_bands_survive_every_kernel_family(env):
    import sanitizer_cases
    env["LBMHD_GUARD_BYTES"] = str(1 << 20)
    sanitizer_cases.main()


def test_guard_band_check_is_live(env):
    """the check itself: damage a guard byte by hand and close() must raise"""
    from paper_2606_00641_b200 import lbmhd
    env["LBMHD_GUARD_BYTES"] = "4096"
    w = random_workload("IDEAL", "D2Q9", (64, 16), (0,) * 6, seed=501)
    g = gpu_from_workload(w)
    g.init(w["fields"])
    g.step(2)
    assert g.guards_intact()
    g.workspace[-1] = 0
    assert not g.guards_intact()
    with pytest.raises(lbmhd.LbmhdError):
        g.close()


@pytest.mark.parametrize("case", ["multi64", "multi32", "cluster", "cell", "edge", "resident"])
def test_in_place_runs_are_bit_reproducible(env, case):
    env["LBMHD_PERSIST"] = "0"
    prec = 64
    if case == "resident":       # halo cells through st.async + mbarrier between the CTAs of one cluster
        env["LBMHD_RESIDENT"] = "1"
        w = random_workload("IDEAL", "D1Q3", (800,), (1, 1, 0, 0, 0, 0), seed=507)
    elif case == "multi64":
        env["LBMHD_MULTI"] = "1"
        w = random_workload("IDEAL", "D3Q19", (292, 6, 5), (2, 1, 0, 0, 0, 0), seed=502)
    elif case == "multi32":
        env["LBMHD_MULTI"] = "1"
        prec = 32
        w = random_workload("IDEAL", "D3Q7", (292, 6, 5), (0, 0, 1, 1, 0, 0), seed=503)
    elif case == "cluster":
        w = resist_workload("D3Q19", (100, 12, 9), (2, 1, 0, 0, 0, 0), seed=504)
    elif case == "cell":
        env["LBMHD_CELL"] = "2"
        w = random_workload("IDEAL", "D2Q5", (292, 10), (0,) * 6, seed=505)
    else:
        w = random_workload("IDEAL", "D2Q9", (150, 37), (1, 1, 1, 1, 0, 0), seed=506)
    runs = []
    for _ in range(3):
        g = gpu_from_workload(w, precision=prec, streaming=1)
        g.init(w["fields"])
        g.step(7)
        runs.append(g.populations())
        g.close()
    assert np.array_equal(runs[0], runs[1]) and np.array_equal(runs[0], runs[2])
