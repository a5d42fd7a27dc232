"""Host-side checks of the input generators and of bench.py's option handling (no GPU)."""
import subprocess
import sys
import os

import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_variant_extends_fields_and_parameters():
    w = W.config5(shape=(24, 16, 16))
    for scheme, K in (("IDEAL_DIVB", 9), ("RESIST", 17), ("FULL", 26)):
        v = W.variant(w, scheme=scheme)
        assert v["scheme"] == scheme and v["fields"].shape == (K, 16, 16, 24)
        assert np.array_equal(v["fields"][:8], w["fields"]) and not v["fields"][8:].any()
        assert v["tau_relax"] > 0 and (scheme == "IDEAL_DIVB" or v["eta"] > 0) and (scheme != "FULL" or v["nu"] > 0)
    assert w["scheme"] == "IDEAL" and w["fields"].shape[0] == 8          # the input is not modified
    assert W.variant(w, lattice="D3Q7")["lattice"] == "D3Q7"
    with pytest.raises(ValueError):
        W.variant(w, lattice="D2Q5")
    with pytest.raises(ValueError):
        W.variant(W.get("C2", small=True), scheme="RESIST")


def test_config2_as_stated_and_its_incres_variant_run_in_the_oracle():
    """C2 = BASELINE's numbers (rms 0.05, nu = eta = 1e-3) on scheme FULL; C2i = the INCRES reading at rms 0.02"""
    from parity_util import oracle_from_workload
    w = W.get("C2", small=True)
    assert w["scheme"] == "FULL" and w["fields"].shape == (20, 1, 128, 128) and w["nu"] == 1e-3 and w["eta"] == 1e-3
    u = w["fields"][1:3] / w["fields"][0]
    assert abs(np.sqrt((u * u).sum(0).mean()) - 0.05) < 1e-12 and abs(np.sqrt((w["fields"][5:7] ** 2).sum(0).mean()) - 0.05) < 1e-12
    wi = W.get("C2i", small=True)
    assert wi["scheme"] == "INCRES" and wi["fields"].shape == (5, 1, 128, 128)
    assert abs(np.sqrt((wi["fields"][1:3] ** 2).sum(0).mean()) - 0.02) < 1e-12
    for ww in (w, wi):
        o = oracle_from_workload(ww)
        o.init(ww["fields"])
        o.step(40)
        Q, dg = o.moments()
        assert dg[-1] == 0 and np.isfinite(Q).all()


def test_variant_runs_in_the_oracle():
    from parity_util import oracle_from_workload
    w = W.variant(W.config5(shape=(24, 16, 16)), scheme="FULL", lattice="D3Q7")
    o = oracle_from_workload(w)
    o.init(w["fields"])
    o.step(3)
    Q, dg = o.moments()
    assert Q.shape[0] == 26 and dg[-1] == 0


def test_bench_refuses_to_run_native_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "1"], capture_output=True, text=True)
    assert r.returncode != 0 and "no CUDA device and no CPU fallback" in (r.stderr + r.stdout)
