import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

# The parity tests step small lattices many times per call; left to itself lbmhd_step would run those calls as ONE cooperative
# launch (step_kernel_persist) and the one-launch-per-step kernels would go untested.  Default for the test
# session: per-step launches; tests/test_persist_gpu.py and the graded / full-size tests set LBMHD_PERSIST themselves.
os.environ.setdefault("LBMHD_PERSIST", "0")
# likewise the register-resident many-step kernel of the 1D lattices: tests/test_resident_gpu.py turns it on
os.environ.setdefault("LBMHD_RESIDENT", "0")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if _has_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
