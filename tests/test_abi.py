"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/lbmhd.h declares,
validates arguments before touching a device, and fails loudly (no CPU fallback) when there is no GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2606_00641_b200 import build as B
from paper_2606_00641_b200 import lbmhd

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return lbmhd.load_library()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "lbmhd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(lbmhd_[a-z_]+)\s*\(", hdr))
    assert {"lbmhd_create", "lbmhd_init", "lbmhd_step", "lbmhd_moments", "lbmhd_set_obstacle"} <= declared
    assert declared == set(lbmhd.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_geometry_and_workspace_arithmetic(lib):
    for scheme, lat, shape, K, Q in [("IDEAL", "D1Q3", (800,), 8, 3), ("INCRES", "D2Q9", (512, 512), 5, 9),
                                     ("IDEAL", "D2Q9", (1024, 1024), 8, 9), ("IDEAL", "D3Q19", (384, 256, 256), 8, 19),
                                     ("INCRES", "D3Q19", (10, 10, 10), 7, 19), ("INCRES", "D1Q3", (10,), 3, 3),
                                     ("IDEAL", "D2Q5", (64, 64), 8, 5), ("INCRES", "D3Q7", (10, 10, 10), 7, 7)]:
        p = lbmhd.make_params(scheme, lat, shape)
        assert lib.lbmhd_num_vars(C.byref(p)) == K and lib.lbmhd_num_dirs(C.byref(p)) == Q
        N = int(np.prod(shape))
        nbytes = lbmhd.workspace_bytes(p)
        pops = 2 * K * Q * ((N + 31) // 32 * 32) * 8
        side = K * N * 8 + N + 3 * N * 8 + N * 8          # moments scratch, mask, B_solid, porosity
        assert pops + side <= nbytes <= pops + side + 2 ** 20
        p32 = lbmhd.make_params(scheme, lat, shape, precision=32)
        assert lbmhd.workspace_bytes(p32) < nbytes
    # config 5 in A/B form fits one B200 (61.2 GB of populations)
    p = lbmhd.make_params("IDEAL", "D3Q19", (384, 256, 256))
    assert 61e9 < lbmhd.workspace_bytes(p) < 66e9
    bad = lbmhd.make_params("IDEAL", 7, (8, 8, 8))
    assert lib.lbmhd_num_vars(C.byref(bad)) == lbmhd.EINVAL and lbmhd.workspace_bytes(bad) == 0


def _create(lib, p, ws=4096):
    p.workspace = ws
    p.workspace_bytes = 1 << 62
    h = C.c_void_p()
    rc = lib.lbmhd_create(C.byref(p), None, C.byref(h))
    return rc, lib.lbmhd_last_error().decode()


def test_create_validates_before_touching_a_device(lib):
    mk = lbmhd.make_params
    cases = [
        (mk("IDEAL", "D2Q9", (16, 16), tau=0.5), "tau"),
        (mk("IDEAL", "D2Q9", (16, 16), tau=[0.6] * 5 + [0.7, 0.8, 0.7]), "magnetic"),
        (mk("IDEAL", "D2Q9", (16, 16), gamma=1.0), "gamma"),
        (mk("IDEAL", "D2Q9", (16, 16), bc=(0, 1, 0, 0, 0, 0)), "paired"),
        (mk("IDEAL", "D2Q9", (2, 16), bc=(1, 1, 0, 0, 0, 0)), ">= 3"),
        (mk("IDEAL", "D1Q3", (16, 2)), "ny must be 1"),
        (mk("IDEAL", "D2Q9", (16, 16, 2)), "nz must be 1"),
        (mk("IDEAL", "D2Q9", (16, 16), precision=16), "precision"),
        (mk("IDEAL", "D2Q9", (16, 16), streaming=2), "streaming"),
        (mk("IDEAL", "D2Q9", (16, 16), bc=(0, 0, 5, 5, 0, 0)), "boundary"),
    ]
    for p, word in cases:
        rc, msg = _create(lib, p)
        assert rc == lbmhd.EINVAL and word in msg, (rc, msg, word)
    p = mk("IDEAL", "D2Q9", (16, 16))
    p.workspace, p.workspace_bytes = 4096, 100
    h = C.c_void_p()
    assert lib.lbmhd_create(C.byref(p), None, C.byref(h)) == lbmhd.ENOMEM
    p.workspace, p.workspace_bytes = 4097, 1 << 40
    assert lib.lbmhd_create(C.byref(p), None, C.byref(h)) == lbmhd.ENOMEM
    p.workspace = None
    assert lib.lbmhd_create(C.byref(p), None, C.byref(h)) == lbmhd.EINVAL
    assert lib.lbmhd_step(None, 1) == lbmhd.EINVAL and lib.lbmhd_init(None, None, 0) == lbmhd.EINVAL


def test_no_cpu_fallback_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    rc, msg = _create(lib, lbmhd.make_params("IDEAL", "D2Q9", (16, 16)))
    assert rc == lbmhd.ECUDA and "cudaSetDevice" in msg
    with pytest.raises(lbmhd.LbmhdError):
        lbmhd.Lbmhd(lbmhd.make_params("IDEAL", "D2Q9", (16, 16)))


def test_product_path_does_not_touch_the_oracle():
    """the CUDA package neither imports nor links anything under oracle/, and the oracle never imports the package"""
    pkg = os.path.join(ROOT, "paper_2606_00641_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the oracle", "").replace("oracle uses", "").replace("like the oracle", "").replace("nor the oracle", ""), (dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_00641_b200" not in txt and "from paper_2606_00641_b200" not in txt
            assert "lbmhd.h" not in txt and "csrc" not in txt
