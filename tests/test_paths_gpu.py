"""The non-default kernel paths stay correct: TMA-staged persistent kernel, fp32 one-cell kernels."""
import os

import numpy as np
import pytest

from paper_2606_00641_b200 import workloads as W
from test_parity_gpu import compare, random_workload

pytestmark = pytest.mark.gpu


@pytest.fixture
def env():
    saved = dict(os.environ)
    yield os.environ
    os.environ.clear()
    os.environ.update(saved)


@pytest.mark.parametrize("knobs", [{"LBMHD_PATH": "tma"}])
def test_alternative_paths_parity(env, knobs):
    env.update(knobs)
    compare(W.get("C5", small=True), 30)
    compare(W.get("C4", small=True), 30)
    compare(random_workload("IDEAL", "D3Q19", (100, 12, 9), (0,) * 6, seed=8), 10)
    compare(random_workload("INCRES", "D2Q9", (150, 37), (1, 1, 0, 0, 0, 0), seed=9), 10)
    compare(random_workload("IDEAL", "D1Q3", (200,), (2, 1, 0, 0, 0, 0), seed=10), 10)
