import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def tiny():
    from paper_2607_05622_b200.inputs import make_workload
    return make_workload("tiny")


@pytest.fixture(scope="session")
def small():
    from paper_2607_05622_b200.inputs import make_workload
    return make_workload("small")


@pytest.fixture(scope="session")
def spd_basis():
    """3 atoms, one contracted s, p and d shell each (N = 30): brute force N^4 with d functions."""
    import numpy as np
    from paper_2607_05622_b200.inputs import custom_basis
    xyz = np.array([[0.0, 0.1, -0.2], [1.9, 0.3, 0.4], [-0.7, 2.1, 1.0]])
    sh = [(0, [0.9, 0.3], [0.6, 0.4]), (1, [0.7, 0.25], [0.6, 0.4]), (2, [0.8, 0.35], [0.6, 0.4])]
    return custom_basis(xyz, [sh, sh, sh])


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """The CUDA library is built in-tree (incremental, a no-op when up to date); tests never run against a stale or
    missing libltjk.so.  nvcc cross-compiles without a GPU, so this also holds for the CPU tier."""
    from paper_2607_05622_b200 import build
    build.build()
