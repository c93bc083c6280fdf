import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def load_golden():
    """tests/golden/paper_values.txt -> {key: float}."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                k, v = line.split()
                out[k] = float(v)
    return out


@pytest.fixture(scope="session")
def golden():
    return load_golden()


def pytest_sessionstart(session):
    """Build libwick_b200.so in-tree if it is missing or older than its sources (nvcc cross-compiles
    sm_100a without a GPU).  The product path itself never builds or falls back: it raises."""
    from paper_2411_08962_b200.build import build_library
    build_library()


@pytest.fixture(scope="session")
def cuda_device():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("this test is marked gpu and needs a CUDA device (no CPU fallback exists)")
    return torch.device("cuda:0")
