import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def phylino_lib():
    """libphylino.so, (re)built in-tree with nvcc if missing or stale.  No GPU needed to build/load."""
    from paper_2502_15253_b200 import build as _b
    _b.build()
    import paper_2502_15253_b200 as pkg
    return pkg


@pytest.fixture(scope="session")
def gpu(phylino_lib):
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    return phylino_lib
