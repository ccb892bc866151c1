import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import dgo
    dgo.lib()
    return dgo


@pytest.fixture(scope="session")
def dg():
    """The Python binding over libdg.so.  Builds the library if it is missing (nvcc cross-compiles without a GPU);
    a failure to build or load is an error, never a skip: there is no fallback path."""
    from paper_2509_25347_b200 import build
    build.build()
    from paper_2509_25347_b200 import binding
    return binding


@pytest.fixture(scope="session")
def cuda(dg):
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    torch.cuda.set_device(0)
    return torch.device("cuda:0")
