import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import avmo
    avmo.build()
    return avmo


@pytest.fixture(scope="session")
def g0():
    from paper_2509_15377_b200.gen import gas
    return gas.gas_g0()


@pytest.fixture(scope="session")
def avm():
    """The CUDA path through its C ABI.  Fails loudly when the library or a GPU is missing."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu test selected but no CUDA device is visible")
    from paper_2509_15377_b200 import build
    build.build()                         # no-op when libavm.so is newer than its sources (nvcc is on the GPU box too)
    from paper_2509_15377_b200 import avm as _avm
    return _avm
