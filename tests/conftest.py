import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def oracle():
    import oracle.nb_oracle as orc
    orc.lib()
    return orc


@pytest.fixture(scope="session")
def nb():
    """The CUDA path through its C-ABI binding.  GPU tests must run the real library: a
    missing device or library is an error, never a skip to a fallback."""
    import torch
    import paper_1207_2367_b200 as nbmod
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    nbmod.lib()
    return nbmod
