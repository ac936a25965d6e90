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
    """The brute-force fp64 oracle (oracle/), built with gcc on first use."""
    from oracle import oracle as _o
    _o.build()
    return _o


@pytest.fixture(scope="session")
def hcgrid_lib():
    """The C-ABI CUDA library, built in-tree with nvcc if missing (no GPU needed to build)."""
    from paper_2012_13173_b200 import binding
    return binding.load_library()
