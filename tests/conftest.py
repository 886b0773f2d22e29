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
    """The CPU oracle (test infrastructure); builds oracle/libmuon_oracle.so with g++ on first use."""
    import oracle as _oracle
    _oracle.lib()
    return _oracle


@pytest.fixture(scope="session")
def mt():
    """The CUDA path's Python binding; builds the C-ABI library with nvcc if it is not there yet."""
    from paper_2512_10520_b200 import build as _build
    _build.build()
    import paper_2512_10520_b200 as _mt
    return _mt


@pytest.fixture(scope="session")
def workloads():
    from paper_2512_10520_b200 import workloads as _w
    return _w
