import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running oracle checks (excluded from the default CPU run)")


@pytest.fixture(scope="session")
def lib():
    """The built CUDA library through its ctypes binding (built on demand; nvcc cross-compiles without a GPU)."""
    import __graft_entry__ as g
    g.build()
    import paper_2503_20700_b200 as P
    return P
