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


def pytest_addoption(parser):
    parser.addoption("--runslow", action="store_true", default=False, help="also run the long oracle checks (marker `slow`)")


def pytest_collection_modifyitems(config, items):
    if config.getoption("--runslow") or "slow" in (config.getoption("-m") or ""):
        return
    skip = pytest.mark.skip(reason="long oracle check: run with --runslow (or -m slow)")
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)
