import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def ref():
    """The CPU oracle binding (builds oracle/libsrhd_ref.so on first use)."""
    from oracle import ref as _ref
    _ref.lib()
    return _ref


@pytest.fixture(scope="session", autouse=True)
def _built_libraries():
    """Make sure the in-tree C-ABI libraries exist and are current (nvcc cross-compiles without a GPU;
    a no-op when they are fresh).  The tests never fall back to anything else if this fails."""
    from paper_2012_11130_b200 import build
    build.build()
