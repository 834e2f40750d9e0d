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
    # tests/mutants.py points SRHD_TEST_ORACLE_ROOT at a scratch tree holding a MUTATED copy of oracle/
    # (mutation check of the pins); it must win over the real one, which pytest keeps at sys.path[0]
    over = os.environ.get("SRHD_TEST_ORACLE_ROOT")
    if over:
        assert "oracle" not in sys.modules
        sys.path.insert(0, over)
    from oracle import ref as _ref
    if over:
        assert os.path.dirname(os.path.dirname(os.path.abspath(_ref.__file__))) == os.path.abspath(over)
    _ref.lib()
    return _ref


@pytest.fixture(scope="session", autouse=True)
def _built_libraries():
    """Make sure the in-tree C-ABI libraries exist and are current (nvcc cross-compiles without a GPU;
    a no-op when they are fresh).  The tests never fall back to anything else if this fails."""
    if os.environ.get("SRHD_TEST_SKIP_CUDA_BUILD"):
        return
    from paper_2012_11130_b200 import build
    build.build()
