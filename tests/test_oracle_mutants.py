"""Every one-line mistake listed in tests/mutants.py, applied to a scratch copy of the oracle, must be
caught by a pin (see that file).  ~1 minute: the mutants build and run four at a time."""
import os

import pytest

from tests import mutants


@pytest.mark.skipif(os.environ.get("SRHD_TEST_ORACLE_ROOT") is not None, reason="already inside a mutant run")
def test_every_mutant_is_killed():
    res = mutants.run_all()
    bad = [(n, v, t) for n, _, v, t in res if v != "KILLED"]
    assert not bad, bad
