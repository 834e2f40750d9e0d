"""-m gpu: the production build's canonical quotients (VERDICT r1 #5/#6a).

The Eq. 30 verdict L = fma(x, x+2, -mu^2) is a discontinuous switch, so x = Etilde/D and u_i = M_i/D must be
the CORRECTLY ROUNDED quotients in both implementations.  The production build forms them as
q = a*y; r = fma(-b, q, a); q + r*y with y = 1/b from a MUFU seed and two Newton steps, and falls back to
IEEE division outside a wide exponent window.  srhd_quotient_check evaluates that device function and IEEE
division side by side on seeded pairs and counts the bit mismatches: there must be none.
"""
import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dist", ["config_ranges", "near_powers_of_two", "wide_exponents"])
def test_canonical_quotient_is_correctly_rounded(dist):
    # 2^32 pairs in total over the three distributions (counter-based generator on the device, seeded)
    n = (1 << 32) // 3
    mism, first = B.quotient_check(n, seed=20121113, dist={"config_ranges": 0, "near_powers_of_two": 1,
                                                           "wide_exponents": 2}[dist])
    assert mism == 0, (dist, mism, first)
