"""Pin of the App.-C exact TM Riemann solver (oracle/exact_riemann.py) to the paper's Table 2."""
import os

import numpy as np
import pytest
from mpmath import mpf

GOLD = os.path.join(os.path.dirname(__file__), "golden", "table2_mixed_limits_exact.txt")


@pytest.fixture(scope="module")
def mixed():
    from oracle.exact_riemann import ExactRiemann
    # Table 1 row 2: left (rho,U,p) = (1e2, 1e-3, 1e-4), right (1e-12, -1e2, 1e-10)
    return ExactRiemann((1e2, 1e-3, 1e-4), (1e-12, -1e2, 1e-10))


def test_table2_star_region_and_waves(mixed):
    rows = np.loadtxt(GOLD)
    # rows 14/15: left of the contact; row 16/17: right of the contact
    assert float(mixed.p_star) == pytest.approx(rows[14, 3], rel=2e-15)
    assert float(mixed.U_star) == pytest.approx(rows[14, 2], rel=2e-15)
    assert float(mixed.rho_CL) == pytest.approx(rows[14, 1], rel=2e-15)
    assert float(mixed.rho_CR) == pytest.approx(rows[16, 1], rel=2e-15)
    assert mixed.L.kind == "rarefaction" and mixed.R.kind == "shock"
    x0, t = 0.05, 80.0
    # wave positions lie between the printed row pairs that straddle them (one cell apart)
    assert rows[1, 0] <= x0 + float(mixed.L.xi_head) * t <= rows[2, 0]
    assert rows[13, 0] <= x0 + float(mixed.L.xi_tail) * t <= rows[14, 0] + 1e-12
    assert rows[15, 0] <= x0 + float(mixed.v_star) * t <= rows[16, 0]
    assert rows[17, 0] <= x0 + float(mixed.R.xi_head) * t <= rows[18, 0]


def test_table2_rarefaction_fan_rows(mixed):
    rows = np.loadtxt(GOLD)
    x0, t = mpf("0.05"), mpf(80)
    for i in (3, 6, 9, 12, 13):                         # fan interior rows
        rho, U, p = mixed.sample((mpf(float(rows[i, 0])) - x0) / t)
        assert float(rho) == pytest.approx(rows[i, 1], rel=4e-15)
        assert float(U) == pytest.approx(rows[i, 2], rel=4e-15)
        assert float(p) == pytest.approx(rows[i, 3], rel=4e-15)


def test_fast_profile_agrees_with_table2(mixed):
    rows = np.loadtxt(GOLD)
    rho, U, p = mixed.profile((rows[:, 0] - 0.05) / 80.0)
    assert np.abs(rho / rows[:, 1] - 1).max() < 1e-7
    assert np.abs(p / rows[:, 3] - 1).max() < 1e-7
    assert np.abs(U / rows[:, 2] - 1).max() < 1e-7      # incl. the 4.6e-10 round-off of the printed row 16
