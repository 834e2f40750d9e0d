"""Pins for the oracle's fluxes, Riemann solvers (O6/O7) and reconstruction (O5b).

Compared against: 40-digit evaluation of the defining fluxes (tests/mp_defs.py), the Newtonian
Euler fluxes in the NR limit, the textbook 3-velocity eigenvalues, and the defining properties of
HLLC/HLLE/PLM/PPM.  P:n = /root/reference/PAPER.md line n.
"""
import numpy as np
import pytest
from mpmath import mpf

from paper_2012_11130_b200 import workloads
from tests import mp_defs

EPS = np.finfo(np.float64).eps


def _p2c(ref, W):
    return ref.prim2cons(np.asarray(W, dtype=float).reshape(5, 1))[:, 0]


def test_phys_flux_vs_defining_form_extended_precision(ref):
    # Eq. 4a, 4b and Eq. 7: (Etilde+p) U/gamma == (M - D U/gamma) exactly
    W = workloads.conversion_states(300, seed=11, log_gamma=(0, 4))
    for i in range(W.shape[1]):
        U = _p2c(ref, W[:, i])
        for d in range(3):
            F = ref.phys_flux(d, W[:, i], U)
            Fe = mp_defs.phys_flux(d, W[:, i])
            scale = max(abs(x) for x in Fe[1:4]) + abs(Fe[4]) + abs(Fe[0])
            for q in range(5):
                assert abs(mpf(float(F[q])) - Fe[q]) <= 16 * EPS * scale
            # the energy flux itself is accurate in a RELATIVE sense (no cancellation):
            if abs(Fe[4]) > 0:
                assert abs(mpf(float(F[4])) / Fe[4] - 1) < 64 * EPS


def test_newtonian_limit_of_conserved_and_fluxes(ref):
    # T, v^2 << 1: D->rho, M->rho v, Etilde -> rho v^2/2 + 1.5 p, F_E -> (rho v^2/2 + 2.5 p) v
    rho, v, p = 2.0, np.array([3e-5, -1e-5, 2e-5]), 4e-10
    W = np.array([rho, *v, p])          # U ~ v at this order
    U = _p2c(ref, W)
    v2 = (v * v).sum()
    assert U[0] == pytest.approx(rho, rel=1e-8)
    assert np.allclose(U[1:4], rho * v, rtol=1e-8)
    assert U[4] == pytest.approx(0.5 * rho * v2 + 1.5 * p, rel=1e-8)
    for d in range(3):
        F = ref.phys_flux(d, W, U)
        assert F[0] == pytest.approx(rho * v[d], rel=1e-8)
        Fm = rho * v * v[d]
        Fm[d] += p
        assert np.allclose(F[1:4], Fm, rtol=1e-8)
        assert F[4] == pytest.approx((0.5 * rho * v2 + 2.5 * p) * v[d], rel=1e-8)


def test_wave_speeds_match_textbook_3velocity_form(ref):
    # reading S6: supersonic iff lambda_- > 0.  The HLLE flux of (L=W, R=W') equals F(L) exactly
    # iff min(lambda_-) >= 0.  Use a boosted family to bracket the sonic point predicted by the
    # 3-velocity eigenvalue formula evaluated in 40 digits.
    for T, ut in ((1e-6, 0.0), (1e-2, 0.5), (10.0, 3.0)):
        from mpmath import findroot
        f = lambda un: mp_defs.lambda_pm_3vel([1.0, un, ut, 0.0, T], 0)[0]
        un0 = float(findroot(f, 0.5 * np.sqrt(T) + 0.1, verify=False))
        for un, sup in ((un0 * (1 + 1e-6), True), (un0 * (1 - 1e-6), False)):
            WL = np.array([1.0, un, ut, 0.0, T])
            WR = np.array([0.5, un, ut, 0.0, 0.5 * T])        # same T and velocity: same eigenvalues
            UL, UR = _p2c(ref, WL), _p2c(ref, WR)
            F = ref.riemann_flux("hlle", 0, WL, UL, WR, UR)
            same = np.array_equal(F, ref.phys_flux(0, WL, UL))
            assert same == sup


def test_riemann_consistency_and_mirror(ref):
    rng = np.random.default_rng(5)
    W = workloads.conversion_states(200, seed=13, log_gamma=(0, 1.5), log_theta=(-6, 3))
    for i in range(0, 200, 2):
        WL, WR = W[:, i].copy(), W[:, i + 1].copy()
        WR[0] = WL[0] * 10 ** rng.uniform(-1, 1)
        UL, UR = _p2c(ref, WL), _p2c(ref, WR)
        for name in ("hlle", "hllc"):
            for d in range(3):
                # consistency: identical states give the physical flux
                F = ref.riemann_flux(name, d, WL, UL, WL, UL)
                Fp = ref.phys_flux(d, WL, UL)
                assert np.allclose(F, Fp, rtol=1e-13, atol=1e-13 * np.abs(Fp).max())
                # mirror: x -> -x, U_n -> -U_n, L <-> R flips the sign of the even-in-U_n fluxes
                F = ref.riemann_flux(name, d, WL, UL, WR, UR)
                ml, mr = WL.copy(), WR.copy()
                ml[1 + d] *= -1
                mr[1 + d] *= -1
                Fm = ref.riemann_flux(name, d, mr, _p2c(ref, mr), ml, _p2c(ref, ml))
                sign = -np.ones(5)
                sign[1 + d] = 1.0
                # the flux can be many orders below the states it is a difference of (a hot, fast
                # left state against a cold one: |F| ~ 1e-2, |U| ~ 1e11), so the absolute
                # tolerance is set by the size of the inputs of the HLL averages
                scale = max(np.abs(F).max(), np.abs(UL).max(), np.abs(UR).max())
                assert np.allclose(Fm, sign * F, rtol=1e-11, atol=1e-13 * scale)


def test_hllc_resolves_isolated_contact_hlle_does_not(ref):
    # defining property of HLLC (Mignone & Bodo 2005): equal p and U_n... equal v_n; rho, U_t jump
    for vn, rho_ratio in ((0.3, 1e-3), (0.2, 1e3), (-0.5, 1e7)):      # all subsonic: S_L < 0 < S_R
        p = 0.7
        # equal normal 3-VELOCITY on both sides with different tangential velocities
        def state(rho, vt):
            g = 1.0 / np.sqrt(1 - vn * vn - vt * vt)
            return np.array([rho, g * vn, g * vt, 0.0, p])
        WL, WR = state(1.0, 0.2), state(rho_ratio, -0.3)
        UL, UR = _p2c(ref, WL), _p2c(ref, WR)
        F = ref.riemann_flux("hllc", 0, WL, UL, WR, UR)
        Fup = ref.phys_flux(0, WL, UL) if vn > 0 else ref.phys_flux(0, WR, UR)
        assert np.allclose(F, Fup, rtol=1e-10, atol=1e-10 * np.abs(Fup).max())
        Fe = ref.riemann_flux("hlle", 0, WL, UL, WR, UR)
        assert abs(Fe[0] / Fup[0] - 1) > 0.01             # HLLE smears the contact


def test_hllc_flux_between_hll_bounds_and_supersonic_upwinding(ref):
    W = np.array([1.0, 5.0, 0.1, 0.0, 1e-3])              # supersonic to the right
    W2 = np.array([2.0, 6.0, 0.0, 0.1, 2e-3])
    U, U2 = _p2c(ref, W), _p2c(ref, W2)
    for name in ("hlle", "hllc"):
        assert np.array_equal(ref.riemann_flux(name, 0, W, U, W2, U2), ref.phys_flux(0, W, U))
        Wl, W2l = W.copy(), W2.copy()
        Wl[1] *= -1
        W2l[1] *= -1
        assert np.array_equal(ref.riemann_flux(name, 0, Wl, _p2c(ref, Wl), W2l, _p2c(ref, W2l)),
                              ref.phys_flux(0, W2l, _p2c(ref, W2l)))


# ------------------------------------------------------------------ reconstruction (S3, S4)
def test_limiter_properties(ref):
    ls = ref.limited_slope
    assert ls(1.0, -1.0, 1.5) == 0.0 and ls(0.0, 1.0, 1.5) == 0.0
    assert ls(1.0, 1.0, 1.5) == 1.0                       # linear data reproduced
    assert ls(-2.0, -2.0, 1.0) == -2.0
    assert ls(1.0, 3.0, 2.0) == pytest.approx(1.5)        # harmonic mean 2*1*3/4
    assert ls(1.0, 9.0, 1.5) == pytest.approx(1.5)        # minmod cap beta*min binds (harmonic = 1.8)
    assert ls(1.0, 9.0, 0.0) == 0.0                       # beta = 0 -> piecewise constant
    rng = np.random.default_rng(0)
    for _ in range(500):
        a, b = rng.standard_normal(2)
        s = ls(a, b, 1.5)
        assert ls(b, a, 1.5) == s and ls(-a, -b, 1.5) == -s          # symmetric, odd
        assert abs(s) <= 1.5 * min(abs(a), abs(b)) + 1e-300


@pytest.mark.parametrize("recon", [0, 1])
def test_reconstruction_properties(ref, recon):
    rng = np.random.default_rng(2)
    # linear data: exact edges a_i -+ slope/2
    a = 3.0 + 0.25 * np.arange(5)
    am, ap = ref.recon_1d(recon, a, 1.5, 1.5)
    assert am == pytest.approx(a[2] - 0.125, abs=1e-15) and ap == pytest.approx(a[2] + 0.125, abs=1e-15)
    # beta = 0: piecewise constant
    am, ap = ref.recon_1d(recon, rng.standard_normal(5), 0.0, 1.5)
    for _ in range(1000):
        a = rng.standard_normal(5) * 10 ** rng.uniform(-3, 3)
        am, ap = ref.recon_1d(recon, a, 1.5, 1.5)
        lo, hi = min(a[1], a[2], a[3]), max(a[1], a[2], a[3])
        assert lo - 1e-12 * abs(lo) <= am <= hi + 1e-12 * abs(hi)     # bounded by neighbours
        assert lo - 1e-12 * abs(lo) <= ap <= hi + 1e-12 * abs(hi)
        if (a[3] - a[2]) * (a[2] - a[1]) <= 0:                        # extremum -> flat
            assert am == a[2] and ap == a[2]
        else:                                                          # monotone profile in the cell
            assert (ap - a[2]) * (a[2] - am) >= 0
        z0, z1 = ref.recon_1d(recon, a, 0.0, 1.5)
        assert z0 == a[2] and z1 == a[2]
        # retry blend shrinks the edges toward the cell value monotonically
        bm, bp = ref.recon_1d(recon, a, 1.5 * 0.75 ** 3, 1.5)
        assert abs(bm - a[2]) <= abs(am - a[2]) * (1 + 1e-12) and abs(bp - a[2]) <= abs(ap - a[2]) * (1 + 1e-12)


def test_ppm_is_fourth_order_face_interpolation_on_smooth_data(ref):
    # CW84: unlimited face value = 7/12 (a_i + a_{i+1}) - 1/12 (a_{i-1} + a_{i+2}) for smooth data
    x = np.arange(-2, 3) * 0.01
    a = 1.0 + x + 0.5 * x ** 2          # cell values of a smooth (monotone here) profile
    am, ap = ref.recon_1d(1, a, 2.0, 2.0)
    # with van Leer slopes the face differs from the 4th-order value only at O(h^3)
    f_hi = 7.0 / 12 * (a[2] + a[3]) - 1.0 / 12 * (a[1] + a[4])
    f_lo = 7.0 / 12 * (a[1] + a[2]) - 1.0 / 12 * (a[0] + a[3])
    assert ap == pytest.approx(f_hi, abs=5e-7) and am == pytest.approx(f_lo, abs=5e-7)
