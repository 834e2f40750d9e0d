"""Pins for the oracle's EoS and conversions (O1-O4) against what the paper and mathematics fix.

Every check compares the oracle with something that is NOT the oracle: 40-digit mpmath evaluation
of the paper's plain definitions (tests/mp_defs.py), closed-form limits, or the paper's own error
bound (Eq. 20).  Citations: P:n = /root/reference/PAPER.md line n.
"""
import numpy as np
import pytest
from mpmath import mp, mpf, sqrt, diff

from paper_2012_11130_b200 import workloads
from tests import mp_defs

EPS = np.finfo(np.float64).eps
T_GRID = 10.0 ** np.linspace(-10, 6, 65)


def test_taub_equality_and_limits(ref):
    # TM EoS satisfies Taub's inequality (Eq. 12) with EQUALITY: (h-T)(h-4T) = 1
    for T in T_GRID:
        h = mpf(1) + mpf(float(ref.htilde_of_T(T)))
        # evaluate the identity in 40 digits with the oracle's fp64 htilde: residual ~ eps*h^2
        res = (h - mpf(T)) * (h - 4 * mpf(T)) - 1
        assert abs(res) <= 8 * EPS * float(h) ** 2
    # limits: htilde -> 2.5 T (cold), -> 4 T (hot)   (Eq. 10 / Eq. 22)
    assert ref.htilde_of_T(1e-10) == pytest.approx(2.5e-10, rel=1e-9)
    assert ref.htilde_of_T(1e8) == pytest.approx(4e8, rel=1e-8)


def test_htilde_matches_eq10_in_extended_precision(ref):
    # Eq. 22 must equal Eq. 10 - 1: plain definition in 40 digits
    for T in T_GRID:
        exact = mp_defs.h_of_T(T) - 1
        assert abs(mpf(float(ref.htilde_of_T(T))) / exact - 1) < 4 * EPS


def test_T_of_htilde_inverts_eq22(ref):
    # Eq. 16 inverts Eq. 10: compare with a 40-digit numerical inversion of Eq. 10
    for T in T_GRID:
        ht = ref.htilde_of_T(T)
        _, T_exact = mp_defs.f_eq15(ht, 0.0)
        assert abs(mpf(float(ref.T_of_htilde(ht))) / T_exact - 1) < 4 * EPS
        assert abs(ref.T_of_htilde(ht) / T - 1) < 8 * EPS          # round trip <= few ulp


def test_sound_speed_limits_and_definition(ref):
    # c_s -> 1/sqrt(3) (hot); Newtonian c_s^2 = (5/3) T (cold, Gamma = 5/3)
    assert ref.cs2_of_T(1e9) == pytest.approx(1.0 / 3.0, rel=1e-8)
    assert ref.cs2_of_T(1e-10) / 1e-10 == pytest.approx(5.0 / 3.0, rel=1e-9)
    # thermodynamic definition c_s^2 = (dp/de)_s with e = rho(h - T)... use the equivalent
    # c_s^2 = T h' / (h (h' - 1)) for h(T) of Eq. 10 (Mignone+ 2005): derivative taken numerically
    for T in T_GRID[::4]:
        hp = diff(mp_defs.h_of_T, mpf(T))
        exact = mpf(T) * hp / (mp_defs.h_of_T(T) * (hp - 1))
        assert abs(mpf(float(ref.cs2_of_T(T))) / exact - 1) < 8 * EPS


def _states(n=4000):
    # config-2 box (BASELINE.json configs[1]) at test size
    return workloads.conversion_states(n, seed=201211130)


def test_prim2cons_vs_plain_definition_extended_precision(ref):
    # O2 against Eq. 5a-5c + Eq. 6 in 40 digits; gate 1e-14 over Theta in [1e-10,1e6], gamma<=1e6
    W = _states(1500)
    U = ref.prim2cons(W)
    worst = 0.0
    for i in range(W.shape[1]):
        Ue = mp_defs.prim2cons(W[:, i])
        errs = [abs(mpf(float(U[q, i])) / Ue[q] - 1) for q in (0, 4)]
        Mn = sqrt(sum(Ue[q] ** 2 for q in (1, 2, 3)))
        errs += [abs(mpf(float(U[q, i])) - Ue[q]) / Mn for q in (1, 2, 3)]
        worst = max(worst, float(max(errs)))
    assert worst < 1e-14


def test_plain_fp64_definition_fails_for_cold_gas():
    # The paper's point: E - D by Eq. 5c + Eq. 6 in fp64 loses the thermal energy.
    W = np.array([1.0, 1e-6, 0.0, 0.0, 1e-12])         # cold, slow
    rho, ux, p = W[0], W[1], W[4]
    T = p / rho
    h = 2.5 * T + np.sqrt(2.25 * T * T + 1.0)
    g = np.sqrt(1 + ux * ux)
    naive = rho * g * h * g - p - rho * g
    exact = float(mp_defs.prim2cons(W)[4])
    assert abs(naive / exact - 1) > 1e-6               # catastrophic


def test_cons2prim_inverts_exactly_rounded_conserved(ref):
    # O3 pinned independently of the oracle's own P2C: conserved values computed in 40 digits from
    # the plain definitions, rounded to fp64, must invert to the primitives within the paper's
    # bound C*(1+Mach^2)*eps (Eq. 20), C = 16, on well-conditioned states.
    W = _states(1500)
    U = np.array([[float(x) for x in mp_defs.prim2cons(W[:, i])] for i in range(W.shape[1])]).T
    W2, ht, it, bad = ref.cons2prim(U, diag=True)
    T = W[4] / W[0]
    cs2 = np.array([float(mp_defs.cs2_of_T(t)) for t in T])
    mach2 = (W[1:4] ** 2).sum(0) / (cs2 / (1 - cs2))
    cond = (1 + mach2) * EPS
    ok = cond < 1e-3
    assert ok.sum() > 500
    assert not bad[cond < 1e-4].any()
    ht0 = np.array([float(mp_defs.h_of_T(t) - 1) for t in T])
    err = np.abs(1 - ht0 / ht)                          # App. B protocol
    assert (err[ok] <= 16 * cond[ok]).all()
    rel_p = np.abs(W2[4] / W[4] - 1)
    assert (rel_p[ok] <= 64 * cond[ok]).all()
    assert (np.abs(W2[0] / W[0] - 1)[ok] <= 64 * cond[ok]).all()
    assert it.max() <= 7


def test_round_trip_fig16_protocol(ref):
    # P:626, Fig. 16: T = 1e-8, U || (1,1,1), Mach 1e-4..1e6: error ~ eps for M<1, ~M^2 eps above
    W, mach = workloads.mach_sweep_states(theta=1e-8, n=81)
    Us = np.sqrt(ref.cs2_of_T(1e-8) / (1 - ref.cs2_of_T(1e-8)))
    W[1:4] *= (mach * Us)[None, :]
    W2, ht2, it, bad = ref.cons2prim(ref.prim2cons(W), diag=True)
    ht0 = ref.htilde_of_T(W[4] / W[0])
    err = np.abs(1 - ht0 / ht2)
    bound = 16 * (1 + mach ** 2) * EPS
    sel = mach < 1e6
    assert (err[sel] <= bound[sel]).all()
    assert err[mach < 0.5].max() < 8 * EPS              # flat part of Fig. 16
    assert err[(mach > 1e4) & sel].max() > 1e-10        # and it does grow like M^2 (not better than physics)


def test_f_matches_eq15_and_is_monotone(ref):
    rng = np.random.default_rng(1)
    for _ in range(200):
        ht = 10.0 ** rng.uniform(-10, 7)
        musq = 10.0 ** rng.uniform(-12, 12)
        fe, _ = mp_defs.f_eq15(ht, musq)
        assert abs(mpf(float(ref.f_eq15(ht, musq))) / fe - 1) < 32 * EPS
        assert ref.f_eq15(ht * 1.001, musq) > ref.f_eq15(ht, musq)        # P:155 monotone
        # A1/A2: derivative of the 40-digit Eq. 15 taken numerically
        dfe = diff(lambda x: mp_defs.f_eq15(x, musq)[0], mpf(ht), h=mpf(ht) * mpf(10) ** -12)
        assert abs(mpf(float(ref.df_eqA1(ht, musq))) / dfe - 1) < 1e-9


def test_initial_guess_asymptotes(ref):
    # A3 series: f = 1.2 ht + (43/125 + 4/(25 s)) ht^2 ; A5: f/ht^2 -> 9/16
    for musq in (0.0, 1.0, 100.0):
        s = 1 + musq
        ht = 1e-5
        series = 1.2 * ht + (43.0 / 125 + 4.0 / (25 * s)) * ht * ht
        assert ref.f_eq15(ht, musq) == pytest.approx(series, rel=1e-9)
        assert ref.f_eq15(1e9, musq) / 1e18 == pytest.approx(9.0 / 16, rel=1e-8)
        # corrected A4 (reading G2) is the positive root of A3: plug back
        L = 1e-3
        g = ref.htilde_guess(L, musq)
        assert 1.2 * g + (43.0 / 125 + 4.0 / (25 * s)) * g * g == pytest.approx(L, rel=1e-12)
        # A4 = A6 at the threshold A7: continuity of the guess across the switch
        thr = (1800.0 * s / (437.0 * musq + 117.0)) ** 2
        lo, hi = ref.htilde_guess(thr * (1 - 1e-12), musq), ref.htilde_guess(thr * (1 + 1e-12), musq)
        assert lo == pytest.approx(hi, rel=1e-9)
        assert hi == pytest.approx(4.0 / 3 * np.sqrt(thr), rel=1e-9)


def test_guess_quality_and_iteration_count(ref):
    W = _states(20000)
    U = ref.prim2cons(W)
    W2, ht, it, bad = ref.cons2prim(U, diag=True)
    good = bad == 0
    assert 0.02 < 1 - good.mean() < 0.10                 # ~5.6 % of the config-2 box violates Eq. 30
    ux = U[1:4] / U[0]
    musq = (ux ** 2).sum(0)
    x = U[4] / U[0]
    L = x * (x + 2) - musq
    # the numpy L above is not the canonical fma sequence: keep states where that cannot matter
    well = good & (musq * EPS < 1e-6 * np.abs(L))
    assert well.sum() > 5000
    guess = np.array([ref.htilde_guess(l, m) for l, m in zip(L[well][:3000], musq[well][:3000])])
    ratio = guess / ht[well][:3000]
    assert 0.9 < ratio.min() and ratio.max() < 1.2
    assert it[good].max() <= 7


def test_unphysical_input_is_flagged_and_finite(ref):
    # Eq. 30 + reading S10: failing states are counted, clamped, and give finite output
    U = np.array([[1.0, 1.0, 1.0, -1.0],          # D
                  [10.0, 0.0, 0.0, 0.0],          # Mx  (|M|/D = 10 with tiny Etilde -> L < 0)
                  [0.0, 0.0, 0.0, 0.0],
                  [0.0, 0.0, 0.0, 0.0],
                  [1e-3, -1e-3, 1e-3, 1e-3]])     # Etilde
    W, st = ref.cons2prim(U)
    assert st.n_c2p_fail == 3                       # states 0 (L<0), 1 (E<0), 3 (D<0)
    assert np.isfinite(W).all()


def test_dt_newtonian_limit_and_ultrarelativistic_limit(ref):
    # P:259 Eq. 29: S_max -> |vx|+|vy|+|vz|+3 c_s for gamma ~ 1
    T = 1e-9
    W = np.array([1.0, 1e-4, -2e-4, 3e-4, T])
    cs = np.sqrt(5.0 / 3 * T)
    s = ref.smax_of_umax(ref.umax_of_prim(W))
    assert s == pytest.approx(6e-4 + 3 * cs, rel=1e-6)
    # S_max -> 1 for gamma >> 1, with 1 - S_max ~ 1/(2 U_max^2)
    W = np.array([1.0, 1e5, 0.0, 0.0, 1.0])
    um = ref.umax_of_prim(W)
    assert 1 - ref.smax_of_umax(um) == pytest.approx(0.5 / um ** 2, rel=1e-3)
    # max_signal_speed over a list == max of the per-state values (order independent)
    Wl = workloads.conversion_states(500, seed=3, log_gamma=(0, 2))
    U = ref.prim2cons(Wl)
    per = max(ref.smax_of_umax(ref.umax_of_prim(ref.cons2prim(U[:, i:i + 1])[0][:, 0])) for i in range(U.shape[1]))
    assert ref.max_signal_speed(U) == per
