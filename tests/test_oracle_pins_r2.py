"""Pins for the five oracle parts that had none ("What's weak" #1), each against something
that is not the oracle: 40-digit definitions (tests/mp_defs.py), identities of special relativity, the
jump conditions, the paper's own 3-D convergence test, and a Python re-assembly of one pass from per-state
calls (tests/py_step.py).  tests/mutants.py applies one-line mistakes to a copy of the oracle and
checks that these tests catch every one of them.  P:n = /root/reference/PAPER.md line n.
"""
import numpy as np
import pytest
from mpmath import asinh, cosh, mpf, sinh, sqrt

from paper_2012_11130_b200 import workloads as wl
from tests import mp_defs, py_step

EPS = np.finfo(np.float64).eps


def _p2c(ref, W):
    return ref.prim2cons(np.asarray(W, dtype=float).reshape(5, 1))[:, 0]


# ------------------------------------------------------------------ (a) Eq. 26, relativistic factors
def test_umax_is_the_relativistic_addition_of_flow_and_sound(ref):
    """P:237 Eq. 25: for sound along the flow the signal's four-velocity is beta gamma gamma_s + gamma U_s,
    i.e. the relativistic ADDITION of the two motions ("essentially the addition of flow speed and sound
    speed in special relativity"): sinh(asinh|U| + asinh U_s).  Eq. 26 bounds each component
    by |U^i| gamma_s + gamma U_s, so for a flow along one axis  U_max - 2 gamma U_s  is exactly that."""
    for T in (1e-6, 1.0, 1e4):
        cs2 = mp_defs.cs2_of_T(T)
        Us = sqrt(cs2 / (1 - cs2))                                   # U_s = c_s / sqrt(1 - c_s^2)
        for gamma in (2.0, 1e2, 1e4):
            U = float(np.sqrt((gamma - 1.0) * (gamma + 1.0)))
            for axis in range(3):
                for sign in (1.0, -1.0):
                    W = np.array([0.7, 0.0, 0.0, 0.0, 0.7 * T])
                    W[1 + axis] = sign * U
                    got = mpf(ref.umax_of_prim(W))
                    g = sqrt(1 + mpf(U) ** 2)
                    want = sinh(asinh(mpf(U)) + asinh(Us)) + 2 * g * Us
                    assert abs(got / want - 1) < 8 * EPS, (T, gamma, axis, float(got / want - 1))


def test_umax_sums_the_three_components_with_gamma_s(ref):
    """Eq. 26 sums |U^i| gamma_s over the components: two flows with the same Lorentz factor differ in
    U_max by gamma_s (|U^x|+|U^y|+|U^z| - |U|), gamma_s = cosh(asinh U_s) (reading G4)."""
    rng = np.random.default_rng(3)
    for T in (1e-4, 0.3, 50.0):
        cs2 = mp_defs.cs2_of_T(T)
        gs = cosh(asinh(sqrt(cs2 / (1 - cs2))))
        for _ in range(20):
            u = rng.standard_normal(3) * 10.0 ** rng.uniform(-1, 3)
            un = float(np.sqrt((u * u).sum()))
            a = mpf(ref.umax_of_prim(np.array([2.0, u[0], u[1], u[2], 2.0 * T])))
            b = mpf(ref.umax_of_prim(np.array([2.0, un, 0.0, 0.0, 2.0 * T])))
            l1 = sum(mpf(abs(x)) for x in u)
            # (a - b) is a difference of O(|U|) numbers: compare at the scale of a
            assert abs((a - b) - gs * (l1 - mpf(un))) < 16 * EPS * a


# ------------------------------------------------------------------ (b) wave-speed VALUES
def _hi_gamma_states():
    out = []
    rng = np.random.default_rng(11)
    for gamma in (1.0, 1.5, 10.0, 1e3, 1e6):
        for T in (1e-8, 1e-2, 1.0, 1e3):
            for _ in range(4):
                n = rng.standard_normal(3)
                n /= np.linalg.norm(n)
                U = np.sqrt((gamma - 1.0) * (gamma + 1.0)) * n
                out.append(np.array([1.3, U[0], U[1], U[2], 1.3 * T]))
    return out


def test_wave_speed_values_match_the_3velocity_eigenvalues(ref):
    """Reading S6 (4-velocity form) against the textbook 3-velocity acoustic eigenvalues in 40 digits,
    value for value, Lorentz factor up to 1e6 with tangential velocity, every direction."""
    for W in _hi_gamma_states():
        for d in range(3):
            lm, lp = ref.wave_speeds(d, W)
            em, ep = mp_defs.lambda_pm_3vel(W, d)
            assert abs(mpf(lm) - em) < 8 * EPS and abs(mpf(lp) - ep) < 8 * EPS, (W, d)
            assert -1 < lm < lp < 1 or (lp == 1.0 or lm == -1.0)   # |lambda| rounds to 1 only beyond fp64 resolution


def test_wave_speed_differences_keep_full_relative_accuracy(ref):
    """at Lorentz factor 1e6 lambda, v_n and 1 agree to 12 digits; their
    DIFFERENCES (which is what the HLL averages and the HLLC star state use) must still be accurate to a
    few ulp of THEMSELVES.  Against plain subtraction of the 40-digit 3-velocity eigenvalues."""
    for W in _hi_gamma_states():
        g = sqrt(1 + sum(mpf(x) ** 2 for x in W[1:4]))
        for d in range(3):
            got = ref.wave_speed_differences(d, W)
            em, ep = mp_defs.lambda_pm_3vel(W, d)
            vn = mpf(W[1 + d]) / g
            for val, want in zip(got[2:], (ep - vn, vn - em, 1 - ep, 1 + em)):
                assert want > 0 and abs(mpf(val) / want - 1) < 32 * EPS, (W, d, float(mpf(val) / want - 1))


# ------------------------------------------------------------------ (c) HLLE / HLLC values
def _pairs(n=60, gmax=30.0, seed=17):
    rng = np.random.default_rng(seed)
    W = wl.conversion_states(2 * n, seed=seed, log_gamma=(0, np.log10(gmax)), log_theta=(-6, 3), log_rho=(-1, 1))
    for i in range(n):
        WL, WR = W[:, 2 * i].copy(), W[:, 2 * i + 1].copy()
        if rng.random() < 0.5:                       # half of them nearly at rest: subsonic, star region active
            WL[1:4] *= 10.0 ** rng.uniform(-4, -1)
            WR[1:4] *= 10.0 ** rng.uniform(-4, -1)
        yield WL, WR


def _flux_scale(ref, WL, UL, WR, UR, d):
    """Per-component size of the terms the HLL averages combine: |S U| + |F| of both sides (|S| <= 1)."""
    FL, FR = ref.phys_flux(d, WL, UL), ref.phys_flux(d, WR, UR)
    return np.abs(UL) + np.abs(UR) + np.abs(FL) + np.abs(FR)


def test_hlle_satisfies_the_jump_conditions_across_both_waves(ref):
    """The HLL flux is DEFINED by the Rankine-Hugoniot conditions across the two bounding waves:
    F - F_L = S_L (U* - U_L) and F - F_R = S_R (U* - U_R) with ONE intermediate state U*, i.e.
    U_L + (F - F_L)/S_L == U_R + (F - F_R)/S_R, S from the 40-digit 3-velocity eigenvalues.  A wrong
    dissipative term or a wrong speed breaks it."""
    nstar = 0
    for WL, WR in _pairs():
        UL, UR = _p2c(ref, WL), _p2c(ref, WR)
        for d in range(3):
            SL, SR = mp_defs.hll_speeds(WL, WR, d)
            if not (SL < 0 < SR):
                continue
            nstar += 1
            F = [mpf(x) for x in ref.riemann_flux("hlle", d, WL, UL, WR, UR)]
            FL, FR = mp_defs.phys_flux(d, WL), mp_defs.phys_flux(d, WR)
            mUL, mUR = mp_defs.prim2cons(WL), mp_defs.prim2cons(WR)
            scale = _flux_scale(ref, WL, UL, WR, UR, d)
            for q in range(5):
                lhs = mUL[q] + (F[q] - FL[q]) / SL
                rhs = mUR[q] + (F[q] - FR[q]) / SR
                # dividing by a small |S| amplifies the fp64 rounding of F by 1/|S|
                tol = 64 * EPS * float(scale[q]) * (1 + 1 / float(min(-SL, SR)))
                assert abs(lhs - rhs) <= tol, (d, q, float(lhs - rhs), tol)
    assert nstar > 40


@pytest.mark.parametrize("name", ["hlle", "hllc"])
def test_riemann_flux_values_match_40_digit_definitions(ref, name):
    """HLLE and HLLC (reading S7: the Etilde adaptation) against the textbook total-energy forms with
    3-velocity eigenvalues in 40 digits, value for value, moderate Lorentz factors."""
    mp_flux = mp_defs.hlle_flux if name == "hlle" else mp_defs.hllc_flux
    nstar = 0
    for WL, WR in _pairs(seed=23):
        UL, UR = _p2c(ref, WL), _p2c(ref, WR)
        for d in range(3):
            SL, SR = mp_defs.hll_speeds(WL, WR, d)
            nstar += bool(SL < 0 < SR)
            F = ref.riemann_flux(name, d, WL, UL, WR, UR)
            Fe = mp_flux(WL, WR, d)
            scale = _flux_scale(ref, WL, UL, WR, UR, d)
            for q in range(5):
                assert abs(mpf(F[q]) - Fe[q]) <= 256 * EPS * float(scale[q]), (d, q, float(mpf(F[q]) - Fe[q]), scale[q])
    assert nstar > 40


def _ur_pairs():
    """Ultra-relativistic Riemann problems, Lorentz factor 1e3 ... 1e6: colliding, receding and co-moving
    streams against a slow or a fast partner, with tangential velocity, cold to hot."""
    rng = np.random.default_rng(29)
    for gamma in (1e3, 1e4, 1e6):
        U = np.sqrt((gamma - 1.0) * (gamma + 1.0))
        for T in (1e-6, 1.0, 1e3):
            for sL, sR in ((1, -1), (-1, 1), (1, 1), (0, 1), (-1, 0), (0, -1), (1, 0)):
                ut = rng.standard_normal(4) * 10.0 ** rng.uniform(-2, 1, 4)
                slow = rng.standard_normal(2) * 0.3
                WL = np.array([1.0, sL * U if sL else slow[0], ut[0], ut[1], T])
                WR = np.array([10.0 ** rng.uniform(-2, 2), sR * U if sR else slow[1], ut[2], ut[3], 0.0])
                WR[4] = WR[0] * T * 10.0 ** rng.uniform(-1, 1)
                yield WL, WR


@pytest.mark.parametrize("name", ["hlle", "hllc"])
def test_riemann_flux_at_lorentz_factor_1e3_to_1e6(ref, name):
    """The same 40-digit definitions at Lorentz factors 1e3 ... 1e6 (section 7: "S - v,
    1 - S ... must be formed without subtracting near-equal numbers").  The error of each flux
    component is measured against the size of the NON-cancelling pieces it is built from -- S U* and
    (S - v_n) U_K for the star flux, S_R (v_L - S_L) U_L and S_L (S_R - v_R) U_R for the HLL flux, plus
    the pressure terms -- evaluated in 40 digits: forming S - v_n by subtracting two fp64 speeds that agree
    to 12 digits loses all of that."""
    nstar = 0
    for WL, WR in _ur_pairs():
        UL, UR = _p2c(ref, WL), _p2c(ref, WR)
        for d in range(3):
            SL, SR = mp_defs.hll_speeds(WL, WR, d)
            nstar += bool(SL < 0 < SR)
            kappa = 1.0
            if name == "hlle" or not (SL < 0 < SR):
                Fe, pieces = (mp_defs.hlle_flux if name == "hlle" else mp_defs.hllc_flux)(WL, WR, d, pieces=True)
            else:
                Fe, pieces, kappa = mp_defs.hllc_flux(WL, WR, d, pieces=True)
            F = ref.riemann_flux(name, d, WL, UL, WR, UR)
            for q in range(5):
                # HLLC: the contact speed is the root of a quadratic whose roots merge at the light cone when
                # an ultra-relativistic stream runs into slow gas (condition number sqrt(kappa), up to 4e6 in
                # this list): that part of S7 is NOT reformulated -- DESIGN.md section 4 lists it
                tol = (512 + 2 * float(sqrt(kappa))) * EPS * pieces[q]
                assert abs(mpf(F[q]) - Fe[q]) <= tol, (name, WL, WR, d, q, float(mpf(F[q]) - Fe[q]), float(tol))
    assert nstar > 60


# ------------------------------------------------------------------ (d) section 4.1 as the paper runs it
def _diagonal_wave(ref, N, T0, amp=1e-6):
    """static homogeneous background rho_0 = 1 at temperature T0, a sound wave of amplitude
    delta rho / rho_0 = 1e-6 along the DIAGONAL of a periodic cube; eigenmode of the linearised equations
    (delta v = c_s delta rho / rho along k, delta p = h c_s^2 delta rho)."""
    cs = float(np.sqrt(ref.cs2_of_T(np.array([T0]))[0]))
    h = 1.0 + float(ref.htilde_of_T(np.array([T0]))[0])
    dh = 1.0 / N
    x = (np.arange(N) + 0.5) * dh
    ph = 2 * np.pi * (x[None, None, :] + x[None, :, None] + x[:, None, None])
    s = np.sin(ph)
    prim = np.zeros((5, N, N, N))
    prim[0] = 1.0 + amp * s
    for d in range(3):
        prim[1 + d] = cs * amp * s / np.sqrt(3.0)
    prim[4] = T0 * (1.0 + h * cs * cs / T0 * amp * s)
    k = 2 * np.pi * np.sqrt(3.0)
    return prim, dh, ph, k * cs, cs


def _run_wave(ref, N, T0, amp=1e-6):
    par = ref.params("plm", "hllc")
    prim, dh, ph, omega, cs = _diagonal_wave(ref, N, T0, amp)
    cons = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    t, t_end = 0.0, 0.5 * np.pi / omega                # a quarter of a period
    while t < t_end:
        dt = min(ref.cfl_dt(cons, 0.5, dh, par), t_end - t)
        cons, st = ref.grid_step_tiled(cons, dt, dh, par, ["periodic"] * 6)
        assert st.n_retry_pg == 0
        t += dt
    rho = ref.cons2prim(cons.reshape(5, -1))[0][0].reshape(N, N, N)
    exact = 1.0 + amp * np.sin(ph - omega * t_end)
    return float(np.abs(1.0 - rho / exact).mean())        # P:297 Eq. 31


@pytest.mark.parametrize("T0", [1e-10, 1e10])
def test_second_order_convergence_on_the_3d_diagonal_wave(ref, T0):
    """P:301 / Fig. 3: L1(rho) ~ N^-2 in the low- and high-temperature limits alike.  In three dimensions
    the order rests on the ONE common half-step increment of the unsplit predictor (reading S5)."""
    e16, e32, e64 = (_run_wave(ref, N, T0) for N in (16, 32, 64))
    assert e16 < 0.5e-6
    o1, o2 = np.log2(e16 / e32), np.log2(e32 / e64)
    assert o1 > 1.8 and o2 > 1.8, (e16, e32, e64, o1, o2)


@pytest.mark.parametrize("recon", ["plm", "ppm"])
def test_one_step_matches_40_digit_evaluation_of_the_definitions(ref, recon):
    """A handful of cells of a small 3-D box, one PLM/PPM + MUSCL-Hancock + HLLC/HLLE step, against
    tests/mp_defs.step_cells: total-energy definitions, numerical root finding, textbook eigenvalues,
    plain subtractions in 40 digits, its own loops.  Pins the assembly (stencils, the coupling of the three
    directions in the predictor, face pairing, update) and the Etilde formulation at once."""
    rng = np.random.default_rng(4)
    n, g = 3, ref.params(recon, "hllc").ghost
    s = n + 2 * g + 2                                 # one spare layer so the mp stencil stays inside
    k = 2 * np.pi * (np.arange(s) + 0.37) / 9.0
    Z, Y, X = np.meshgrid(k, 0.8 * k, 1.3 * k, indexing="ij")
    prim = np.empty((5, s, s, s))
    prim[0] = 1.0 + 0.4 * np.sin(X + 0.3) * np.cos(Y) + 0.05 * rng.standard_normal(X.shape)
    prim[1] = 0.6 * np.sin(Y + Z)
    prim[2] = -0.4 * np.cos(X - Z)
    prim[3] = 0.2 + 0.3 * np.sin(X + Y + Z)
    prim[4] = prim[0] * 10.0 ** (-1.0 + 0.7 * np.sin(Z) * np.sin(X))
    big = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    dh = 1.0 / 16
    dt = 0.4 * dh / ref.max_signal_speed(big.reshape(5, -1))
    tile = np.ascontiguousarray(big[:, 1:-1, 1:-1, 1:-1])
    for riemann in ("hllc", "hlle"):
        par = ref.params(recon, riemann)
        out, st, passes = ref.step_box(tile, dt, dh, par)
        assert passes == 1
        cells = [(0, 0, 0), (1, 2, 0), (2, 1, 2)] if recon == "plm" else [(1, 2, 0)]
        off = g + 1                                   # interior cell (i,j,k) sits at big[..., k+off, j+off, i+off]
        want = mp_defs.step_cells(big, [(i + off, j + off, k + off) for i, j, k in cells], dt, dh, riemann,
                                  recon=recon)
        for (i, j, k) in cells:
            w = want[(i + off, j + off, k + off)]
            scale = [abs(w[0]), abs(w[4]) + float(np.sqrt(sum(float(x) ** 2 for x in w[1:4]))), abs(w[4])]
            for q, sc in zip(range(5), (scale[0], scale[1], scale[1], scale[1], scale[2])):
                assert abs(mpf(out[q, k, j, i]) - w[q]) <= 2e-13 * float(sc), (riemann, (i, j, k), q)


# ------------------------------------------------------------------ (e) retry ladder (S9, S10, S15)
def _rough_box(ref, seed, ghost, n=4):
    prim = wl.random_patch_groups(1, ghost, seed=seed, umax=30.0, rough=3.0, log_theta=(-8.0, 2.0))[0]
    s = n + 2 * ghost
    prim = np.ascontiguousarray(prim[:, 3:3 + s, 2:2 + s, 4:4 + s])
    return ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)


# (recon, seed, dt / CFL-dt): chosen so that the ladder ends on every kind of rung -- see the asserts
LADDER_CASES = [("plm", 4, 6.0), ("plm", 12, 1.0), ("plm", 6, 2.5), ("ppm", 2, 1.0), ("ppm", 10, 1.0),
                ("ppm", 12, 1.0), ("ppm", 4, 6.0), ("plm", 4, 1.0)]


def test_retry_ladder_equals_its_python_reassembly(ref):
    """step_box against tests/py_step.ladder (reduce the minmod coefficient by a factor 0.75 until
    Eq. 30 passes, finally a vanished coefficient), bit for bit, with the same number of passes and the
    same counters, on boxes whose ladders end after 1, 2, 3, 4 passes and on the last rung."""
    seen, s15, final_bad = set(), 0, 0
    for recon, seed, mult in LADDER_CASES:
        par = ref.params(recon, "hllc", max_retry=3)
        cons = _rough_box(ref, seed, par.ghost)
        dh = 1.0 / 64
        dt = mult * 0.4 * dh / ref.max_signal_speed(cons.reshape(5, -1))
        out, passes, ff, cf, hist = py_step.ladder(ref, cons, dt, dh, par)
        got, st, got_passes = ref.step_box(cons, dt, dh, par)
        assert got_passes == passes, (recon, seed, mult, hist)
        assert np.array_equal(got, out, equal_nan=True)
        assert (st.n_retry_pg, st.n_c2p_fail, st.n_unphys_final) == (int(passes > 1), ff, cf)
        seen.add(passes)
        # S15: a pass whose updated cells are all physical but a half-step face state is not must retry
        s15 += sum(1 for (_, f, c) in hist[:-1] if f > 0 and c == 0)
        final_bad += int(cf > 0)
        if 1 < passes <= par.max_retry + 1:
            # the accepted rung k is a single pass with the coefficient 1.5 * 0.75^k
            beta = par.minmod_coeff
            for _ in range(passes - 1):
                beta *= 0.75
            single, _, p1 = ref.step_box(cons, dt, dh, ref.params(recon, "hllc", minmod_coeff=beta, max_retry=0))
            if recon == "plm":                        # (PPM blends by beta/beta0: another beta0, another blend)
                assert p1 == 1 and np.array_equal(single, got)
    assert seen == {1, 2, 3, 4, 5} and s15 >= 3 and final_bad >= 2, (seen, s15, final_bad)


@pytest.mark.parametrize("recon", ["plm", "ppm"])
def test_vanished_coefficient_is_first_order_godunov(ref, recon):
    """"interpolating with a vanished minmod coefficient is essentially equivalent to the piece-wise
    constant spatial reconstruction": the last rung equals a first-order Godunov update assembled in numpy
    from cell-centre states (edge states = cell states, zero predictor increment)."""
    par = ref.params(recon, "hllc", max_retry=1)
    seed, mult = (6, 2.5) if recon == "plm" else (4, 6.0)
    cons = _rough_box(ref, seed, par.ghost)
    dh = 1.0 / 64
    dt = mult * 0.4 * dh / ref.max_signal_speed(cons.reshape(5, -1))
    got, st, passes = ref.step_box(cons, dt, dh, par)
    assert passes == 3                                # beta0, 0.75 beta0, 0
    g, n = par.ghost, 4
    W = ref.cons2prim(cons.reshape(5, -1), par)[0]
    Ub = ref.prim2cons(W)                             # the edge state of a constant cell: p2c(c2p(U)) + (-0)
    Wb = ref.cons2prim(Ub, par)[0].reshape(cons.shape)
    Ub = Ub.reshape(cons.shape)
    out = cons[:, g:-g, g:-g, g:-g].copy()
    tot = np.zeros_like(out)
    for d, ax in ((0, 3), (1, 2), (2, 1)):
        F = {}
        for k in range(n):
            for j in range(n):
                for i in range(n):
                    for sh in (-1, 0):
                        c = [k + g, j + g, i + g]
                        c[ax - 1] += sh
                        r = list(c)
                        r[ax - 1] += 1
                        F[(k, j, i, sh)] = ref.riemann_flux("hllc", d, Wb[(slice(None), *c)], Ub[(slice(None), *c)],
                                                            Wb[(slice(None), *r)], Ub[(slice(None), *r)])
                    df = F[(k, j, i, 0)] - F[(k, j, i, -1)]
                    tot[:, k, j, i] = df if d == 0 else tot[:, k, j, i] + df      # ((x)+(y))+(z), S12
    out = out - (dt / dh) * tot
    assert np.array_equal(got, out, equal_nan=True)
