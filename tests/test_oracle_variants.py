"""Pins for the oracle's compile-time variants (oracle/srhd_ref.cpp header):
the polytropic EoS of P:107 Eq. 11 (Gamma = 5/3, 4/3) and the paper's "original scheme" that evolves the total
energy E (section 4, App. B), pinned against the definitions in 40-digit arithmetic, against
the paper's own error estimates Eq. 20 / 21 / 32 and its Fig. 3 / Fig. 16 statements, and against each other.
"""
import numpy as np
import pytest
from mpmath import mp, mpf, sqrt, diff

from paper_2012_11130_b200 import workloads

mp.dps = 40
EPS = np.finfo(float).eps
GAMMAS = {"gamma53": (5, 3), "gamma43": (4, 3)}


def _h_gamma(T, num, den):
    return 1 + mpf(num) / (num - den) * mpf(T)


# ------------------------------------------------------------------ polytropic EoS (Eq. 11)
@pytest.mark.parametrize("name", sorted(GAMMAS))
def test_gamma_law_eos_is_eq11(ref, name):
    num, den = GAMMAS[name]
    with ref.variant(name):
        for T in 10.0 ** np.linspace(-10, 8, 37):
            ht = ref.htilde_of_T(float(T))
            assert abs(mpf(ht) - (_h_gamma(T, num, den) - 1)) <= 2 * EPS * mpf(ht)
            assert abs(ref.T_of_htilde(ht) / T - 1) <= 4 * EPS
            # c_s^2 = (dp/drho)_s / h on the isentrope p = K rho^Gamma, by numerical differentiation in 40 digits
            G = mpf(num) / den
            p_of_rho = lambda r: mpf(T) * r ** G           # K chosen so that rho = 1, p = T
            cs2 = diff(p_of_rho, mpf(1)) / _h_gamma(T, num, den)
            assert abs(mpf(ref.cs2_of_T(float(T))) / cs2 - 1) <= 8 * EPS
        # limits: Newtonian Gamma T, and Gamma - 1 for T -> infinity (1/3 only for Gamma = 4/3: the paper's
        # point that the polytropic EoS is unphysical for a relativistic Gamma = 5/3 gas)
        assert abs(ref.cs2_of_T(1e-12) / 1e-12 - num / den) < 1e-10
        assert abs(ref.cs2_of_T(1e12) - (num / den - 1)) < 1e-10


def _states(n, seed=5):
    rng = np.random.default_rng(seed)
    W = np.empty((5, n))
    W[0] = 10.0 ** rng.uniform(-6, 6, n)
    T = 10.0 ** rng.uniform(-10, 6, n)
    g = 10.0 ** rng.uniform(0, 4, n)
    u = rng.normal(size=(3, n))
    W[1:4] = u / np.sqrt((u ** 2).sum(0)) * np.sqrt((g - 1) * (g + 1))
    W[4] = W[0] * T
    return W


@pytest.mark.parametrize("name", sorted(GAMMAS))
def test_gamma_law_prim2cons_vs_definition_and_round_trip(ref, name):
    num, den = GAMMAS[name]
    W = _states(300)
    with ref.variant(name):
        U = ref.prim2cons(W)
        for i in range(0, W.shape[1], 3):          # Etilde = D h gamma - p - D (Eq. 5c, 6) in 40 digits
            rho, ux, uy, uz, p = [mpf(float(v)) for v in W[:, i]]
            h = _h_gamma(p / rho, num, den)
            g = sqrt(1 + ux * ux + uy * uy + uz * uz)
            D = rho * g
            want = [D, D * h * ux, D * h * uy, D * h * uz, D * h * g - p - D]
            for q in range(5):
                assert abs(mpf(float(U[q, i])) - want[q]) <= 8 * EPS * abs(want[q]), (name, i, q)
        # Eq. 15 holds for ANY EoS with p = rho T: its left-hand side from the 40-digit conserved variables equals f(htilde)
        for i in range(0, W.shape[1], 7):
            rho, ux, uy, uz, p = [mpf(float(v)) for v in W[:, i]]
            T = p / rho
            h = _h_gamma(T, num, den)
            g2 = 1 + ux * ux + uy * uy + uz * uz
            x = h * sqrt(g2) - T / sqrt(g2) - 1                         # Etilde / D
            musq = h * h * (g2 - 1)
            lhs = x * x + 2 * x - musq
            f = ref.f_eq15(float(h - 1), float(musq))
            assert abs(mpf(f) / lhs - 1) <= 64 * EPS * (1 + float(musq / lhs)), (name, i)
        W2, ht2, it, bad = ref.cons2prim(U, diag=True)
        cs2 = np.array([ref.cs2_of_T(float(t)) for t in W[4] / W[0]])
        mach2 = (W[1:4] ** 2).sum(0) / (cs2 / (1 - cs2))
        cond = (1 + mach2) * EPS                                        # Eq. 20
        ok = (cond < 1e-3) & (bad == 0)
        assert ok.sum() > 100
        ht0 = np.array([ref.htilde_of_T(float(t)) for t in W[4] / W[0]])
        assert (np.abs(1 - ht0 / ht2)[ok] <= 16 * cond[ok]).all()
        assert (np.abs(W2[0] / W[0] - 1)[ok] <= 64 * cond[ok]).all()
        assert it.max() <= 9
        # reading S20: the guess is an upper bound of the root (Newton-Raphson then descends monotonically)
        x = U[4] / U[0]
        musq = ((U[1:4] / U[0]) ** 2).sum(0)
        L = x * x + 2 * x - musq
        for i in np.flatnonzero(ok)[::5]:
            assert ref.htilde_guess(float(L[i]), float(musq[i])) >= ht2[i] * (1 - 64 * cond[i] - 1e-12)   # L in plain fp64 here


def test_gamma_law_agrees_with_taub_mathews_in_its_limit(ref):
    """Eq. 10 -> 1 + 2.5 T for T -> 0 (Gamma = 5/3) and -> 4 T for T -> infinity (Gamma = 4/3) (Fig. 1)."""
    W = _states(200, seed=9)
    for name, T, tol in (("gamma53", 1e-7, 1e-6), ("gamma43", 1e7, 1e-6)):
        Wv = W.copy()
        Wv[4] = Wv[0] * T
        cs2 = ref.cs2_of_T(T)                          # subsonic: a supersonic state amplifies the O(T) (O(1/T))
        Wv[1:4] *= 0.5 * np.sqrt(cs2 / (1 - cs2)) / np.sqrt((Wv[1:4] ** 2).sum(0))   # difference of the EoS by M^2 (Eq. 20)
        Utm = ref.prim2cons(Wv)
        with ref.variant(name):
            Ug = ref.prim2cons(Wv)
            Wback, _ = ref.cons2prim(Utm)            # TM conserved variables read with the polytropic EoS
        assert (np.abs(Ug / Utm - 1) <= tol).all(), name
        assert (np.abs(Wback[4] / Wv[4] - 1) <= 10 * tol).all(), name


@pytest.mark.parametrize("name,T0", [("gamma53", 1e-10), ("gamma43", 1e10), ("gamma53", 1.0)])
def test_gamma_law_sound_wave_converges_at_second_order(ref, name, T0):
    """Section 4.1's diagonal wave with the polytropic EoS: the analytic phase speed is
    c_s = sqrt(Gamma T / h), so second-order convergence pins the EoS through the whole step."""
    from tests.test_oracle_pins_r2 import _run_wave
    with ref.variant(name):
        e16, e32 = (_run_wave(ref, N, T0) for N in (16, 32))
    assert e16 < 0.5e-6 and np.log2(e16 / e32) > 1.8, (e16, e32)


@pytest.mark.parametrize("name", sorted(GAMMAS))
def test_gamma_law_step_structure(ref, name):
    """Uniform state = bit-exact fixed point; periodic box conserves D, M, Etilde; tiled = whole box."""
    rng = np.random.default_rng(2)
    with ref.variant(name):
        par = ref.params("plm", "hllc")
        W = np.array([0.7, 3.0, -1.0, 0.5, 1e-3])
        cons = ref.prim2cons(np.repeat(W[:, None], 16 ** 3, 1)).reshape(5, 16, 16, 16)
        out, st, _ = ref.grid_step_whole(cons, 1e-3, 1e-2, par, ["periodic"] * 6)
        assert np.array_equal(out, cons)
        prim = np.empty((5, 16, 16, 32))
        x = (np.arange(32) + 0.5) / 32
        prim[0] = 1 + 0.3 * np.sin(2 * np.pi * x)[None, None, :]
        prim[1] = 0.5 * np.cos(2 * np.pi * x)[None, None, :]
        prim[2] = 0.2
        prim[3] = -0.1 + 0.05 * rng.standard_normal((16, 16, 1))
        prim[4] = 0.1 * prim[0] ** (5 / 3)
        cons = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
        dt = ref.cfl_dt(cons, 0.4, 1 / 32, par)
        whole, st, _ = ref.grid_step_whole(cons, dt, 1 / 32, par, ["periodic"] * 6)
        tiled, st2 = ref.grid_step_tiled(cons, dt, 1 / 32, par, ["periodic"] * 6)
        assert st.n_retry_pg == 0 and np.array_equal(whole, tiled)
        for q in range(5):
            assert abs(whole[q].sum() - cons[q].sum()) <= 64 * EPS * np.abs(cons[q]).sum()


def test_gamma_law_shock_obeys_the_taub_adiabat(ref):
    """A strong shock tube run with the polytropic EoS: the post-shock plateau of the NUMERICAL solution and the
    undisturbed gas ahead of it must satisfy the Taub adiabat (P:659 Eq. C10, valid for any EoS) with
    h = 1 + Gamma/(Gamma-1) T -- the conversions, the sound speed in the solver and the update all enter."""
    with ref.variant("gamma53"):
        par = ref.params("plm", "hllc")
        prim, dh, bc = workloads.shock_tube(n_long=256, n_trans=16, left=(1.0, 0.0, 10.0), right=(1.0, 0.0, 1e-2))
        cons = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
        t = 0.0
        while t < 0.35:
            dt = ref.cfl_dt(cons, 0.5, dh, par)
            cons, _ = ref.grid_step_tiled(cons, dt, dh, par, bc)
            t += dt
        W = ref.cons2prim(cons.reshape(5, -1))[0].reshape(cons.shape)
    ax = int(np.argmax(cons.shape[1:]))                     # the long axis
    line = np.moveaxis(W, 1 + ax, 1)[:, :, 0, 0]
    rho, p = line[0], line[4]
    i_sh = int(np.argmax(np.abs(np.diff(np.log(p)))[128:])) + 128        # the shock: steepest pressure jump on the right
    down, up = slice(i_sh - 12, i_sh - 5), slice(i_sh + 6, i_sh + 11)
    # the dense shell between contact and shock is a handful of cells wide: its density is the peak value there,
    # the pressure is flat across the contact
    rd, pd, ru, pu = rho[i_sh - 10:i_sh + 1].max(), p[down].mean(), rho[up].mean(), p[up].mean()
    assert p[down].std() < 0.01 * pd and pd > 10 * pu and rd > 4 * ru    # a plateau behind a strong shock
    hd, hu = 1 + 2.5 * pd / rd, 1 + 2.5 * pu / ru
    lhs = hu * hu - hd * hd
    rhs = (hd / rd + hu / ru) * (pu - pd)
    assert abs(lhs / rhs - 1) < 0.02, (lhs, rhs)


# ------------------------------------------------------------------ the "original scheme"
def _eq20_eq21(T, U2, ht):
    """The paper's round-off estimates of the new (Eq. 20) and the original (Eq. 21) conversion, in units of eps."""
    g2 = 1 + U2
    h = ht + 1
    beta2 = U2 / g2
    den20 = h * h + T * T / g2 - 2 * h * T - 1
    e20 = (g2 * h * h * (1 + beta2) + T * T / g2 - 2 * h * T - 1) / den20
    e21 = (2 * g2 * h * h + T * T / g2 - 2 * h * T + h * h + 1) / ((ht + 2) * ht + T * T / g2 - 2 * h * T)
    return e20, e21


def test_original_scheme_prim2cons_is_eq5c(ref):
    W = _states(120, seed=3)
    with ref.variant("orig"):
        U = ref.prim2cons(W)
    Un = ref.prim2cons(W)
    assert np.array_equal(U[:4], Un[:4])
    for i in range(W.shape[1]):
        rho, ux, uy, uz, p = [mpf(float(v)) for v in W[:, i]]
        T = p / rho
        h = mpf(5) / 2 * T + sqrt(mpf(9) / 4 * T * T + 1)
        g = sqrt(1 + ux * ux + uy * uy + uz * uz)
        E = rho * g * h * g - p
        assert abs(mpf(float(U[4, i])) - E) <= 4 * EPS * E


def test_fig16_round_trip_errors_follow_eq20_and_eq21(ref):
    """P:626 App. B / Fig. 16: T = 1e-8, U parallel to (1,1,1), Mach 1e-4 .. 1e6; |1 - htilde_0/htilde_2| of the
    original scheme follows Eq. 21 (~ 4/(3T) eps for M << 1, Eq. 32), that of the new scheme Eq. 20."""
    T = 1e-8
    W, mach = workloads.mach_sweep_states(theta=T, n=61)
    cs2 = ref.cs2_of_T(T)
    W[1:4] *= (mach * np.sqrt(cs2 / (1 - cs2)))[None, :]
    ht0 = ref.htilde_of_T(T)
    U2 = (W[1:4] ** 2).sum(0)
    e20, e21 = _eq20_eq21(T, U2, ht0)
    _, ht_new, _, _ = ref.cons2prim(ref.prim2cons(W), diag=True)
    with ref.variant("orig"):
        _, ht_orig, _, bad = ref.cons2prim(ref.prim2cons(W), diag=True)
    err_new, err_orig = np.abs(1 - ht0 / ht_new), np.abs(1 - ht0 / ht_orig)
    sel = mach < 1e5
    assert (err_new[sel] <= 16 * e20[sel] * EPS).all()
    # the original scheme: never better than a small fraction of its estimate on average, never worse than it
    assert (err_orig[sel] <= 4 * e21[sel] * EPS).all()
    low = mach < 1e-1
    assert abs(e21[low].mean() / (4 / (3 * T)) - 1) < 0.05             # Eq. 32 is the low-Mach value of Eq. 21
    assert np.median(err_orig[low]) > 0.02 * (4 / (3 * T)) * EPS        # ~1e-8 ... 1e-9, against ~1e-16 below
    assert err_new[low].max() < 8 * EPS
    assert np.median(err_orig[low] / np.maximum(err_new[low], EPS)) > 1e6


@pytest.mark.parametrize("T0", [1e-10, 1e10])
def test_fig3_original_scheme_stalls_in_the_cold_limit(ref, T0):
    """P:301-311 / Fig. 3: for the diagonal sound wave the new scheme converges as N^-2 at T = 1e-10 and 1e10; the
    original scheme converges at T = 1e10 too, but at T = 1e-10 its L1 error is 'much larger and roughly equal to a
    constant of 2e-6' (the cancellation error of Eq. 32, 4/(3T) eps ~ 1e-6)."""
    from tests.test_oracle_pins_r2 import _run_wave
    new = [_run_wave(ref, N, T0) for N in (16, 32)]
    with ref.variant("orig"):
        orig = [_run_wave(ref, N, T0) for N in (16, 32)]
    assert np.log2(new[0] / new[1]) > 1.8
    if T0 > 1:
        assert np.log2(orig[0] / orig[1]) > 1.8 and abs(orig[1] / new[1] - 1) < 0.05
    else:
        for e in orig:
            assert 1e-7 < e < 2e-5, orig                                # the plateau of Fig. 3, no convergence
        assert orig[1] > 0.3 * orig[0] and orig[1] > 100 * new[1]


def test_original_and_new_scheme_are_the_same_method_in_exact_arithmetic(ref):
    """E = Etilde + D and F_E = F_Etilde + F_D (Eq. 4a, 4c, 7): on well-conditioned (hot, moderately relativistic)
    data the two schemes must give the same fluxes and the same updated state up to round-off."""
    rng = np.random.default_rng(8)
    for riemann in ("hlle", "hllc"):
        for _ in range(40):
            WL = np.array([10 ** rng.uniform(-1, 1), *rng.normal(0, 1.5, 3), 10 ** rng.uniform(-1, 1)])
            WR = np.array([10 ** rng.uniform(-1, 1), *rng.normal(0, 1.5, 3), 10 ** rng.uniform(-1, 1)])
            d = int(rng.integers(3))
            UL, UR = ref.prim2cons(WL[:, None])[:, 0], ref.prim2cons(WR[:, None])[:, 0]
            Fn = ref.riemann_flux(riemann, d, WL, UL, WR, UR)
            with ref.variant("orig"):
                ULo, URo = ref.prim2cons(WL[:, None])[:, 0], ref.prim2cons(WR[:, None])[:, 0]
                Fo = ref.riemann_flux(riemann, d, WL, ULo, WR, URo)
            scale = np.abs(Fn).max() + np.abs(Fo).max()
            assert np.abs(Fo[:4] - Fn[:4]).max() <= 256 * EPS * scale
            assert abs(Fo[4] - (Fn[4] + Fn[0])) <= 256 * EPS * scale
    # one step of a smooth periodic box
    par = ref.params("plm", "hllc")
    x = (np.arange(32) + 0.5) / 32
    prim = np.empty((5, 16, 16, 32))
    prim[0] = 1 + 0.3 * np.sin(2 * np.pi * x)[None, None, :]
    prim[1] = 0.8 * np.cos(2 * np.pi * x)[None, None, :]
    prim[2], prim[3] = 0.3, -0.2
    prim[4] = 2.0 * prim[0] ** (4 / 3)
    cons = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    dt = ref.cfl_dt(cons, 0.4, 1 / 32, par)
    new, _ = ref.grid_step_tiled(cons, dt, 1 / 32, par, ["periodic"] * 6)
    with ref.variant("orig"):
        conso = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
        orig, st = ref.grid_step_tiled(conso, dt, 1 / 32, par, ["periodic"] * 6)
        assert st.n_retry_pg == 0
        W = np.array([0.7, 3.0, -1.0, 0.5, 1e-3])                      # and a uniform state stays a fixed point
        cu = ref.prim2cons(np.repeat(W[:, None], 16 ** 3, 1)).reshape(5, 16, 16, 16)
        out, _, _ = ref.grid_step_whole(cu, 1e-3, 1e-2, par, ["periodic"] * 6)
        assert np.array_equal(out, cu)
    assert np.abs(orig[:4] - new[:4]).max() <= 1e-13 * np.abs(new[:4]).max()
    assert np.abs(orig[4] - (new[4] + new[0])).max() <= 1e-13 * np.abs(orig[4]).max()


# ------------------------------------------------------------------ single precision (eps_machine = 1e-7)
EPS32 = float(np.finfo(np.float32).eps)


def test_f32_conversions_follow_eq20_with_single_precision_epsilon(ref):
    """The single-precision variant against the double-precision oracle: both are the same algorithm, so they may
    differ by the paper's error model with eps_machine = FLT_EPSILON (Eq. 20), and no more."""
    W = workloads.conversion_states(n=4000, log_rho=(-3, 3), log_theta=(-6, 3), log_gamma=(0, 1.5))
    U64 = ref.prim2cons(W)
    _, ht64, _, bad64 = ref.cons2prim(U64, diag=True)
    cs2 = ref.cs2_of_T(W[4] / W[0])
    cond = (1 + (W[1:4] ** 2).sum(0) * (1 - cs2) / cs2) * EPS32
    with ref.variant("f32"):
        par = ref.params(newton_rtol=1e-6)
        U32 = ref.prim2cons(W)
        assert U32.dtype == np.float32
        W32, ht32, it, bad32 = ref.cons2prim(U32, par, diag=True)
    assert (np.abs(U32 / U64 - 1)[:, np.isfinite(U64).all(0)] <= 8 * EPS32).all()       # prim -> cons has no cancellation
    ok = (cond < 1e-2) & (bad32 == 0)
    assert ok.sum() > 1500
    assert (np.abs(1 - ht32[ok] / ht64[ok]) <= 16 * cond[ok]).all()
    assert (np.abs(W32[0] / W[0] - 1)[ok] <= 64 * cond[ok]).all()
    assert it.max() <= 8
    # Eq. 30 with the single-precision eps_machine: L between the two epsilons passes in double only
    L = 3e-9
    x = L / 2                                          # at rest: L = x^2 + 2x
    U = np.array([[1.0], [0.0], [0.0], [0.0], [x]])
    assert ref.cons2prim(U, diag=True)[3][0] == 0
    with ref.variant("f32"):
        assert ref.cons2prim(U, diag=True)[3][0] == 1


def test_f32_step_tracks_the_double_precision_step(ref):
    rng = np.random.default_rng(4)
    x = (np.arange(32) + 0.5) / 32
    prim = np.empty((5, 16, 16, 32))
    prim[0] = 1 + 0.3 * np.sin(2 * np.pi * x)[None, None, :]
    prim[1] = 0.8 * np.cos(2 * np.pi * x)[None, None, :]
    prim[2], prim[3] = 0.3, -0.2 + 0.05 * rng.standard_normal((16, 16, 1))
    prim[4] = 0.5 * prim[0] ** (4 / 3)
    par64 = ref.params("plm", "hllc")
    c64 = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    dt = ref.cfl_dt(c64, 0.4, 1 / 32, par64)
    n64, _ = ref.grid_step_tiled(c64, dt, 1 / 32, par64, ["periodic"] * 6)
    with ref.variant("f32"):
        par = ref.params("plm", "hllc", newton_rtol=1e-6)
        c32 = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
        whole, st, _ = ref.grid_step_whole(c32, dt, 1 / 32, par, ["periodic"] * 6)
        tiled, _ = ref.grid_step_tiled(c32, dt, 1 / 32, par, ["periodic"] * 6)
        assert tiled.dtype == np.float32 and np.array_equal(whole, tiled) and st.n_retry_pg == 0
        for q in range(5):                              # conservation to single-precision round-off
            assert abs(float(tiled[q].astype(np.float64).sum() - c32[q].astype(np.float64).sum())) <= \
                64 * EPS32 * float(np.abs(c32[q]).sum()) / np.sqrt(c32[q].size)
        Wu = np.array([0.7, 3.0, -1.0, 0.5, 1e-3])
        cu = ref.prim2cons(np.repeat(Wu[:, None], 16 ** 3, 1)).reshape(5, 16, 16, 16)
        assert np.array_equal(ref.grid_step_whole(cu, 1e-3, 1e-2, par, ["periodic"] * 6)[0], cu)
    scale = np.abs(n64).reshape(5, -1).max(1)[:, None, None, None]
    assert (np.abs(tiled - n64) / scale).max() <= 64 * EPS32
