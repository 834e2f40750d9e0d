"""Exact solution of the 1-D relativistic Riemann problem with the Taub-Mathews EoS.

TEST INFRASTRUCTURE ONLY (oracle side).  Follows PAPER.md App. C step by step, in
four-velocities, with mpmath arithmetic (default 30 digits) so that the 16-digit rows of Table 2
 can be reproduced to round-off.  No tangential velocities (the paper's problems are
purely 1-D).  Units c = k_B = m = 1.

  * Eq. 10  h(T) = 2.5 T + sqrt(2.25 T^2 + 1)
  * Eq. 14  c_s(T)
  * Eq. C9a dU/drho = -/+ c_s gamma / rho  (upper sign right wave)
            <=> d asinh(U) = -/+ c_s dln(rho)
  * Eq. C9b p rho^(-5/3) (h - T) = const  <=> T (h - T) = K rho^(2/3)
  * Eq. C10 Taub adiabat, C11 mass flux J, C12/C13 boosts              (reading G3)
  * Eq. C8  p* from matching the contact four-velocity from both sides
"""
from mpmath import mp, mpf, sqrt, asinh, sinh, quad, findroot, log, exp

mp.dps = 30


def h_of_T(T):
    return mpf(5) / 2 * T + sqrt(mpf(9) / 4 * T * T + 1)


def dh_dT(T):
    return mpf(5) / 2 + mpf(9) / 4 * T / sqrt(mpf(9) / 4 * T * T + 1)


def cs_of_T(T):
    h = h_of_T(T)
    return sqrt(T / (3 * h) * (5 * h - 8 * T) / (h - T))


def _bisect_log(fun, lo, hi, tol=None):
    """Root of a monotone function on [lo, hi] (positive reals), bisection in log then secant."""
    tol = tol or mpf(10) ** (-(mp.dps - 3))
    flo, fhi = fun(lo), fun(hi)
    if flo == 0:
        return lo
    if fhi == 0:
        return hi
    assert (flo < 0) != (fhi < 0), "root not bracketed"
    a, b = log(lo), log(hi)
    for _ in range(60):
        m = (a + b) / 2
        fm = fun(exp(m))
        if (fm < 0) == (flo < 0):
            a = m
        else:
            b = m
        if b - a < 1.0:
            break
    return findroot(fun, (exp(a), exp(b)), solver="illinois", tol=tol * tol, maxsteps=200,
                    verify=False)


class Wave:
    """One nonlinear wave: side = -1 (left wave, lower signs) or +1 (right wave, upper signs)."""

    def __init__(self, side, rho, U, p):
        self.side = side
        self.rho0, self.U0, self.p0 = mpf(rho), mpf(U), mpf(p)
        self.T0 = self.p0 / self.rho0
        self.h0 = h_of_T(self.T0)
        # isentrope constant of Eq. C9b written as T (h - T) = K rho^(2/3)
        self.K = self.T0 * (self.h0 - self.T0) / self.rho0 ** (mpf(2) / 3)

    # --- rarefaction branch (p* <= p0) ---
    def _rho_on_isentrope(self, T):
        return (T * (h_of_T(T) - T) / self.K) ** (mpf(3) / 2)

    def _T_on_isentrope_at_p(self, p):
        # T (h - T) = K (p/T)^(2/3); isentropic exponent (Gamma-1)/Gamma lies in [1/4, 2/5]
        r = p / self.p0
        lo, hi = self.T0 * r ** mpf("0.41"), self.T0 * r ** mpf("0.24")
        fun = lambda T: T * (h_of_T(T) - T) * T ** (mpf(2) / 3) - self.K * p ** (mpf(2) / 3)
        return _bisect_log(fun, lo, hi)

    def _invariant_integral(self, T):
        """int_{rho(T)}^{rho0} c_s dln(rho) along the isentrope (T <= T0), variable s = ln T."""
        if T == self.T0:
            return mpf(0)

        def integrand(s):
            t = exp(s)
            h = h_of_T(t)
            return cs_of_T(t) * mpf(3) / 2 * (1 + t * (dh_dT(t) - 1) / (h - t))

        return quad(integrand, [log(T), log(self.T0)])

    def _U_in_fan(self, T):
        # Eq. C9a integrated: asinh U = asinh U0 -/+ int_{rho0}^{rho} c_s dln rho  (upper: right wave)
        # left wave (lower sign): asinh U = asinh U0 + int_{rho}^{rho0} c_s dln rho
        return sinh(asinh(self.U0) - self.side * self._invariant_integral(T))

    # --- shock branch (p* > p0): upstream = the unperturbed state ---
    def _shock(self, p):
        rho_u, p_u, U_u, h_u = self.rho0, self.p0, self.U0, self.h0

        def taub(T):  # Eq. C10 with rho_down = p/T
            h_d = h_of_T(T)
            return h_d * h_d - h_u * h_u + (h_d * T / p + h_u / rho_u) * (p_u - p)

        T_d = _bisect_log(taub, self.T0, max(self.T0, p / rho_u, mpf(1)) * mpf(10) ** 12)
        rho_d = p / T_d
        h_d = h_of_T(T_d)
        J = sqrt((p - p_u) / (h_u / rho_u - h_d / rho_d))                       # Eq. C11
        s = self.side
        U_sh = s * (J / rho_u) * sqrt(1 + U_u ** 2) + U_u * sqrt(1 + (J / rho_u) ** 2)      # C12 (G3)
        U_post = -s * (J / rho_d) * sqrt(1 + U_sh ** 2) + U_sh * sqrt(1 + (J / rho_d) ** 2)  # C13
        return rho_d, U_post, U_sh, J

    def star(self, p):
        """(rho*, U*) behind the wave for contact pressure p."""
        p = mpf(p)
        if p > self.p0:
            rho_d, U_post, _, _ = self._shock(p)
            return rho_d, U_post
        T = self._T_on_isentrope_at_p(p)
        return p / T, self._U_in_fan(T)


class ExactRiemann:
    def __init__(self, left, right):
        """left/right = (rho, U, p) with U the four-velocity along x."""
        self.L = Wave(-1, *left)
        self.R = Wave(+1, *right)
        lo = min(self.L.p0, self.R.p0) * mpf(10) ** -12
        hi = max(self.L.p0, self.R.p0, self.L.rho0, self.R.rho0) * mpf(10) ** 14 * \
            (1 + self.L.U0 ** 2 + self.R.U0 ** 2)
        fun = lambda p: self.L.star(p)[1] - self.R.star(p)[1]                   # Eq. C8
        self.p_star = _bisect_log(fun, lo, hi)
        self.rho_CL, self.U_star = self.L.star(self.p_star)
        self.rho_CR, U2 = self.R.star(self.p_star)
        self.U_star_right = U2
        self.v_star = self.U_star / sqrt(1 + self.U_star ** 2)
        self._setup_wave(self.L, self.rho_CL)
        self._setup_wave(self.R, self.rho_CR)

    def _setup_wave(self, w, rho_star):
        s = w.side
        if self.p_star > w.p0:
            _, _, U_sh, J = w._shock(self.p_star)
            w.kind = "shock"
            w.xi_head = w.xi_tail = U_sh / sqrt(1 + U_sh ** 2)
            w.J = J
        else:
            w.kind = "rarefaction"
            w.T_star = self.p_star / rho_star
            v0 = w.U0 / sqrt(1 + w.U0 ** 2)
            c0, c1 = cs_of_T(w.T0), cs_of_T(w.T_star)
            w.xi_head = (v0 + s * c0) / (1 + s * v0 * c0)
            w.xi_tail = (self.v_star + s * c1) / (1 + s * self.v_star * c1)

    def _fan(self, w, xi):
        s = w.side

        def fun(T):
            U = w._U_in_fan(T)
            v = U / sqrt(1 + U * U)
            c = cs_of_T(T)
            return (v + s * c) / (1 + s * v * c) - xi

        T = _bisect_log(fun, w.T_star, w.T0)
        rho = w._rho_on_isentrope(T)
        return rho, w._U_in_fan(T), rho * T

    def sample(self, xi):
        """(rho, U, p) at xi = (x - x0)/t."""
        xi = mpf(xi)
        L, R = self.L, self.R
        if xi <= self.v_star:
            if xi <= L.xi_head:
                return L.rho0, L.U0, L.p0
            if xi >= L.xi_tail:
                return self.rho_CL, self.U_star, self.p_star
            return self._fan(L, xi)
        if xi >= R.xi_head:
            return R.rho0, R.U0, R.p0
        if xi <= R.xi_tail:
            return self.rho_CR, self.U_star, self.p_star
        return self._fan(R, xi)

    # ---- fast float64 profile for comparing against a numerical solution (error ~1e-9) ----
    def profile(self, xis, n_table=4001):
        """(rho, U, p) arrays at xi values; rarefaction fans are tabulated in float64.

        The fan table integrates Eq. C9a with 8-point Gauss-Legendre per log-T segment and is
        inverted by monotone interpolation in xi, so it is accurate to ~1e-9, far below the
        O(dx) truncation error of any finite-volume solution it is compared with.
        """
        import numpy as np
        xis = np.asarray(xis, dtype=np.float64)
        rho = np.empty_like(xis)
        U = np.empty_like(xis)
        p = np.empty_like(xis)
        L, R = self.L, self.R
        vs = float(self.v_star)
        regions = [
            (xis <= float(L.xi_head), (float(L.rho0), float(L.U0), float(L.p0))),
            ((xis >= float(L.xi_tail)) & (xis <= vs), (float(self.rho_CL), float(self.U_star), float(self.p_star))),
            ((xis > vs) & (xis <= float(R.xi_tail)), (float(self.rho_CR), float(self.U_star), float(self.p_star))),
            (xis >= float(R.xi_head), (float(R.rho0), float(R.U0), float(R.p0))),
        ]
        done = np.zeros(xis.shape, dtype=bool)
        for m, (a, b, c) in regions:
            m = m & ~done
            rho[m], U[m], p[m] = a, b, c
            done |= m
        for w in (L, R):
            if w.kind != "rarefaction":
                continue
            s = w.side
            m = ~done & ((xis < vs) if s < 0 else (xis > vs))
            if not m.any():
                continue
            lnT = np.linspace(float(log(w.T_star)), float(log(w.T0)), n_table)

            def hT(t): return 2.5 * t + np.sqrt(2.25 * t * t + 1.0)
            def cs(t):
                h = hT(t)
                return np.sqrt(t / (3 * h) * (5 * h - 8 * t) / (h - t))
            def integrand(sv):
                t = np.exp(sv)
                h = hT(t)
                dh = 2.5 + 2.25 * t / np.sqrt(2.25 * t * t + 1.0)
                return cs(t) * 1.5 * (1 + t * (dh - 1) / (h - t))
            gx, gw = np.polynomial.legendre.leggauss(8)
            a, b = lnT[:-1], lnT[1:]
            mid, half = 0.5 * (a + b), 0.5 * (b - a)
            seg = (integrand(mid[:, None] + half[:, None] * gx[None, :]) * gw[None, :]).sum(1) * half
            # I(T) = int_T^{T0}: cumulative from the top
            I = np.concatenate([np.cumsum(seg[::-1])[::-1], [0.0]])
            T = np.exp(lnT)
            Uf = np.sinh(np.arcsinh(float(w.U0)) - s * I)
            v = Uf / np.sqrt(1 + Uf * Uf)
            c = cs(T)
            xi_tab = (v + s * c) / (1 + s * v * c)
            K = float(w.K)
            rho_tab = (T * (hT(T) - T) / K) ** 1.5
            order = np.argsort(xi_tab)
            lt = np.interp(xis[m], xi_tab[order], lnT[order])
            rho[m] = np.interp(lt, lnT, rho_tab)
            U[m] = np.interp(lt, lnT, Uf)
            p[m] = rho[m] * np.exp(lt)
            done |= m
        return rho, U, p
