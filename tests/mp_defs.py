"""Plain DEFINITIONS from the paper evaluated with mpmath (40 digits) -- used to pin the oracle.

These are the textbook forms the paper says NOT to use in fp64 (they cancel catastrophically);
in 40-digit arithmetic they are exact for our purposes, so they pin the cancellation-free forms
of the oracle against something other than itself.  Units c = 1.
  h(T) = 2.5 T + sqrt(2.25 T^2 + 1)            PAPER.md line 104, Eq. 10
  D = rho gamma, M = D h U, E = D h gamma - p   lines 71-75, Eq. 5a-5c
  Etilde = E - D                                line 79, Eq. 6
  gamma = sqrt(1 + U.U)                         line 90, Eq. 8
  fluxes: D v, M v + p e_n, (E - D) ... = M_n - D v   lines 61-65 Eq. 4a-4c, line 81
"""
from mpmath import mp, mpf, sqrt

mp.dps = 40


def _mp(w):
    """fp64 inputs enter exactly; values that are already 40-digit numbers stay as they are."""
    return w if isinstance(w, mpf) else mpf(float(w))


def h_of_T(T):
    T = mpf(T)
    return mpf(5) / 2 * T + sqrt(mpf(9) / 4 * T * T + 1)


def cs2_of_T(T):
    T = mpf(T)
    h = h_of_T(T)
    return T / (3 * h) * (5 * h - 8 * T) / (h - T)


def prim2cons(W):
    rho, ux, uy, uz, p = [_mp(w) for w in W]
    T = p / rho
    h = h_of_T(T)
    g = sqrt(1 + ux * ux + uy * uy + uz * uz)
    D = rho * g
    E = D * h * g - p
    return [D, D * h * ux, D * h * uy, D * h * uz, E - D]


def phys_flux(d, W):
    """Eq. 4a, 4b, and the reduced-energy flux in its DEFINING form (M_n - D v_n), line 81."""
    rho, ux, uy, uz, p = [_mp(w) for w in W]
    U = prim2cons(W)
    g = sqrt(1 + ux * ux + uy * uy + uz * uz)
    v = [ux, uy, uz][d] / g
    F = [U[0] * v, U[1] * v, U[2] * v, U[3] * v, U[1 + d] - U[0] * v]
    F[1 + d] += p
    return F


def f_eq15(ht, musq):
    """Right-hand side of Eq. 15 (lines 140-144) with T from the definition h = Eq. 10 inverted
    numerically (not via Eq. 16), so that Eq. 16 itself is pinned."""
    from mpmath import findroot
    ht = mpf(ht)
    T = findroot(lambda t: h_of_T(t) - 1 - ht, ht / 3 + mpf(10) ** -40) if ht > 0 else mpf(0)
    h = ht + 1
    return ht * ht + 2 * ht - 2 * T * h + T * T * h * h / (h * h + mpf(musq)), T


def lambda_pm_3vel(W, d):
    """Textbook acoustic eigenvalues in 3-velocity form (Mignone & Bodo 2005 Eq. 23 form)."""
    rho, ux, uy, uz, p = [_mp(w) for w in W]
    g = sqrt(1 + ux * ux + uy * uy + uz * uz)
    v = [ux / g, uy / g, uz / g]
    v2 = sum(x * x for x in v)
    cs2 = cs2_of_T(p / rho)
    vn = v[d]
    disc = sqrt(cs2 * (1 - v2) * (1 - v2 * cs2 - vn * vn * (1 - cs2)))
    return (vn * (1 - cs2) - disc) / (1 - v2 * cs2), (vn * (1 - cs2) + disc) / (1 - v2 * cs2)


# ---------------------------------------------------------------------------------------------
# Riemann solvers written out from their plain definitions (Mignone & Bodo 2005/2006 as the paper
# adapts them: TM sound speed, E = Etilde + D) in 40-digit arithmetic, with the
# TEXTBOOK 3-velocity eigenvalues above.  Plain subtractions everywhere: at 40 digits they are exact
# for our purposes, which is what makes these a pin for any fp64 evaluation order.
def _rot(d):
    return [0, 1 + d, 1 + (d + 1) % 3, 1 + (d + 2) % 3, 4]


def _side(W, d):
    rho, ux, uy, uz, p = [_mp(w) for w in W]
    U = prim2cons(W)
    F = phys_flux(d, W)
    g = sqrt(1 + ux * ux + uy * uy + uz * uz)
    lm, lp = lambda_pm_3vel(W, d)
    return dict(U=U, F=F, p=p, vn=[ux, uy, uz][d] / g, lm=lm, lp=lp)


def hll_speeds(WL, WR, d):
    L, R = _side(WL, d), _side(WR, d)
    return min(L["lm"], R["lm"]), max(L["lp"], R["lp"])


def _pt(K, d):
    """pressure terms of the physical flux: F = U v_n + pt."""
    out = [mpf(0)] * 5
    out[1 + d] = K["p"]
    out[4] = K["p"] * K["vn"]
    return out


def _upwind_pieces(K, d):
    return [abs(K["U"][c] * K["vn"]) + abs(_pt(K, d)[c]) for c in range(5)]


def hlle_flux(WL, WR, d, pieces=False):
    """F = (S_R F_L - S_L F_R + S_L S_R (U_R - U_L)) / (S_R - S_L), upwinded outside [S_L, S_R].
    pieces=True also returns, per component, the summed magnitude of the terms that do not cancel by
    arithmetic alone: S_R (v_L - S_L) U_L, S_L (S_R - v_R) U_R and the two pressure terms (a tolerance scale)."""
    L, R = _side(WL, d), _side(WR, d)
    SL, SR = min(L["lm"], R["lm"]), max(L["lp"], R["lp"])
    if SL >= 0:
        return (L["F"], _upwind_pieces(L, d)) if pieces else L["F"]
    if SR <= 0:
        return (R["F"], _upwind_pieces(R, d)) if pieces else R["F"]
    F = [(SR * L["F"][c] - SL * R["F"][c] + SL * SR * (R["U"][c] - L["U"][c])) / (SR - SL) for c in range(5)]
    if not pieces:
        return F
    ptL, ptR = _pt(L, d), _pt(R, d)
    pc = [(abs(SR * (L["vn"] - SL) * L["U"][c]) + abs(SL * (SR - R["vn"]) * R["U"][c]) + abs(SR * ptL[c]) + abs(SL * ptR[c]))
          / (SR - SL) for c in range(5)]
    return F, pc


def hllc_flux(WL, WR, d, pieces=False):
    """HLLC with the contact speed from the HLL averages of (D, M_n, E = Etilde + D) and the star state
    of the side the contact leaves behind (reading S7), all in plain 40-digit arithmetic on the TOTAL
    energy E (the textbook form); the reduced-energy flux is F_E - F_D at the end."""
    L, R = _side(WL, d), _side(WR, d)
    SL, SR = min(L["lm"], R["lm"]), max(L["lp"], R["lp"])
    if SL >= 0:
        return (L["F"], _upwind_pieces(L, d)) if pieces else L["F"]
    if SR <= 0:
        return (R["F"], _upwind_pieces(R, d)) if pieces else R["F"]
    n = 1 + d
    # total energy and its flux: E = Etilde + D, F_E = F_Etilde + F_D = M_n
    EL, ER = L["U"][4] + L["U"][0], R["U"][4] + R["U"][0]
    FEL, FER = L["U"][n], R["U"][n]

    def hll(uL, uR, fL, fR):
        return (SR * uR - SL * uL + fL - fR) / (SR - SL), (SR * fL - SL * fR + SL * SR * (uR - uL)) / (SR - SL)

    Eh, FEh = hll(EL, ER, FEL, FER)
    mh, Fmh = hll(L["U"][n], R["U"][n], L["F"][n], R["F"][n])
    a, b, c = FEh, -(Eh + Fmh), mh
    lam = (-b - sqrt(b * b - 4 * a * c)) / (2 * a) if a != 0 else -c / b     # the root in (-1, 1)
    ps = Fmh - lam * FEh
    K, S, EK = (L, SL, EL) if lam >= 0 else (R, SR, ER)
    A, den = S - K["vn"], S - lam
    Us = [K["U"][c_] * A / den for c_ in range(5)]
    Us[n] = (K["U"][n] * A + ps - K["p"]) / den
    Es = (EK * A + ps * lam - K["p"] * K["vn"]) / den
    Us[4] = Es - Us[0]                                                       # Etilde* = E* - D*
    F = [K["F"][c_] + S * (Us[c_] - K["U"][c_]) for c_ in range(5)]
    if not pieces:
        return F
    ptK = _pt(K, d)
    # the star state itself is a sum of pieces, (U_K A + pressure terms)/(S - lam): take their magnitudes
    star = [abs(K["U"][c_] * A / den) for c_ in range(5)]
    # (p* = F_M^hll - lam* F_E^hll is a subtraction in the DEFINITION of the solver, reading S7: its two
    # operands count as pieces, not their difference)
    psz = abs(Fmh) + abs(lam * FEh)
    star[n] += (psz + abs(K["p"])) / abs(den)
    star[4] += (psz * abs(lam) + abs(K["p"] * K["vn"])) / abs(den)
    # conditioning of the contact speed: the two roots of a lam^2 - b lam + m = 0 approach each other (and the
    # light cone) when an ultra-relativistic stream hits slow gas; lam* then carries sqrt(kappa) ulp
    kappa = b * b / (b * b - 4 * a * c)
    pc = [abs(S) * star[c_] + abs(A * K["U"][c_]) + abs(ptK[c_]) for c_ in range(5)]
    pc[n] += psz                                       # F*_n = M_n* lam* + p*,  F*_E = (Etilde* + p*) lam*
    pc[4] += psz * abs(lam)
    return F, pc, kappa


# ---------------------------------------------------------------------------------------------
# cons -> prim from the DEFINITIONS (Eq. 5a-5c, 8, 10): find h with D h gamma - p = Etilde + D where
# gamma^2 = 1 + |M|^2/(D h)^2, rho = D/gamma, p = rho T(h), T(h) = (5h - sqrt(9h^2+16))/8 (Eq. 10
# solved for T; the subtraction is harmless at 40 digits).  No Eq. 15/16, no App. A guess.
def T_of_h(h):
    return (5 * h - sqrt(9 * h * h + 16)) / 8


def cons2prim(U):
    from mpmath import findroot
    D, mx, my, mz, Et = [_mp(u) for u in U]
    m2 = mx * mx + my * my + mz * mz

    def resid(h):
        g = sqrt(1 + m2 / (D * h) ** 2)
        return (D * h * g - (D / g) * T_of_h(h)) / (Et + D) - 1

    hi = 2 + 2 * (Et + D) / D
    h = findroot(resid, (mpf(1), hi), solver="anderson", tol=mpf(10) ** -70, maxsteps=200)
    g = sqrt(1 + m2 / (D * h) ** 2)
    rho = D / g
    return [rho, mx / (D * h), my / (D * h), mz / (D * h), rho * T_of_h(h)]


def limited_slope(sL, sR, beta):
    """reading S3: van Leer harmonic mean capped by the generalised minmod."""
    if sL * sR <= 0:
        return mpf(0)
    mag = min(2 * abs(sL * sR) / abs(sL + sR), mpf(beta) * min(abs(sL), abs(sR)))
    return mag if sL > 0 else -mag


def plm_edges(am1, a0, ap1, beta):
    d = limited_slope(a0 - am1, ap1 - a0, beta)
    return a0 - d / 2, a0 + d / 2


def ppm_edges(a, beta):
    """reading S4: Colella & Woodward (1984) on a uniform grid from a = (a_{i-2} .. a_{i+2}): limited slopes
    as S3, face = (a_i + a_{i+1})/2 - (d_{i+1} - d_i)/6, monotonisation CW84 Eq. 1.10 (first pass: no blend)."""
    dm, d0, dp = (limited_slope(a[k + 1] - a[k], a[k + 2] - a[k + 1], beta) for k in range(3))
    ai = a[2]
    am = (a[1] + a[2]) / 2 - (d0 - dm) / 6
    ap = (a[2] + a[3]) / 2 - (dp - d0) / 6
    if (ap - ai) * (ai - am) <= 0:
        return ai, ai
    dd, c6 = ap - am, 6 * (ai - (am + ap) / 2)
    if dd * c6 > dd * dd:
        am = 3 * ai - 2 * ap
    elif -(dd * dd) > dd * c6:
        ap = 3 * ai - 2 * am
    return am, ap


def step_cells(cons, cells, dt, dh, riemann="hllc", beta=1.5, recon="plm"):
    """One PLM/PPM + MUSCL-Hancock + HLLE/HLLC update (readings S3, S5, S12) of the
    listed cells (i, j, k) of a conserved box cons[5][nz][ny][nx] (numpy float64; every cell within two (PLM) or three (PPM)
    of a listed cell must be inside the box), in 40-digit arithmetic from the definitions above.
    Returns {cell: [5 mpf]}.  Python loops with memoisation: a handful of cells only."""
    dt, dh = mpf(dt), mpf(dh)
    flux_fn = hllc_flux if riemann == "hllc" else hlle_flux
    Wc, edges, fluxes = {}, {}, {}

    def prim(c):
        if c not in Wc:
            i, j, k = c
            Wc[c] = cons2prim([float(cons[q, k, j, i]) for q in range(5)])
        return Wc[c]

    def shift(c, d, s):
        c = list(c)
        c[d] += s
        return tuple(c)

    def half_step(c):
        """Evolved PRIMITIVE edge states of cell c: {(d, side): W}, side 0 = minus edge, 1 = plus edge."""
        if c in edges:
            return edges[c]
        W0 = prim(c)
        Wm, Wp = {}, {}
        for d in range(3):
            a, b = prim(shift(c, d, -1)), prim(shift(c, d, +1))
            if recon == "plm":
                em, ep = zip(*[plm_edges(a[q], W0[q], b[q], beta) for q in range(5)])
            else:
                a2, b2 = prim(shift(c, d, -2)), prim(shift(c, d, +2))
                em, ep = zip(*[ppm_edges([a2[q], a[q], W0[q], b[q], b2[q]], beta) for q in range(5)])
            Wm[d], Wp[d] = list(em), list(ep)
        # one COMMON increment from all three directions (unsplit, reading S5)
        dU = [mpf(0)] * 5
        for d in range(3):
            Fm, Fp = phys_flux(d, Wm[d]), phys_flux(d, Wp[d])
            dU = [dU[q] - dt / (2 * dh) * (Fp[q] - Fm[q]) for q in range(5)]
        out = {}
        for d in range(3):
            for side, W in ((0, Wm[d]), (1, Wp[d])):
                U = prim2cons(W)
                out[(d, side)] = cons2prim([U[q] + dU[q] for q in range(5)])
        edges[c] = out
        return out

    def face_flux(c, d):
        """Flux through the face between c and c + e_d."""
        if (c, d) not in fluxes:
            fluxes[(c, d)] = flux_fn(half_step(c)[(d, 1)], half_step(shift(c, d, +1))[(d, 0)], d)
        return fluxes[(c, d)]

    res = {}
    for c in cells:
        i, j, k = c
        tot = [mpf(0)] * 5
        for d in range(3):
            Fp, Fm = face_flux(c, d), face_flux(shift(c, d, -1), d)
            tot = [tot[q] + (Fp[q] - Fm[q]) for q in range(5)]
        res[c] = [mpf(float(cons[q, k, j, i])) - dt / dh * tot[q] for q in range(5)]
    return res
