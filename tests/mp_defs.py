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


def h_of_T(T):
    T = mpf(T)
    return mpf(5) / 2 * T + sqrt(mpf(9) / 4 * T * T + 1)


def cs2_of_T(T):
    T = mpf(T)
    h = h_of_T(T)
    return T / (3 * h) * (5 * h - 8 * T) / (h - T)


def prim2cons(W):
    rho, ux, uy, uz, p = [mpf(float(w)) for w in W]
    T = p / rho
    h = h_of_T(T)
    g = sqrt(1 + ux * ux + uy * uy + uz * uz)
    D = rho * g
    E = D * h * g - p
    return [D, D * h * ux, D * h * uy, D * h * uz, E - D]


def phys_flux(d, W):
    """Eq. 4a, 4b, and the reduced-energy flux in its DEFINING form (M_n - D v_n), line 81."""
    rho, ux, uy, uz, p = [mpf(float(w)) for w in W]
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
    rho, ux, uy, uz, p = [mpf(float(w)) for w in W]
    g = sqrt(1 + ux * ux + uy * uy + uz * uz)
    v = [ux / g, uy / g, uz / g]
    v2 = sum(x * x for x in v)
    cs2 = cs2_of_T(p / rho)
    vn = v[d]
    disc = sqrt(cs2 * (1 - v2) * (1 - v2 * cs2 - vn * vn * (1 - cs2)))
    return (vn * (1 - cs2) - disc) / (1 - v2 * cs2), (vn * (1 - cs2) + disc) / (1 - v2 * cs2)
