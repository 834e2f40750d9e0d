"""One pass of the fluid step and the retry ladder (readings S9/S10/S15)
re-assembled in numpy/Python from the oracle's PER-STATE functions (ref.cons2prim, ref.recon_1d,
ref.prim2cons, ref.phys_flux, ref.riemann_flux), each of which has its own pins.  It shares no line with
oracle/srhd_ref.cpp's step_box: cell loops, stencil indexing, the Hancock coupling of the three directions,
face pairing, the update and the pass / retry logic are all written again here, in the order the
readings fix (S5: one common increment; S12: ((x)+(y))+(z)), so that step_box can be compared with it
BIT FOR BIT on small boxes.  Test infrastructure only; slow (ctypes calls in Python loops).
"""
import numpy as np


def _c2p(ref, U, par):
    """U (5,n) -> (W (5,n), bad (n,) bool): Eq. 15-18 with the Eq. 30 verdict of each state."""
    W, _, _, bad = ref.cons2prim(np.ascontiguousarray(U), par, diag=True)
    return W, bad.astype(bool)


def one_pass(ref, cons_in, dt, dh, par, beta):
    """cons_in (5, nz+2g, ny+2g, nx+2g) -> (cons_out (5,nz,ny,nx), face_fail, cell_fail, flux dict)."""
    g = par.ghost
    _, sz, sy, sx = cons_in.shape
    nx, ny, nz = sx - 2 * g, sy - 2 * g, sz - 2 * g
    W, _ = _c2p(ref, cons_in.reshape(5, -1), par)
    W = W.reshape(cons_in.shape)                      # index [q, k+g, j+g, i+g]
    ext = (nx, ny, nz)
    hdt, dtdh = dt / (2.0 * dh), dt / dh
    # ---- O5b + O6: evolved conserved edge states of every cell with at most one index outside
    Um, Up = {}, {}
    for k in range(-1, nz + 1):
        for j in range(-1, ny + 1):
            for i in range(-1, nx + 1):
                c = (i, j, k)
                if sum(1 for a, n in zip(c, ext) if a < 0 or a >= n) > 1:
                    continue
                Wm, Wp = np.empty((3, 5)), np.empty((3, 5))
                for d in range(3):
                    for q in range(5):
                        a = np.zeros(5)
                        for m in range(-2, 3):
                            if par.recon == 0 and abs(m) == 2:
                                continue              # PLM never reads them (and g = 2 may not hold them)
                            cc = list(c)
                            cc[d] += m
                            a[m + 2] = W[q, cc[2] + g, cc[1] + g, cc[0] + g]
                        Wm[d, q], Wp[d, q] = ref.recon_1d(par.recon, a, beta, par.minmod_coeff)
                Ucm, Ucp = ref.prim2cons(Wm.T.copy()).T, ref.prim2cons(Wp.T.copy()).T
                dF = np.empty((3, 5))
                for d in range(3):
                    dF[d] = ref.phys_flux(d, Wp[d], Ucp[d]) - ref.phys_flux(d, Wm[d], Ucm[d])
                dU = -hdt * ((dF[0] + dF[1]) + dF[2])                  # S5: ONE common increment
                Um[c], Up[c] = Ucm + dU, Ucp + dU
    # ---- O7: one Riemann problem per face that touches an interior cell
    flux, face_fail = {}, 0
    for d in range(3):
        lo = [0, 0, 0]
        lo[d] = -1
        for k in range(lo[2], nz):
            for j in range(lo[1], ny):
                for i in range(lo[0], nx):
                    c = (i, j, k)
                    cr = list(c)
                    cr[d] += 1
                    UL, UR = Up[c][d], Um[tuple(cr)][d]
                    WLR, bad = _c2p(ref, np.stack([UL, UR], axis=1), par)
                    face_fail += int(bad.sum())                        # S15
                    flux[(c, d)] = ref.riemann_flux(par.riemann, d, WLR[:, 0], UL, WLR[:, 1], UR)
    # ---- O8 + O9
    out = np.empty((5, nz, ny, nx))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                df = [flux[((i, j, k), d)] - flux[(tuple(np.subtract((i, j, k), np.eye(3, dtype=int)[d])), d)]
                      for d in range(3)]
                out[:, k, j, i] = cons_in[:, k + g, j + g, i + g] - dtdh * ((df[0] + df[1]) + df[2])   # S12
    _, bad = _c2p(ref, out.reshape(5, -1), par)
    return out, face_fail, int(bad.sum()), flux


def ladder(ref, cons_in, dt, dh, par):
    """P:273 / S9: redo the box with the minmod coefficient reduced by a factor 0.75, at most max_retry
    times, then with a vanished coefficient, whose result is kept (S10).  A failing half-step face state
    fails the pass like a failing updated cell (S15).  Returns (out, passes, face_fail, cell_fail, history)."""
    beta, hist = par.minmod_coeff, []
    for reductions in range(par.max_retry + 2):
        if reductions > 0:
            beta = beta * 0.75 if reductions <= par.max_retry else 0.0
        out, ff, cf, _ = one_pass(ref, cons_in, dt, dh, par, beta)
        hist.append((beta, ff, cf))
        if (ff == 0 and cf == 0) or beta == 0.0:
            return out, reductions + 1, ff, cf, hist
    raise AssertionError("unreachable")


# ---------------------------------------------------------------------------------------------------------
# VL integrator (reading S18), re-assembled the same way
def vl_predictor(ref, cons_in, dt, dh, par):
    """Stages V1-V3: primitives of the half-step state U - dt/(2 dh) div F1 (first-order fluxes from cell-centre
    states) for the cells with all indices in -(g-1)..n+g-2.  Returns (Wh dict, number of Eq. 30 failures)."""
    g = par.ghost
    _, sz, sy, sx = cons_in.shape
    nx, ny, nz = sx - 2 * g, sy - 2 * g, sz - 2 * g
    W, _ = _c2p(ref, cons_in.reshape(5, -1), par)
    W = W.reshape(cons_in.shape)
    hdt = dt / (2.0 * dh)
    at = lambda c: (slice(None), c[2] + g, c[1] + g, c[0] + g)
    lo, hi = -(g - 1), (nx + g - 2, ny + g - 2, nz + g - 2)
    F1 = {}

    def flux1(c, d):
        if (c, d) not in F1:
            r = list(c)
            r[d] += 1
            r = tuple(r)
            F1[(c, d)] = ref.riemann_flux(par.riemann, d, W[at(c)], cons_in[at(c)], W[at(r)], cons_in[at(r)])
        return F1[(c, d)]

    Wh, fails = {}, 0
    for k in range(lo, hi[2] + 1):
        for j in range(lo, hi[1] + 1):
            for i in range(lo, hi[0] + 1):
                c = (i, j, k)
                df = []
                for d in range(3):
                    l = list(c)
                    l[d] -= 1
                    df.append(flux1(c, d) - flux1(tuple(l), d))
                Uh = cons_in[at(c)] - hdt * ((df[0] + df[1]) + df[2])
                w, bad = _c2p(ref, Uh.reshape(5, 1), par)
                fails += int(bad[0])
                Wh[c] = w[:, 0]
    return Wh, fails


def one_pass_vl(ref, cons_in, Wh, dt, dh, par, beta):
    """Stages V4-V6 with coefficient beta -> (cons_out, cell_fail)."""
    g = par.ghost
    _, sz, sy, sx = cons_in.shape
    nx, ny, nz = sx - 2 * g, sy - 2 * g, sz - 2 * g
    ext = (nx, ny, nz)
    edges = {}
    for k in range(-1, nz + 1):
        for j in range(-1, ny + 1):
            for i in range(-1, nx + 1):
                c = (i, j, k)
                if sum(1 for a, n in zip(c, ext) if a < 0 or a >= n) > 1:
                    continue
                Wm, Wp = np.empty((3, 5)), np.empty((3, 5))
                for d in range(3):
                    for q in range(5):
                        a = np.zeros(5)
                        for m in range(-2, 3):
                            if par.recon == 0 and abs(m) == 2:
                                continue
                            cc = list(c)
                            cc[d] += m
                            a[m + 2] = Wh[tuple(cc)][q]
                        Wm[d, q], Wp[d, q] = ref.recon_1d(par.recon, a, beta, par.minmod_coeff)
                edges[c] = (Wm, Wp, ref.prim2cons(Wm.T.copy()).T, ref.prim2cons(Wp.T.copy()).T)
    flux = {}
    for d in range(3):
        lo = [0, 0, 0]
        lo[d] = -1
        for k in range(lo[2], nz):
            for j in range(lo[1], ny):
                for i in range(lo[0], nx):
                    c = (i, j, k)
                    r = list(c)
                    r[d] += 1
                    L, R = edges[c], edges[tuple(r)]
                    flux[(c, d)] = ref.riemann_flux(par.riemann, d, L[1][d], L[3][d], R[0][d], R[2][d])
    out = np.empty((5, nz, ny, nx))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                df = [flux[((i, j, k), d)] - flux[(tuple(np.subtract((i, j, k), np.eye(3, dtype=int)[d])), d)]
                      for d in range(3)]
                out[:, k, j, i] = cons_in[:, k + g, j + g, i + g] - (dt / dh) * ((df[0] + df[1]) + df[2])
    _, bad = _c2p(ref, out.reshape(5, -1), par)
    return out, int(bad.sum())


def ladder_vl(ref, cons_in, dt, dh, par):
    """The retry ladder around the corrector; the predictor (beta independent) is computed once and its
    Eq. 30 failures are counted, not retried (S18).  Returns (out, passes, half_fail, cell_fail, history)."""
    Wh, half_fail = vl_predictor(ref, cons_in, dt, dh, par)
    beta, hist = par.minmod_coeff, []
    for reductions in range(par.max_retry + 2):
        if reductions > 0:
            beta = beta * 0.75 if reductions <= par.max_retry else 0.0
        out, cf = one_pass_vl(ref, cons_in, Wh, dt, dh, par, beta)
        hist.append((beta, cf))
        if cf == 0 or beta == 0.0:
            return out, reductions + 1, half_fail, cf, hist
    raise AssertionError("unreachable")
