"""Helpers shared by the -m gpu parity tests: error norms of DESIGN.md reading S14."""
import numpy as np


def conv_err_prim(a, b):
    """Per-state relative error of primitives (5,n): |d rho|/rho, |dp|/p, max|dU|/||U||_2."""
    with np.errstate(divide="ignore", invalid="ignore"):
        e_rho = np.abs(a[0] - b[0]) / np.abs(b[0])
        e_p = np.abs(a[4] - b[4]) / np.abs(b[4])
        un = np.sqrt((b[1:4] ** 2).sum(0))
        e_u = np.abs(a[1:4] - b[1:4]).max(0) / np.where(un > 0, un, 1.0)
    return np.maximum(np.maximum(e_rho, e_p), e_u)


def conv_err_cons(a, b):
    with np.errstate(divide="ignore", invalid="ignore"):
        e_d = np.abs(a[0] - b[0]) / np.abs(b[0])
        e_e = np.abs(a[4] - b[4]) / np.abs(b[4])
        mn = np.sqrt((b[1:4] ** 2).sum(0))
        e_m = np.abs(a[1:4] - b[1:4]).max(0) / np.where(mn > 0, mn, 1.0)
    return np.maximum(np.maximum(e_d, e_e), e_m)


def step_err(a, b, comp_axis):
    """Per-cell one-step error (S14): |dD|/D, |dE|/E, max|dM|/(||M||_2 + E); arrays with the 5
    components along comp_axis."""
    a = np.moveaxis(a, comp_axis, 0)
    b = np.moveaxis(b, comp_axis, 0)
    with np.errstate(divide="ignore", invalid="ignore"):
        e_d = np.abs(a[0] - b[0]) / np.abs(b[0])
        e_e = np.abs(a[4] - b[4]) / np.abs(b[4])
        mn = np.sqrt((b[1:4] ** 2).sum(0)) + np.abs(b[4])
        e_m = np.abs(a[1:4] - b[1:4]).max(0) / mn
    return np.maximum(np.maximum(e_d, e_e), e_m)


def l1_rel(a, b, comp_axis=0):
    """Many-step tolerance (S14): Sum|dq| / Sum|q| for D and Etilde; for each momentum component
    Sum|dM_i| / Sum(||M||_2 + Etilde) (c = 1: same units) -- a momentum component that is zero by
    symmetry has no scale of its own."""
    a = np.moveaxis(a, comp_axis, 0).reshape(5, -1)
    b = np.moveaxis(b, comp_axis, 0).reshape(5, -1)
    num = np.abs(a - b).sum(1)
    den = np.abs(b).sum(1)
    den[1:4] = (np.sqrt((b[1:4] ** 2).sum(0)) + np.abs(b[4])).sum()
    return num / np.maximum(den, 1e-300)


def patches_to_block(patches):
    """(npg,8,5,8,8,8) patch layout (S13: p = ix + 2 iy + 4 iz) -> (npg,5,16,16,16)."""
    npg = patches.shape[0]
    a = patches.reshape(npg, 2, 2, 2, 5, 8, 8, 8)            # pz, py, px, c, z, y, x
    return a.transpose(0, 4, 1, 5, 2, 6, 3, 7).reshape(npg, 5, 16, 16, 16)


def step_err_local(got, want, tiles, ghost):
    """Per-cell one-step error (S14) relative to the LOCAL scale of the conserved field: the update
    subtracts face fluxes whose size is set by the neighbours, so a nearly empty cell next to a
    relativistic beam carries round-off of the beam's magnitude.  scale = max over the cell and its
    six face neighbours (in the ghosted input tile) of |D|, |Etilde|, ||M||_2 + Etilde resp., and
    the cell's own updated value.  got, want: (npg,8,5,8,8,8); tiles: (npg,5,nxt,nxt,nxt)."""
    g, w = patches_to_block(got), patches_to_block(want)
    t = tiles
    sc = [np.abs(t[:, 0]), np.sqrt((t[:, 1:4] ** 2).sum(1)) + np.abs(t[:, 4]), np.abs(t[:, 4])]
    out = []
    G = ghost
    for k, s0 in enumerate(sc):
        m = s0.copy()
        for ax in (1, 2, 3):
            for sh in (-1, 1):
                m = np.maximum(m, np.roll(s0, sh, axis=ax))    # wrap only touches ghost layers (G >= 2)
        out.append(m[:, G:G + 16, G:G + 16, G:G + 16])
    sD = np.maximum(out[0], np.abs(w[:, 0]))
    sM = np.maximum(out[1], np.sqrt((w[:, 1:4] ** 2).sum(1)) + np.abs(w[:, 4]))
    sE = np.maximum(out[2], np.abs(w[:, 4]))
    e = np.maximum(np.abs(g[:, 0] - w[:, 0]) / sD, np.abs(g[:, 4] - w[:, 4]) / sE)
    return np.maximum(e, np.abs(g[:, 1:4] - w[:, 1:4]).max(1) / sM)


# ---------------------------------------------------------------------------------------------------------
# Tolerance of a one-step comparison DERIVED from the paper's error model (Eq. 20): the inversion of a
# state with Mach number M returns h, rho, p (and U = M/(D h)) with relative uncertainty (1 + M^2) eps, whatever
# the order of evaluation.  The conserved state itself re-enters the fluxes exactly (F = U v_n + pressure terms)
# and v_n = M_n/(E + p) is well conditioned, so what two correct fp64 implementations whose half-step states
# differ in the last bit disagree on is (i) the PRESSURE of the face states, delta p = (1 + M^2) eps p, which
# enters the momentum and energy fluxes directly and the mass flux through v_n and lambda* with a factor
# D/(E + p), and (ii) the SOUND SPEED (T = p/rho), i.e. the wave speeds: in the two-wave averages the weights
# (v_L - S_L)/(S_R - S_L) and (S_R - v_R)/(S_R - S_L) are ratios of sound-speed-sized numbers, uncertain by
# (1 + M^2) eps RELATIVELY, and they multiply S U with |S| <~ c_s wherever the averages are used at all
# (a supersonic face takes the upwind flux): delta F ~ (1 + M^2) eps c_s times the largest neighbouring scale.
# Per cell and per norm q of S14, with the (2g+1)^3 stencil the update depends on:
#     tol_q = max(1e-11, C (dt/dh) { max_stencil[(1 + M^2) eps p w_q] + max_stencil[(1 + M^2) eps c_s] L_q } / own_q)
# w_D = D/(D + Etilde), w_M = w_E = 1; L_q = largest scale of norm q among the cell and its face neighbours;
# C = 4 (six faces, dt/dh <= 0.5).
def _cs2_numpy(T):
    """P:129 Eq. 14 with h = Eq. 10 (tolerance scale only: not a parity reference)."""
    h = 2.5 * T + np.sqrt(2.25 * T * T + 1.0)
    return T * (5.0 * h - 8.0 * T) / (3.0 * h * (h - T))


def eq20_uncertainties(ref, tiles):
    """((1 + Mach^2) eps p, (1 + Mach^2) eps c_s) of every tile cell from the ORACLE's primitives;
    tiles (npg,5,n,n,n)."""
    npg = tiles.shape[0]
    sh = tiles.shape[2:]
    W = ref.cons2prim(np.ascontiguousarray(tiles.transpose(1, 0, 2, 3, 4)).reshape(5, -1))[0].reshape(5, npg, *sh)
    cs2 = _cs2_numpy(W[4] / W[0])
    usq = (W[1:4] ** 2).sum(0)
    cond = (1.0 + usq * (1.0 - cs2) / cs2) * np.finfo(np.float64).eps
    return cond * W[4], cond * np.sqrt(cs2)


def blocks_of_cells(a):
    """(npg,8,8,8,8) per-cell values in patch order (S13) -> (npg,16,16,16)."""
    npg = a.shape[0]
    return a.reshape(npg, 2, 2, 2, 8, 8, 8).transpose(0, 1, 4, 2, 5, 3, 6).reshape(npg, 16, 16, 16)


def step_err_eq20(ref, got, want, tiles, ghost, dt, dh, C=4.0, floor=1e-11):
    """Per-cell S14 errors of got vs want (npg,8,5,8,8,8) and their Eq.-20-derived tolerances.
    Returns (err (npg,16,16,16), tol (npg,16,16,16)): the comparison passes where err <= tol."""
    from scipy.ndimage import maximum_filter
    g, w = patches_to_block(got), patches_to_block(want)
    G = ghost
    size = (1, 2 * G + 1, 2 * G + 1, 2 * G + 1)
    dp, ds = eq20_uncertainties(ref, tiles)
    t = tiles
    dp_d = dp * np.abs(t[:, 0]) / (np.abs(t[:, 0]) + np.abs(t[:, 4]))
    sl = (slice(None), slice(G, G + 16), slice(G, G + 16), slice(G, G + 16))
    dpm = maximum_filter(dp, size=size, mode="nearest")[sl]
    dpd = maximum_filter(dp_d, size=size, mode="nearest")[sl]
    dsm = maximum_filter(ds, size=size, mode="nearest")[sl]
    sc = [np.abs(t[:, 0]), np.sqrt((t[:, 1:4] ** 2).sum(1)) + np.abs(t[:, 4]), np.abs(t[:, 4])]
    loc = []
    for s0 in sc:
        m = s0.copy()
        for ax in (1, 2, 3):
            for sh in (-1, 1):
                m = np.maximum(m, np.roll(s0, sh, axis=ax))       # wrap only touches ghost layers
        loc.append(m[sl])
    own = [np.abs(w[:, 0]), np.sqrt((w[:, 1:4] ** 2).sum(1)) + np.abs(w[:, 4]), np.abs(w[:, 4])]
    errs = [np.abs(g[:, 0] - w[:, 0]), np.abs(g[:, 1:4] - w[:, 1:4]).max(1), np.abs(g[:, 4] - w[:, 4])]
    err = np.zeros_like(own[0])
    tol = np.full_like(own[0], floor)
    ratio = np.zeros_like(own[0])
    with np.errstate(divide="ignore", invalid="ignore"):
        for e, o, d, l in zip(errs, own, (dpd, dpm, dpm), loc):
            en = np.where(o > 0, e / o, np.where(e > 0, np.inf, 0.0))
            tn = np.maximum(floor, C * (dt / dh) * (d + dsm * np.maximum(l, o)) / o)
            worse = en / tn > ratio
            ratio = np.where(worse, en / tn, ratio)
            err = np.where(worse, en, err)
            tol = np.where(worse, tn, tol)
    return err, tol


def report(name, **kw):
    """Append one line of measured parity figures to gpurun_out/parity_report.jsonl (documentation only)."""
    import json
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    os.makedirs(os.path.join(root, "gpurun_out"), exist_ok=True)
    with open(os.path.join(root, "gpurun_out", "parity_report.jsonl"), "a") as f:
        f.write(json.dumps({"test": name, **{k: (float(v) if isinstance(v, (np.floating, float)) else v) for k, v in kw.items()}}) + "\n")
