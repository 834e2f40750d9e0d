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
