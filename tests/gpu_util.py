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
    """Sum|dq| / Sum|q| per component (100-step tolerance, S14)."""
    a = np.moveaxis(a, comp_axis, 0).reshape(5, -1)
    b = np.moveaxis(b, comp_axis, 0).reshape(5, -1)
    return np.abs(a - b).sum(1) / np.maximum(np.abs(b).sum(1), 1e-300)
