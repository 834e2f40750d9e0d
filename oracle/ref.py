"""ctypes/numpy binding of the CPU oracle (TEST INFRASTRUCTURE ONLY -- see srhd_ref.hpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from paper_2012_11130_b200.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_LIB = None
_DP = C.POINTER(C.c_double)


def _is_f32():
    return _VARIANT == "f32"


def rdtype():
    """numpy dtype of the oracle's `real` in the current variant (float32 for "f32", x87 long double for "ext",
    else float64)."""
    if _VARIANT == "ext":
        return np.longdouble
    return np.float32 if _is_f32() else np.float64


def _D(x=None):
    """ctypes type of `real` (called without an argument) or a `real` scalar argument."""
    t = C.c_longdouble if _VARIANT == "ext" else (C.c_float if _is_f32() else C.c_double)
    return t if x is None else t(x)


class Params(C.Structure):
    """srhd_ref_params; defaults are the readings S2/S3/S9 of DESIGN.md."""
    _fields_ = [("recon", C.c_int), ("riemann", C.c_int), ("minmod_coeff", C.c_double),
                ("max_retry", C.c_int), ("newton_rtol", C.c_double), ("newton_max_iter", C.c_int),
                ("ghost", C.c_int), ("integrator", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("n_c2p_fail", C.c_ulonglong), ("n_retry_pg", C.c_ulonglong),
                ("n_unphys_final", C.c_ulonglong), ("newton_iters", C.c_ulonglong),
                ("max_speed", C.c_double), ("n_passes", C.c_ulonglong)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def params(recon="plm", riemann="hllc", minmod_coeff=1.5, max_retry=8, newton_rtol=1e-15,
           newton_max_iter=20, integrator="mhm"):
    r = {"plm": 0, "ppm": 1}[recon] if isinstance(recon, str) else int(recon)
    s = {"hlle": 0, "hllc": 1}[riemann] if isinstance(riemann, str) else int(riemann)
    v = {"mhm": 0, "vl": 1}[integrator] if isinstance(integrator, str) else int(integrator)
    return Params(r, s, minmod_coeff, max_retry, newton_rtol, newton_max_iter, (2 if r == 0 else 3) + v, v)


_LIBS = {}
_VARIANT = ""


class variant:
    """with ref.variant("fma"): ... -- route every call to the oracle built with FMA contraction allowed (a
    second rounding of the same formulas; oracle/build.py).  Never the parity reference."""

    def __init__(self, name):
        self.name = name

    def __enter__(self):
        global _VARIANT, _LIB
        self.prev = _VARIANT
        _VARIANT, _LIB = self.name, _LIBS.get(self.name)
        lib()

    def __exit__(self, *a):
        global _VARIANT, _LIB
        _VARIANT, _LIB = self.prev, _LIBS.get(self.prev)


def lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(_build.build(variant=_VARIANT))
        _LIBS[_VARIANT] = L
        for name in ("htilde_of_T", "T_of_htilde", "dT_dhtilde", "cs2_of_T", "smax_of_umax"):
            f = getattr(L, "srhd_ref_" + name)
            f.restype, f.argtypes = _D(), [_D()]
        for name in ("f_eq15", "df_eqA1", "htilde_guess"):
            f = getattr(L, "srhd_ref_" + name)
            f.restype, f.argtypes = _D(), [_D(), _D()]
        L.srhd_ref_limited_slope.restype = _D()
        L.srhd_ref_limited_slope.argtypes = [_D(), _D(), _D()]
        L.srhd_ref_umax_of_prim.restype = _D()
        L.srhd_ref_umax_of_prim.argtypes = [_DP]
        L.srhd_ref_step_box.restype = C.c_int
        _LIB = L
    return _LIB


def _p(a):
    return a.ctypes.data_as(_DP)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=rdtype())
    return a


# ---- scalar EoS helpers (vectorised over numpy inputs by a Python loop; test-sized only) ----
def _vec1(name, x):
    f = getattr(lib(), "srhd_ref_" + name)
    x = np.asarray(x, dtype=np.float64)   # scalar hooks take Python floats
    return np.array([f(float(v)) for v in x.ravel()]).reshape(x.shape) if x.ndim else f(float(x))


def htilde_of_T(T): return _vec1("htilde_of_T", T)
def T_of_htilde(ht): return _vec1("T_of_htilde", ht)
def dT_dhtilde(ht): return _vec1("dT_dhtilde", ht)
def cs2_of_T(T): return _vec1("cs2_of_T", T)
def smax_of_umax(u): return _vec1("smax_of_umax", u)
def f_eq15(ht, musq): return lib().srhd_ref_f_eq15(float(ht), float(musq))
def df_eqA1(ht, musq): return lib().srhd_ref_df_eqA1(float(ht), float(musq))
def htilde_guess(L, musq): return lib().srhd_ref_htilde_guess(float(L), float(musq))
def limited_slope(sL, sR, beta): return lib().srhd_ref_limited_slope(float(sL), float(sR), float(beta))


def umax_of_prim(W):
    W = _f64(W)
    return lib().srhd_ref_umax_of_prim(_p(W))


def recon_1d(recon, a, beta, beta0):
    a = _f64(a)
    am, ap = _D()(), _D()()
    lib().srhd_ref_recon_1d(C.c_int(recon), _p(a), _D(beta), _D(beta0), C.byref(am), C.byref(ap))
    return am.value, ap.value


# ---- conversions on SoA arrays of shape (5, n) ----
def prim2cons(prim):
    prim = _f64(prim)
    assert prim.ndim == 2 and prim.shape[0] == 5
    cons = np.empty_like(prim)
    n = prim.shape[1]
    lib().srhd_ref_prim2cons(_p(prim), _p(cons), C.c_size_t(n), C.c_size_t(n))
    return cons


def cons2prim(cons, par=None, diag=False):
    cons = _f64(cons)
    assert cons.ndim == 2 and cons.shape[0] == 5
    par = par or params()
    prim = np.empty_like(cons)
    n = cons.shape[1]
    if diag:
        ht = np.empty(n, dtype=rdtype())
        it = np.empty(n, dtype=np.int32)
        bad = np.empty(n, dtype=np.uint8)
        lib().srhd_ref_cons2prim_diag(_p(cons), _p(prim), C.c_size_t(n), C.c_size_t(n), C.byref(par),
                                      _p(ht), it.ctypes.data_as(C.POINTER(C.c_int)),
                                      bad.ctypes.data_as(C.POINTER(C.c_ubyte)))
        return prim, ht, it, bad
    st = Stats()
    lib().srhd_ref_cons2prim(_p(cons), _p(prim), C.c_size_t(n), C.c_size_t(n), C.byref(par), C.byref(st))
    return prim, st


def is_physical(cons):
    """Eq. 30 as the update applies it to an updated cell (O9): bool per state of a (5, n) list."""
    cons = _f64(cons)
    assert cons.ndim == 2 and cons.shape[0] == 5
    n = cons.shape[1]
    ok = np.empty(n, dtype=np.uint8)
    lib().srhd_ref_is_physical(_p(cons), ok.ctypes.data_as(C.POINTER(C.c_ubyte)), C.c_size_t(n), C.c_size_t(n))
    return ok.astype(bool)


def max_signal_speed(cons, par=None):
    cons = _f64(cons)
    par = par or params()
    n = cons.shape[1]
    out = _D()()
    lib().srhd_ref_max_signal_speed(_p(cons), C.c_size_t(n), C.c_size_t(n), C.byref(par), C.byref(out))
    return out.value


def phys_flux(d, W, U):
    W, U = _f64(W), _f64(U)
    F = np.empty(5, dtype=rdtype())
    lib().srhd_ref_phys_flux(C.c_int(d), _p(W), _p(U), _p(F))
    return F


def wave_speeds(d, W):
    """(lambda_-, lambda_+) of one primitive state along direction d (reading S6)."""
    return tuple(wave_speed_differences(d, W)[:2])


def wave_speed_differences(d, W):
    """[lambda_-, lambda_+, lambda_+ - v_n, v_n - lambda_-, 1 - lambda_+, 1 + lambda_-] (reading S6)."""
    W = _f64(W)
    out = np.empty(6, dtype=rdtype())
    lib().srhd_ref_wave_speeds(C.c_int(d), _p(W), _p(out))
    return out


def riemann_flux(riemann, d, WL, UL, WR, UR):
    WL, UL, WR, UR = map(_f64, (WL, UL, WR, UR))
    s = {"hlle": 0, "hllc": 1}[riemann] if isinstance(riemann, str) else int(riemann)
    F = np.empty(5, dtype=rdtype())
    lib().srhd_ref_riemann_flux(C.c_int(s), C.c_int(d), _p(WL), _p(UL), _p(WR), _p(UR), _p(F))
    return F


# ---- fluid step ----
def step_box(cons_in, dt, dh, par):
    """cons_in (5, nz+2g, ny+2g, nx+2g) -> (cons_out (5,nz,ny,nx), stats, passes)."""
    cons_in = _f64(cons_in)
    g = par.ghost
    _, sz, sy, sx = cons_in.shape
    nx, ny, nz = sx - 2 * g, sy - 2 * g, sz - 2 * g
    out = np.empty((5, nz, ny, nx), dtype=rdtype())
    st = Stats()
    passes = lib().srhd_ref_step_box(_p(cons_in), _p(out), C.c_int(nx), C.c_int(ny), C.c_int(nz),
                                     _D(dt), _D(dh), C.byref(par), C.byref(st))
    return out, st, passes


def fluid_step(cons_in, dt, dh, par, nthreads=0):
    """cons_in (npg,5,nxt,nxt,nxt) -> (cons_out (npg,8,5,8,8,8), stats)."""
    cons_in = _f64(cons_in)
    npg = cons_in.shape[0]
    nxt = 16 + 2 * par.ghost
    assert cons_in.shape == (npg, 5, nxt, nxt, nxt)
    out = np.empty((npg, 8, 5, 8, 8, 8), dtype=rdtype())
    st = Stats()
    lib().srhd_ref_fluid_step(_p(cons_in), _p(out), C.c_int(npg), _D(dt), _D(dh), C.byref(par),
                              C.byref(st), C.c_int(nthreads))
    return out, st


def fluid_step_fluxes(cons_in, dt, dh, par, nthreads=0):
    """As fluid_step, plus the patch-boundary fluxes (npg,8,6,5,8,8) of the accepted pass."""
    cons_in = _f64(cons_in)
    npg = cons_in.shape[0]
    out = np.empty((npg, 8, 5, 8, 8, 8), dtype=rdtype())
    flux = np.empty((npg, 8, 6, 5, 8, 8), dtype=rdtype())
    st = Stats()
    lib().srhd_ref_fluid_step_fluxes(_p(cons_in), _p(out), _p(flux), C.c_int(npg), _D(dt), _D(dh),
                                     C.byref(par), C.byref(st), C.c_int(nthreads))
    return out, flux, st


REFINE_Q = {None: 0, "none": 0, "D": 1, "Etilde": 2, "rho": 3, "gamma": 4}


def refine_flags(cons_in, par, quantity="rho", c_q=0.3, mom_over_d=0.0):
    """(npg,5,nxt,nxt,nxt) tiles -> (npg,8) uint8 patch flags (Eq. 33 / |M|/D criteria)."""
    cons_in = _f64(cons_in)
    npg = cons_in.shape[0]
    flags = np.zeros((npg, 8), dtype=np.uint8)
    lib().srhd_ref_refine_flags(_p(cons_in), C.c_int(npg), C.c_int(REFINE_Q[quantity]), _D(c_q), _D(mom_over_d),
                                C.byref(par), flags.ctypes.data_as(C.POINTER(C.c_ubyte)))
    return flags


def flux_correction(patches, flux_coarse, flux_fine, face_patch, face_id, dt, dh):
    """(corrected copy of patches (np,5,8,8,8), number of skipped cells)."""
    out = _f64(patches).copy()
    fc, ff = _f64(flux_coarse), _f64(flux_fine)
    fp = np.ascontiguousarray(face_patch, dtype=np.int32)
    fi = np.ascontiguousarray(face_id, dtype=np.int32)
    f = lib().srhd_ref_flux_correction
    f.restype = C.c_ulonglong
    ip = C.POINTER(C.c_int)
    n = f(_p(out), _p(fc), _p(ff), fp.ctypes.data_as(ip), fi.ctypes.data_as(ip), C.c_int(len(fp)), _D(dt), _D(dh))
    return out, int(n)


def ghost_interp(coarse, beta, par=None):
    """coarse (5,nz,ny,nx) -> (fine (5,2(nz-2),2(ny-2),2(nx-2)), fallback flags (nz-2,ny-2,nx-2), count)."""
    coarse = _f64(coarse)
    par = par or params()
    _, nz, ny, nx = coarse.shape
    fine = np.empty((5, 2 * (nz - 2), 2 * (ny - 2), 2 * (nx - 2)))
    fb = np.zeros((nz - 2, ny - 2, nx - 2), dtype=np.uint8)
    f = lib().srhd_ref_ghost_interp
    f.restype = C.c_ulonglong
    n = f(_p(coarse), C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(fine), _D(beta), C.byref(par),
          fb.ctypes.data_as(C.POINTER(C.c_ubyte)))
    return fine, fb, int(n)


def _bc(bc):
    m = {"periodic": 0, "outflow": 1}
    return (C.c_int * 6)(*[m[b] if isinstance(b, str) else int(b) for b in bc])


def _inflow(inflow):
    if inflow is None:
        return None, None
    mask, cons = inflow
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    cons = _f64(cons)
    return mask, cons


def grid_pad(grid, g, bc, inflow=None):
    grid = _f64(grid)
    _, nz, ny, nx = grid.shape
    out = np.empty((5, nz + 2 * g, ny + 2 * g, nx + 2 * g), dtype=rdtype())
    mask, cons = _inflow(inflow)
    lib().srhd_ref_grid_pad(_p(grid), _p(out), C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(g), _bc(bc),
                            mask.ctypes.data_as(C.POINTER(C.c_ubyte)) if mask is not None else None,
                            _p(cons) if cons is not None else None)
    return out


def grid_gather(grid, g, bc, inflow=None):
    grid = _f64(grid)
    _, nz, ny, nx = grid.shape
    assert nx % 16 == 0 and ny % 16 == 0 and nz % 16 == 0
    npg = (nx // 16) * (ny // 16) * (nz // 16)
    nxt = 16 + 2 * g
    out = np.empty((npg, 5, nxt, nxt, nxt), dtype=rdtype())
    mask, cons = _inflow(inflow)
    lib().srhd_ref_grid_gather(_p(grid), _p(out), C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_int(g), _bc(bc),
                               mask.ctypes.data_as(C.POINTER(C.c_ubyte)) if mask is not None else None,
                               _p(cons) if cons is not None else None)
    return out


def grid_scatter(cons_out, shape):
    cons_out = _f64(cons_out)
    nz, ny, nx = shape
    grid = np.empty((5, nz, ny, nx), dtype=rdtype())
    lib().srhd_ref_grid_scatter(_p(cons_out), _p(grid), C.c_int(nx), C.c_int(ny), C.c_int(nz))
    return grid


def grid_step_tiled(grid, dt, dh, par, bc, inflow=None, nthreads=0):
    """One step of the uniform grid through the patch-group path: gather -> fluid_step -> scatter."""
    tiles = grid_gather(grid, par.ghost, bc, inflow)
    out, st = fluid_step(tiles, dt, dh, par, nthreads)
    return grid_scatter(out, grid.shape[1:]), st


def grid_step_whole(grid, dt, dh, par, bc, inflow=None):
    """One step of the uniform grid as ONE box (no tiling): pad -> step_box."""
    out, st, passes = step_box(grid_pad(grid, par.ghost, bc, inflow), dt, dh, par)
    return out, st, passes


def cfl_dt(grid, cfl, dh, par=None):
    """P:252 Eq. 28: dt = C_CFL * dh / S_max."""
    s = max_signal_speed(grid.reshape(5, -1), par)
    return cfl * dh / s
