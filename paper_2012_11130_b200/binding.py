"""Thin Python binding of the C-ABI library (include/srhd.h): argument marshalling only.

Every function here has the name of the C entry point it calls and does nothing but check tensor
dtype/device/contiguity, allocate the output with torch, and pass raw device pointers plus the
current CUDA stream.  All arithmetic runs in the CUDA kernels of libsrhd_b200.so.  There is no CPU
fallback: if the library is missing or no CUDA device is present, the calls raise.
"""
import ctypes as C
import os

import torch

from . import build as _build

_D = C.c_double
_VP = C.c_void_p

RECON = {"plm": 0, "ppm": 1}
RIEMANN = {"hlle": 0, "hllc": 1}
INTEGRATOR = {"mhm": 0, "vl": 1}
BC = {"periodic": 0, "outflow": 1}


class Params(C.Structure):
    """srhd_params (include/srhd.h)."""
    _fields_ = [("recon", C.c_int), ("riemann", C.c_int), ("minmod_coeff", C.c_double),
                ("max_retry", C.c_int), ("newton_rtol", C.c_double), ("newton_max_iter", C.c_int),
                ("ghost", C.c_int), ("integrator", C.c_int)]


class Stats(C.Structure):
    """srhd_stats (include/srhd.h); lives in device memory, read back with stats_to_host()."""
    _fields_ = [("n_c2p_fail", C.c_ulonglong), ("n_retry_pg", C.c_ulonglong),
                ("n_unphys_final", C.c_ulonglong), ("newton_iters", C.c_ulonglong),
                ("max_speed", C.c_double), ("n_passes", C.c_ulonglong), ("exec_c2p", C.c_ulonglong),
                ("exec_newton", C.c_ulonglong), ("exec_riemann", C.c_ulonglong), ("exec_hancock", C.c_ulonglong),
                ("n_uniform_pg", C.c_ulonglong)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}

    def algorithm_dict(self):
        """The counters the algorithm defines (everything but the executed-work figures)."""
        return {k: getattr(self, k) for k, _ in self._fields_ if not k.startswith("exec_") and k != "n_uniform_pg"}


SYMBOLS = ["srhd_default_params", "srhd_prim2cons", "srhd_cons2prim", "srhd_max_signal_speed",
           "srhd_fluid_step", "srhd_fluid_step_noalloc", "srhd_fluid_step_fluxes", "srhd_fluid_step_cfl", "srhd_refine_flags", "srhd_flux_correction", "srhd_ghost_interp", "srhd_workspace_bytes", "srhd_grid_gather", "srhd_grid_scatter", "srhd_grid_scatter_speed", "srhd_patch_gather_speed", "srhd_grid_step_cfl",
           "srhd_fp64_peak_probe", "srhd_issue_probe", "srhd_quotient_check", "srhd_error_string", "srhd_build_is_exact", "srhd_build_variant"]

_LIBS = {}
_CUR_REAL = torch.float64   # srhd_real of the library selected by the latest load_library() call


class SrhdError(RuntimeError):
    pass


def load_library(exact=False):
    """dlopen libsrhd_b200[_exact].so (built in-tree by paper_2012_11130_b200.build); `exact` may also name one of
    the variant libraries of build.VARIANTS ("gamma53", "gamma53_exact", "gamma43_exact", "orig_exact")."""
    global _CUR_REAL
    if exact in _LIBS:
        _CUR_REAL = _LIBS[exact]._real_dtype
        return _LIBS[exact]
    path = _build.lib_path(exact)
    if not os.path.exists(path):
        raise SrhdError(f"{path} is missing: run `python -m paper_2012_11130_b200.build` "
                        "(there is no CPU fallback)")
    L = C.CDLL(path)
    L.srhd_default_params.restype = None
    L.srhd_default_params.argtypes = [C.POINTER(Params), C.c_int, C.c_int]
    L.srhd_prim2cons.restype = C.c_int
    L.srhd_prim2cons.argtypes = [_VP, _VP, C.c_size_t, C.c_size_t, _VP]
    L.srhd_cons2prim.restype = C.c_int
    L.srhd_cons2prim.argtypes = [_VP, _VP, C.c_size_t, C.c_size_t, C.POINTER(Params), _VP, _VP]
    L.srhd_max_signal_speed.restype = C.c_int
    L.srhd_max_signal_speed.argtypes = [_VP, C.c_size_t, C.c_size_t, C.POINTER(Params), _VP, _VP]
    L.srhd_fluid_step.restype = C.c_int
    L.srhd_fluid_step.argtypes = [_VP, _VP, C.c_int, _D, _D, C.POINTER(Params), _VP, _VP]
    L.srhd_fluid_step_fluxes.restype = C.c_int
    L.srhd_fluid_step_noalloc.argtypes = [_VP, _VP, C.c_int, _D, _D, C.POINTER(Params), _VP, _VP]
    L.srhd_fluid_step_noalloc.restype = C.c_int
    L.srhd_fluid_step_fluxes.argtypes = [_VP, _VP, _VP, C.c_int, _D, _D, C.POINTER(Params), _VP, _VP]
    L.srhd_fluid_step_cfl.restype = C.c_int
    L.srhd_fluid_step_cfl.argtypes = [_VP, _VP, _VP, C.c_int, _D, _D, _VP, _D, C.POINTER(Params), _VP, _VP]
    L.srhd_refine_flags.restype = C.c_int
    L.srhd_refine_flags.argtypes = [_VP, C.c_int, C.c_int, _D, _D, C.POINTER(Params), _VP, _VP]
    L.srhd_flux_correction.restype = C.c_int
    L.srhd_flux_correction.argtypes = [_VP, _VP, _VP, _VP, _VP, C.c_int, _D, _D, _VP, _VP]
    L.srhd_ghost_interp.restype = C.c_int
    L.srhd_ghost_interp.argtypes = [_VP, C.c_int, C.c_int, C.c_int, _VP, _D, C.POINTER(Params), _VP, _VP, _VP]
    L.srhd_workspace_bytes.restype = C.c_size_t
    L.srhd_workspace_bytes.argtypes = [C.c_int, C.POINTER(Params)]
    L.srhd_grid_gather.restype = C.c_int
    L.srhd_grid_gather.argtypes = [_VP, _VP, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), _VP,
                                   C.POINTER(C.c_double), _VP]
    L.srhd_grid_scatter.restype = C.c_int
    L.srhd_grid_scatter.argtypes = [_VP, _VP, C.c_int, C.c_int, C.c_int, _VP]
    L.srhd_grid_scatter_speed.restype = C.c_int
    L.srhd_grid_scatter_speed.argtypes = [_VP, _VP, C.c_int, C.c_int, C.c_int, C.POINTER(Params), _VP, _VP]
    L.srhd_patch_gather_speed.restype = C.c_int
    L.srhd_patch_gather_speed.argtypes = [_VP, _VP, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), _VP,
                                          C.POINTER(C.c_double), C.POINTER(Params), _VP, _VP]
    L.srhd_grid_step_cfl.restype = C.c_int
    L.srhd_grid_step_cfl.argtypes = [_VP, _VP, _VP, _VP, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), _VP,
                                     C.POINTER(C.c_double), C.c_double, C.c_double, C.c_double, C.POINTER(Params),
                                     _VP, _VP, _VP]
    L.srhd_fp64_peak_probe.restype = C.c_int
    L.srhd_fp64_peak_probe.argtypes = [_VP, C.c_int, C.POINTER(C.c_ulonglong), _VP]
    L.srhd_issue_probe.restype = C.c_int
    L.srhd_issue_probe.argtypes = [_VP, C.c_int, C.c_int, C.POINTER(C.c_ulonglong), _VP]
    L.srhd_quotient_check.restype = C.c_int
    L.srhd_quotient_check.argtypes = [C.c_ulonglong, C.c_ulonglong, C.c_int, _VP, _VP]
    L.srhd_error_string.restype = C.c_char_p
    L.srhd_error_string.argtypes = [C.c_int]
    L.srhd_build_is_exact.restype = C.c_int
    L.srhd_build_is_exact.argtypes = []
    L.srhd_build_variant.restype = C.c_char_p
    L.srhd_build_variant.argtypes = []
    L._real_dtype = torch.float32 if b"precision=f32" in L.srhd_build_variant() else torch.float64
    _CUR_REAL = L._real_dtype
    _LIBS[exact] = L
    return L


def params(recon="plm", riemann="hllc", minmod_coeff=None, max_retry=None, newton_rtol=None,
           newton_max_iter=None, exact=False, integrator="mhm"):
    """srhd_default_params + overrides."""
    p = Params()
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    s = RIEMANN[riemann] if isinstance(riemann, str) else int(riemann)
    load_library(exact).srhd_default_params(C.byref(p), r, s)
    if minmod_coeff is not None:
        p.minmod_coeff = minmod_coeff
    if max_retry is not None:
        p.max_retry = max_retry
    if newton_rtol is not None:
        p.newton_rtol = newton_rtol
    if newton_max_iter is not None:
        p.newton_max_iter = newton_max_iter
    v = INTEGRATOR[integrator] if isinstance(integrator, str) else int(integrator)
    p.integrator = v                    # the VL integrator needs one more layer of ghost zones (include/srhd.h)
    p.ghost += v
    return p


def _check(code, L):
    if code != 0:
        raise SrhdError(f"srhd error {code}: {L.srhd_error_string(code).decode()}")


def _dev(t, name):
    """A state array handed to the library most recently selected by load_library(): contiguous, on the GPU, of
    that library's srhd_real (float64; float32 for the f32 builds)."""
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == _CUR_REAL and t.is_contiguous()):
        raise SrhdError(f"{name} must be a contiguous {_CUR_REAL} CUDA tensor (no CPU fallback)")
    return t


def _stream():
    return torch.cuda.current_stream().cuda_stream


def _tiles(cons_in, par):
    """Validate the ghosted tiles handed to a tile-consuming call: (npg,5,nxt,nxt,nxt), nxt = 16 + 2*par.ghost
    (the C ABI sees only a pointer; a PLM-shaped tile with PPM parameters would be read out of bounds)."""
    cons_in = _dev(cons_in, "cons_in")
    nxt = 16 + 2 * par.ghost
    if cons_in.dim() != 5 or tuple(cons_in.shape[1:]) != (5, nxt, nxt, nxt):
        raise SrhdError(f"cons_in must have shape (npg,5,{nxt},{nxt},{nxt}) for ghost = {par.ghost}")
    return cons_in, cons_in.shape[0]


def _shaped(t, shape, name):
    t = _dev(t, name)
    if tuple(t.shape) != tuple(shape):
        raise SrhdError(f"{name} must have shape {tuple(shape)}, not {tuple(t.shape)}")
    return t


def _inflow(inflow, ny, nx):
    """(mask pointer, 5 doubles) of a fixed-inflow boundary, validated: uint8 CUDA mask of shape (ny,nx)."""
    if inflow is None:
        return None, None
    mask, vals = inflow
    if not (isinstance(mask, torch.Tensor) and mask.is_cuda and mask.dtype == torch.uint8 and mask.is_contiguous()
            and tuple(mask.shape) == (ny, nx)):
        raise SrhdError(f"inflow mask must be a contiguous uint8 CUDA tensor of shape ({ny},{nx})")
    if len(vals) != 5:
        raise SrhdError("inflow state must have 5 components")
    return mask.data_ptr(), (C.c_double * 5)(*[float(v) for v in vals])


def new_stats(device="cuda"):
    """Device buffer holding one srhd_stats (sizeof(Stats) = 88 bytes), zeroed."""
    return torch.zeros(C.sizeof(Stats), dtype=torch.uint8, device=device)


def stats_to_host(stats_buf):
    """One small device->host copy; returns a Stats struct."""
    raw = stats_buf.cpu().numpy().tobytes()
    return Stats.from_buffer_copy(raw)


def prim2cons(prim, cons=None, exact=False):
    """srhd_prim2cons on a (5, n) SoA tensor."""
    L = load_library(exact)
    prim = _dev(prim, "prim")
    n = prim.shape[1]
    cons = torch.empty_like(prim) if cons is None else _dev(cons, "cons")
    _check(L.srhd_prim2cons(prim.data_ptr(), cons.data_ptr(), n, prim.stride(0) if n else 0, _stream()), L)
    return cons


def cons2prim(cons, par=None, prim=None, stats=None, exact=False):
    """srhd_cons2prim on a (5, n) SoA tensor; returns (prim, stats device buffer)."""
    L = load_library(exact)
    cons = _dev(cons, "cons")
    par = par or params(exact=exact)
    n = cons.shape[1]
    prim = torch.empty_like(cons) if prim is None else _dev(prim, "prim")
    stats = new_stats(cons.device) if stats is None else stats
    _check(L.srhd_cons2prim(cons.data_ptr(), prim.data_ptr(), n, cons.stride(0) if n else 0, C.byref(par),
                            stats.data_ptr(), _stream()), L)
    return prim, stats


def max_signal_speed(cons, par=None, out=None, exact=False):
    """srhd_max_signal_speed on a (5, n) SoA tensor; returns a 1-element device tensor."""
    L = load_library(exact)
    cons = _dev(cons, "cons")
    par = par or params(exact=exact)
    n = cons.shape[1]
    out = torch.empty(1, dtype=cons.dtype, device=cons.device) if out is None else out
    _check(L.srhd_max_signal_speed(cons.data_ptr(), n, cons.stride(0) if n else 0, C.byref(par),
                                   out.data_ptr(), _stream()), L)
    return out


def fluid_step(cons_in, dt, dh, par, cons_out=None, stats=None, exact=False):
    """srhd_fluid_step: cons_in (npg,5,nxt,nxt,nxt) -> cons_out (npg,8,5,8,8,8); returns (cons_out, stats)."""
    L = load_library(exact)
    cons_in, npg = _tiles(cons_in, par)
    if cons_out is None:
        cons_out = torch.empty((npg, 8, 5, 8, 8, 8), dtype=cons_in.dtype, device=cons_in.device)
    stats = new_stats(cons_in.device) if stats is None else stats
    _check(L.srhd_fluid_step(cons_in.data_ptr(), _shaped(cons_out, (npg, 8, 5, 8, 8, 8), "cons_out").data_ptr(), npg, float(dt),
                             float(dh), C.byref(par), stats.data_ptr(), _stream()), L)
    return cons_out, stats


NOALLOC_MAX_NPG = 65536   # SRHD_NOALLOC_MAX_NPG of include/srhd.h


def fluid_step_noalloc(cons_in, dt, dh, par, cons_out, stats, exact=False):
    """srhd_fluid_step_noalloc: the MUSCL-Hancock step for programs in which this library must not allocate GPU
    memory (a host code whose pool owns the device, a fixed-footprint step loop).  Same result as fluid_step; the
    pre-pass flags live in a 64 KiB array inside the library instead of a cudaMallocAsync block.  To keep the
    promise on the Python side too, `cons_out` (npg,8,5,8,8,8) and `stats` (new_stats()) are REQUIRED here: this
    wrapper creates no tensor.  At most NOALLOC_MAX_NPG groups per call; calls on one GPU must not overlap (they
    share the array); make the first call on each device during set-up.  Returns (cons_out, stats)."""
    L = load_library(exact)
    cons_in, npg = _tiles(cons_in, par)
    if cons_out is None or stats is None:
        raise SrhdError("fluid_step_noalloc allocates nothing: pass cons_out and stats")
    _check(L.srhd_fluid_step_noalloc(cons_in.data_ptr(), _shaped(cons_out, (npg, 8, 5, 8, 8, 8), "cons_out").data_ptr(),
                                     npg, float(dt), float(dh), C.byref(par), stats.data_ptr(), _stream()), L)
    return cons_out, stats


def fluid_step_fluxes(cons_in, dt, dh, par, cons_out=None, flux_out=None, stats=None, exact=False):
    """srhd_fluid_step_fluxes: as fluid_step, plus the patch-boundary fluxes (npg,8,6,5,8,8)."""
    L = load_library(exact)
    cons_in, npg = _tiles(cons_in, par)
    if cons_out is None:
        cons_out = torch.empty((npg, 8, 5, 8, 8, 8), dtype=cons_in.dtype, device=cons_in.device)
    if flux_out is None:
        flux_out = torch.empty((npg, 8, 6, 5, 8, 8), dtype=cons_in.dtype, device=cons_in.device)
    stats = new_stats(cons_in.device) if stats is None else stats
    _check(L.srhd_fluid_step_fluxes(cons_in.data_ptr(), _shaped(cons_out, (npg, 8, 5, 8, 8, 8), "cons_out").data_ptr(),
                                    _shaped(flux_out, (npg, 8, 6, 5, 8, 8), "flux_out").data_ptr(), npg, float(dt), float(dh),
                                    C.byref(par), stats.data_ptr(), _stream()), L)
    return cons_out, flux_out, stats


def fluid_step_cfl(cons_in, cfl, dh, max_speed, par, min_speed=0.0, cons_out=None, flux_out=None, stats=None,
                   exact=False):
    """srhd_fluid_step_cfl: dt = cfl*dh/max(*max_speed, min_speed) formed on the device (no host sync)."""
    L = load_library(exact)
    cons_in, npg = _tiles(cons_in, par)
    if cons_out is None:
        cons_out = torch.empty((npg, 8, 5, 8, 8, 8), dtype=cons_in.dtype, device=cons_in.device)
    stats = new_stats(cons_in.device) if stats is None else stats
    _check(L.srhd_fluid_step_cfl(cons_in.data_ptr(), _shaped(cons_out, (npg, 8, 5, 8, 8, 8), "cons_out").data_ptr(),
                                 0 if flux_out is None else _shaped(flux_out, (npg, 8, 6, 5, 8, 8), "flux_out").data_ptr(), npg,
                                 float(cfl), float(dh), _shaped(max_speed, (1,), "max_speed").data_ptr(), float(min_speed),
                                 C.byref(par), stats.data_ptr(), _stream()), L)
    return cons_out, stats


REFINE_Q = {None: 0, "none": 0, "D": 1, "Etilde": 2, "rho": 3, "gamma": 4}


def refine_flags(cons_in, par, quantity="rho", c_q=0.3, mom_over_d=0.0, flags=None, exact=False):
    """srhd_refine_flags: (npg,5,nxt,nxt,nxt) tiles -> (npg,8) uint8 patch flags."""
    L = load_library(exact)
    cons_in, npg = _tiles(cons_in, par)
    if flags is None:
        flags = torch.empty((npg, 8), dtype=torch.uint8, device=cons_in.device)
    if not (flags.is_cuda and flags.dtype == torch.uint8 and flags.is_contiguous() and flags.numel() == npg * 8):
        raise SrhdError(f"flags must be a contiguous uint8 CUDA tensor of {npg * 8} elements")
    q = REFINE_Q[quantity] if not isinstance(quantity, int) else quantity
    _check(L.srhd_refine_flags(cons_in.data_ptr(), npg, q, float(c_q), float(mom_over_d), C.byref(par),
                               flags.data_ptr(), _stream()), L)
    return flags


def flux_correction(patches, flux_coarse, flux_fine, face_patch, face_id, dt, dh, exact=False):
    """srhd_flux_correction (in place on patches (np,5,8,8,8)); returns a 1-element int64 device tensor: skipped cells."""
    L = load_library(exact)
    _dev(patches, "patches"), _dev(flux_coarse, "flux_coarse"), _dev(flux_fine, "flux_fine")
    for t, nm in ((face_patch, "face_patch"), (face_id, "face_id")):
        if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
            raise SrhdError(f"{nm} must be a contiguous int32 CUDA tensor")
    nf = face_patch.numel()
    if tuple(flux_coarse.shape) != (nf, 5, 8, 8) or tuple(flux_fine.shape) != (nf, 5, 8, 8) or face_id.numel() != nf:
        raise SrhdError("flux_coarse / flux_fine must have shape (nf,5,8,8) and face_id nf entries")
    if patches.dim() != 5 or tuple(patches.shape[1:]) != (5, 8, 8, 8) or (nf and int(face_patch.max()) >= patches.shape[0]):
        raise SrhdError("patches must have shape (np,5,8,8,8) and face_patch must index it")
    out = torch.zeros(1, dtype=torch.int64, device=patches.device)
    _check(L.srhd_flux_correction(patches.data_ptr(), flux_coarse.data_ptr(), flux_fine.data_ptr(), face_patch.data_ptr(),
                                  face_id.data_ptr(), nf, float(dt), float(dh), out.data_ptr(), _stream()), L)
    return out


def ghost_interp(coarse, minmod_coeff, par=None, exact=False):
    """srhd_ghost_interp: coarse (5,nz,ny,nx) -> (fine (5,2(nz-2),2(ny-2),2(nx-2)), fallback flags uint8, count tensor)."""
    L = load_library(exact)
    coarse = _dev(coarse, "coarse")
    par = par or params(exact=exact)
    _, nz, ny, nx = coarse.shape
    fine = torch.empty((5, 2 * (nz - 2), 2 * (ny - 2), 2 * (nx - 2)), dtype=coarse.dtype, device=coarse.device)
    fb = torch.zeros((nz - 2, ny - 2, nx - 2), dtype=torch.uint8, device=coarse.device)
    cnt = torch.zeros(1, dtype=torch.int64, device=coarse.device)
    _check(L.srhd_ghost_interp(coarse.data_ptr(), nx, ny, nz, fine.data_ptr(), float(minmod_coeff), C.byref(par),
                               fb.data_ptr(), cnt.data_ptr(), _stream()), L)
    return fine, fb, cnt


def _bc(bc):
    return (C.c_int * 6)(*[BC[b] if isinstance(b, str) else int(b) for b in bc])


def grid_gather(grid, ghost, bc, inflow=None, cons_in=None, exact=False):
    """srhd_grid_gather: grid (5,nz,ny,nx) -> cons_in (npg,5,nxt,nxt,nxt).
    inflow = (mask uint8 CUDA tensor (ny,nx), cons 5 floats) or None."""
    L = load_library(exact)
    grid = _dev(grid, "grid")
    _, nz, ny, nx = grid.shape
    npg = (nx // 16) * (ny // 16) * (nz // 16)
    nxt = 16 + 2 * ghost
    if cons_in is None:
        cons_in = torch.empty((npg, 5, nxt, nxt, nxt), dtype=grid.dtype, device=grid.device)
    mask_ptr, icons = _inflow(inflow, ny, nx)
    _check(L.srhd_grid_gather(grid.data_ptr(), cons_in.data_ptr(), nx, ny, nz, ghost, _bc(bc), mask_ptr,
                              icons, _stream()), L)
    return cons_in


def grid_scatter(cons_out, shape, grid=None, exact=False):
    """srhd_grid_scatter: cons_out (npg,8,5,8,8,8) -> grid (5,nz,ny,nx)."""
    L = load_library(exact)
    cons_out = _dev(cons_out, "cons_out")
    nz, ny, nx = shape
    if grid is None:
        grid = torch.empty((5, nz, ny, nx), dtype=cons_out.dtype, device=cons_out.device)
    _check(L.srhd_grid_scatter(cons_out.data_ptr(), grid.data_ptr(), nx, ny, nz, _stream()), L)
    return grid


def grid_scatter_speed(cons_out, shape, par, grid=None, out=None, exact=False):
    """srhd_grid_scatter_speed: scatter + S_max of the scattered state (1-element device tensor)."""
    L = load_library(exact)
    cons_out = _dev(cons_out, "cons_out")
    nz, ny, nx = shape
    if grid is None:
        grid = torch.empty((5, nz, ny, nx), dtype=cons_out.dtype, device=cons_out.device)
    out = torch.empty(1, dtype=cons_out.dtype, device=cons_out.device) if out is None else out
    _check(L.srhd_grid_scatter_speed(cons_out.data_ptr(), grid.data_ptr(), nx, ny, nz, C.byref(par),
                                     out.data_ptr(), _stream()), L)
    return grid, out


def patch_gather_speed(patches, shape, par, bc, inflow=None, cons_in=None, out=None, exact=False):
    """srhd_patch_gather_speed: patches (npg,8,5,8,8,8) -> tiles (npg,5,nxt,nxt,nxt) and S_max (1 element)."""
    L = load_library(exact)
    nz, ny, nx = shape
    npg = (nx // 16) * (ny // 16) * (nz // 16)
    patches = _shaped(patches, (npg, 8, 5, 8, 8, 8), "patches")
    nxt = 16 + 2 * par.ghost
    if cons_in is not None:
        cons_in = _shaped(cons_in, (npg, 5, nxt, nxt, nxt), "cons_in")
    if cons_in is None:
        cons_in = torch.empty((patches.shape[0], 5, nxt, nxt, nxt), dtype=patches.dtype, device=patches.device)
    out = torch.empty(1, dtype=patches.dtype, device=patches.device) if out is None else out
    mask_ptr, icons = _inflow(inflow, ny, nx)
    _check(L.srhd_patch_gather_speed(patches.data_ptr(), cons_in.data_ptr(), nx, ny, nz, _bc(bc), mask_ptr, icons,
                                     C.byref(par), out.data_ptr(), _stream()), L)
    return cons_in, out


def grid_step_cfl(patches_in, patches_out, cons_in, shape, cfl, dh, par, bc, inflow=None, min_speed=0.0,
                  flux_out=None, stats=None, out=None, exact=False):
    """srhd_grid_step_cfl: one whole step of a uniform grid in the patch layout (patches_in -> patches_out);
    cons_in is the tile scratch (npg,5,nxt,nxt,nxt); returns (patches_out, S_max tensor, stats)."""
    L = load_library(exact)
    patches_in, patches_out, cons_in = _dev(patches_in, "patches_in"), _dev(patches_out, "patches_out"), _dev(cons_in, "cons_in")
    nz, ny, nx = shape
    npg = (nx // 16) * (ny // 16) * (nz // 16)
    nxt = 16 + 2 * par.ghost
    if tuple(patches_in.shape) != (npg, 8, 5, 8, 8, 8) or tuple(patches_out.shape) != (npg, 8, 5, 8, 8, 8):
        raise SrhdError(f"patches must have shape ({npg}, 8, 5, 8, 8, 8)")
    if tuple(cons_in.shape) != (npg, 5, nxt, nxt, nxt):
        raise SrhdError(f"cons_in must have shape ({npg}, 5, {nxt}, {nxt}, {nxt})")
    if flux_out is not None and tuple(_dev(flux_out, "flux_out").shape) != (npg, 8, 6, 5, 8, 8):
        raise SrhdError(f"flux_out must have shape ({npg}, 8, 6, 5, 8, 8)")
    out = torch.empty(1, dtype=patches_in.dtype, device=patches_in.device) if out is None else out
    stats = new_stats(patches_in.device) if stats is None else stats
    mask_ptr, icons = _inflow(inflow, ny, nx)
    _check(L.srhd_grid_step_cfl(patches_in.data_ptr(), patches_out.data_ptr(), cons_in.data_ptr(),
                                None if flux_out is None else flux_out.data_ptr(), nx, ny, nz, _bc(bc), mask_ptr,
                                icons, float(cfl), float(dh), float(min_speed), C.byref(par), stats.data_ptr(),
                                out.data_ptr(), _stream()), L)
    return patches_out, out, stats


def fp64_peak_probe(iters=4096, reps=5):
    """srhd_fp64_peak_probe timed with CUDA events on the current stream: measured DFMA TFLOP/s."""
    L = load_library(False)
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    flops = C.c_ulonglong(0)
    best = 0.0
    for r in range(reps + 1):                       # first launch is warm-up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _check(L.srhd_fp64_peak_probe(sink.data_ptr(), iters, C.byref(flops), _stream()), L)
        e1.record()
        e1.synchronize()
        if r:
            best = max(best, flops.value / (e0.elapsed_time(e1) * 1e-3) / 1e12)
    return best


def quotient_check(n, seed=1, dist=0, exact=False):
    """srhd_quotient_check: (bit mismatches, index of the first) of the canonical quotient vs IEEE division."""
    L = load_library(exact)
    out = torch.zeros(2, dtype=torch.int64, device="cuda")
    _check(L.srhd_quotient_check(int(n), int(seed), int(dist), out.data_ptr(), _stream()), L)
    o = out.cpu().numpy().view("uint64")
    return int(o[0]), int(o[1])


def issue_probe(iters=2048, reps=3):
    """srhd_issue_probe timed with CUDA events: {FFMA per 8 DFMA: DFMA TFLOP/s}.  `python -m
    paper_2012_11130_b200.binding issue_probe` prints the table kept under profiles/."""
    L = load_library(False)
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    out = {}
    for ni in (0, 4, 8, 12, 16):
        flops, best = C.c_ulonglong(0), 0.0
        for r in range(reps + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            _check(L.srhd_issue_probe(sink.data_ptr(), iters, ni, C.byref(flops), _stream()), L)
            e1.record()
            e1.synchronize()
            if r:
                best = max(best, flops.value / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        out[ni] = best
    return out


if __name__ == "__main__":
    import sys
    if sys.argv[1:] == ["issue_probe"]:
        t = issue_probe()
        print("| FFMA per 8 DFMA | DFMA TFLOP/s | relative to 0 | 16/(16+NI) |\n|---|---|---|---|")
        for ni, v in t.items():
            print(f"| {ni} | {v:.2f} | {v / t[0]:.3f} | {16 / (16 + ni):.3f} |")
