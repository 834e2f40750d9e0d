"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It holds none of
the method's arithmetic: it only produces PRIMITIVE fields (rho, U^x, U^y, U^z, p) with
four-velocities, boundary-condition descriptors and masks, as numpy arrays.  Converting them to
conserved variables is the job of srhd_prim2cons (either implementation).  numpy only; importing
it never loads the CUDA extension or the oracle.

Array convention: fields are (5, nz, ny, nx), x fastest; state lists are (5, n).
"""
import numpy as np

PERIODIC, OUTFLOW = 0, 1


# ------------------------------------------------------------------ counter-based uniform numbers
def splitmix64(seed, n, stream=0):
    """n uint64 values of the splitmix64 sequence started at seed + stream*2^32 (vectorised)."""
    with np.errstate(over="ignore"):
        idx = np.arange(1, n + 1, dtype=np.uint64)
        z = (np.uint64(seed) + np.uint64(stream) * np.uint64(1 << 32)) + idx * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def uniform01(seed, n, stream=0):
    """Uniform doubles in (0,1) from the top 53 bits of splitmix64."""
    return ((splitmix64(seed, n, stream) >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def _gauss(seed, n, stream):
    u1, u2 = uniform01(seed, n, stream), uniform01(seed, n, stream + 1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# ------------------------------------------------------------------ config 2: conversion stress
def conversion_states(n=1 << 24, seed=201211130, log_rho=(-6.0, 6.0), log_theta=(-10.0, 6.0),
                      log_gamma=(0.0, 6.0)):
    """(5, n) primitive states: rho, Theta=p/rho and Lorentz factor log-uniform, direction isotropic.

    BASELINE.json configs[1] / PAPER.md App. B: |U| = sqrt((gamma-1)(gamma+1)).
    """
    rho = 10.0 ** (log_rho[0] + (log_rho[1] - log_rho[0]) * uniform01(seed, n, 0))
    theta = 10.0 ** (log_theta[0] + (log_theta[1] - log_theta[0]) * uniform01(seed, n, 1))
    gamma = 10.0 ** (log_gamma[0] + (log_gamma[1] - log_gamma[0]) * uniform01(seed, n, 2))
    g = np.stack([_gauss(seed, n, 3), _gauss(seed, n, 5), _gauss(seed, n, 7)])
    g /= np.sqrt((g * g).sum(0))
    umag = np.sqrt((gamma - 1.0) * (gamma + 1.0))
    out = np.empty((5, n))
    out[0] = rho
    out[1:4] = g * umag
    out[4] = rho * theta
    return out


def mach_sweep_states(theta=1e-8, n=101, log_mach=(-4.0, 6.0)):
    """PAPER.md App. B / Fig. 16 protocol: fixed Theta, U parallel to (1,1,1).

    Returns (prim (5,n), |U| (n,)): the caller turns a Mach number into |U| = Mach * U_s itself,
    so this generator only provides the unit direction and a log-spaced multiplier grid.
    """
    mult = 10.0 ** np.linspace(log_mach[0], log_mach[1], n)
    out = np.empty((5, n))
    out[0] = 1.0
    out[1:4] = 1.0 / np.sqrt(3.0)
    out[4] = theta
    return out, mult


# ------------------------------------------------------------------ config 1: 1-D TM shock tube
def shock_tube(n_long=256, n_trans=16, left=(1.0, 0.0, 1e3), right=(1.0, 0.0, 1e-6),
               x_diaphragm=0.5, axis=0, length=1.0):
    """BASELINE.json configs[0]: (rho, U, p) left/right of the diaphragm on [0,length]; uniform and
    periodic in the two transverse axes, outflow along the tube.

    n_trans = 16 (two periodic images of the 8-cell extent each way) so that the grid is a whole
    number of 16^3 patch groups.  axis = 0/1/2 puts the tube along x/y/z
    (used by the axis-permutation tests).  Returns (prim, dh, bc).
    """
    dh = length / n_long
    xc = (np.arange(n_long) + 0.5) * dh
    is_left = xc < x_diaphragm
    shape = [n_trans, n_trans, n_trans]          # (nz, ny, nx)
    shape[2 - axis] = n_long
    bshape = [1, 1, 1]
    bshape[2 - axis] = n_long
    prim = np.zeros([5] + shape)
    prim[0] = np.where(is_left, left[0], right[0]).reshape(bshape)
    prim[1 + axis] = np.where(is_left, left[1], right[1]).reshape(bshape)
    prim[4] = np.where(is_left, left[2], right[2]).reshape(bshape)
    bc = [PERIODIC] * 6
    bc[2 * axis] = bc[2 * axis + 1] = OUTFLOW
    return prim, dh, bc


# ------------------------------------------------------------------ config 3: spherical blast
def blast_wave(n=256, r_src=0.1, p_src=1e3, p_amb=1e-6, rho=1.0):
    """BASELINE.json configs[2]: unit box, periodic; rho=1, U=0; p = p_src for r<r_src else p_amb."""
    dh = 1.0 / n
    x = (np.arange(n) + 0.5) * dh - 0.5
    r2 = x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2
    prim = np.zeros((5, n, n, n))
    prim[0] = rho
    prim[4] = np.where(r2 < r_src * r_src, p_src, p_amb)
    return prim, dh, [PERIODIC] * 6


# ------------------------------------------------------------------ config 4: random field
def _grf(rng, n, dtype=np.float64):
    """Real Gaussian random field on n^3 with P(k) ~ k^-2 (amplitude ~ 1/k), zero mean, unit std."""
    white = rng.standard_normal((n, n, n)).astype(dtype)
    fk = np.fft.rfftn(white)
    del white
    k1 = np.fft.fftfreq(n) * n
    kr = np.fft.rfftfreq(n) * n
    k2 = k1[:, None, None] ** 2 + k1[None, :, None] ** 2 + kr[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    fk /= np.sqrt(k2)
    fk[0, 0, 0] = 0.0
    f = np.fft.irfftn(fk, s=(n, n, n), axes=(0, 1, 2))
    f -= f.mean()
    f /= f.std()
    return f


def _affine(f, lo, hi):
    a, b = f.min(), f.max()
    return lo + (f - a) * ((hi - lo) / (b - a))


def random_field(n=512, seed=2012, log_theta=(-8.0, 4.0), log_rho=(-3.0, 3.0), gamma_max=1e3):
    """BASELINE.json configs[3]: log10 rho, log10 Theta and U^i as k^-2 Gaussian random fields.

    log10 Theta spans log_theta exactly (affine map of the field's min/max); log10 rho spans
    log_rho (range is our choice); the three U fields share one scale factor chosen so
    that the largest Lorentz factor is gamma_max.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    dh = 1.0 / n
    prim = np.empty((5, n, n, n))
    lr = _affine(_grf(rng, n), *log_rho)
    lt = _affine(_grf(rng, n), *log_theta)
    prim[0] = 10.0 ** lr
    prim[4] = prim[0] * 10.0 ** lt
    for d in range(3):
        prim[1 + d] = _grf(rng, n)
    u2max = (prim[1:4] ** 2).sum(0).max()
    prim[1:4] *= np.sqrt((gamma_max - 1.0) * (gamma_max + 1.0) / u2max)
    return prim, dh, [PERIODIC] * 6


# ------------------------------------------------------------------ config 5: relativistic jet
def jet(nx=512, ny=512, nz=1024, radius=0.02, rho_jet=1e-2, theta_jet=10.0, gamma_jet=1e3,
        rho_amb=1.0, theta_amb=1e-6):
    """BASELINE.json configs[4]: domain 1 x 1 x 2 (dh = 1/nx), outflow; ambient at rest; fixed inflow.

    Returns (prim, dh, bc, (mask, prim_jet)): mask (ny,nx) uint8 marks the columns whose centre lies
    inside the nozzle circle of the z=0 face; ghost cells below those columns hold prim_jet.
    """
    dh = 1.0 / nx
    prim = np.zeros((5, nz, ny, nx))
    prim[0] = rho_amb
    prim[4] = rho_amb * theta_amb
    x = (np.arange(nx) + 0.5) * dh - 0.5
    y = (np.arange(ny) + 0.5) * dh - 0.5 * ny * dh
    mask = ((x[None, :] ** 2 + y[:, None] ** 2) < radius * radius).astype(np.uint8)
    prim_jet = np.array([rho_jet, 0.0, 0.0, np.sqrt((gamma_jet - 1.0) * (gamma_jet + 1.0)), rho_jet * theta_jet])
    return prim, dh, [OUTFLOW] * 6, (mask, prim_jet)


# ------------------------------------------------------------------ kernel-level parity inputs
def random_patch_groups(npg, ghost, seed=7, log_theta=(-6.0, 3.0), umax=3.0, rough=0.3):
    """(npg, 5, nxt, nxt, nxt) primitive tiles for one-step parity tests of srhd_fluid_step.

    Each tile is an independent smooth random field (a few low-order Fourier modes) plus a planar
    jump through the tile and `rough` relative white noise, so that limiter branches, shocks and
    smooth regions all occur.  log10 Theta and velocities vary from tile to tile.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    nxt = 16 + 2 * ghost
    c = (np.arange(nxt) - ghost + 0.5) / 16.0
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    out = np.empty((npg, 5, nxt, nxt, nxt))
    for pg in range(npg):
        def smooth():
            f = np.zeros_like(X)
            for _ in range(4):
                k = rng.integers(-2, 3, size=3)
                ph = rng.uniform(0, 2 * np.pi)
                f += rng.standard_normal() * np.cos(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + ph)
            return f / 2.0
        nrm = rng.standard_normal(3)
        nrm /= np.linalg.norm(nrm)
        side = ((X - 0.5) * nrm[0] + (Y - 0.5) * nrm[1] + (Z - 0.5) * nrm[2] + rng.uniform(-0.3, 0.3)) > 0
        lt0 = rng.uniform(*log_theta)
        jump = rng.uniform(0.0, 2.0) * (rng.random() < 0.7)
        log_rho = 0.5 * smooth() + jump * side + rough * rng.standard_normal(X.shape) * 0.1
        log_th = lt0 + 0.5 * smooth() + jump * side * rng.uniform(-1, 1)
        log_th = np.clip(log_th, log_theta[0] - 1, log_theta[1] + 1)
        us = umax * 10.0 ** rng.uniform(-3, 0)
        out[pg, 0] = 10.0 ** log_rho
        for d in range(3):
            out[pg, 1 + d] = us * (smooth() + rough * 0.1 * rng.standard_normal(X.shape)) + us * rng.standard_normal()
        out[pg, 4] = out[pg, 0] * 10.0 ** log_th
    return out
