"""Pins of the oracle's coarse-fine hooks: the flux correction with its "skip if
unphysical" rule (section 3.3(4)) and the ghost-zone interpolation with the primitive-variable fallback
(section 3.3(3)) -- against conservation, the divergence theorem, linear data, and constructed cases."""
import numpy as np
import pytest

from paper_2012_11130_b200 import workloads as wl

EPS = np.finfo(np.float64).eps


def _tiles(ref, npg, ghost, seed, **kw):
    prim = wl.random_patch_groups(npg, ghost, seed=seed, **kw)
    nxt = 16 + 2 * ghost
    cons = ref.prim2cons(prim.transpose(1, 0, 2, 3, 4).reshape(5, -1))
    return np.ascontiguousarray(cons.reshape(5, npg, nxt, nxt, nxt).transpose(1, 0, 2, 3, 4))


def test_flux_correction_restores_the_fine_flux_in_the_budget(ref):
    """Update a patch with coarse fluxes, then correct its x-hi and z-lo faces with other ("fine") fluxes: the
    patch content must change by exactly -+ dt/dh times the summed flux difference (divergence theorem), the
    cells away from those faces must not change, and nothing is skipped on benign data."""
    par = ref.params("plm", "hllc")
    tiles = _tiles(ref, 1, par.ghost, seed=13, rough=0.0)
    dh = 1.0 / 64
    dt = 0.4 * dh / ref.max_signal_speed(tiles.transpose(1, 0, 2, 3, 4).reshape(5, -1))
    out, flux, st = ref.fluid_step_fluxes(tiles, dt, dh, par)
    patches = out[0]                                          # (8,5,8,8,8)
    rng = np.random.default_rng(1)
    faces = [(0, 1), (0, 4), (5, 0), (7, 3)]
    fc = np.stack([flux[0, p, f] for p, f in faces])
    ff = fc * (1.0 + 1e-3 * rng.standard_normal(fc.shape))    # "fine" fluxes: a little off
    got, skipped = ref.flux_correction(patches, fc, ff, [p for p, _ in faces], [f for _, f in faces], dt, dh)
    assert skipped == 0
    for p in range(8):
        d_content = (got[p] - patches[p]).reshape(5, -1).sum(1)
        want = np.zeros(5)
        for n, (fp, fid) in enumerate(faces):
            if fp == p:
                sgn = -1.0 if fid & 1 else 1.0
                want += sgn * dt / dh * (ff[n] - fc[n]).reshape(5, -1).sum(1)
        scale = np.abs(patches[p]).reshape(5, -1).sum(1)
        assert np.all(np.abs(d_content - want) <= 64 * EPS * scale)
    untouched = got[0][:, 1:, :, :7] == patches[0][:, 1:, :, :7]       # patch 0: only x-hi (i = 7) and z-lo (k = 0) change
    assert untouched.all()
    assert not np.array_equal(got[0][:, :, :, 7], patches[0][:, :, :, 7])


def test_flux_correction_is_skipped_where_it_would_break_eq30(ref):
    """"If unphysical results are found after this flux correction, we simply ignore the correction on the
    failed cells."  A fine energy flux that would drain more than the cell holds must leave those cells as they were."""
    W = np.array([1.0, 0.1, 0.0, 0.0, 1e-3])
    U = ref.prim2cons(W.reshape(5, 1))[:, 0]
    patches = np.broadcast_to(U[None, :, None, None, None], (2, 5, 8, 8, 8)).copy()
    fc = np.zeros((2, 5, 8, 8))
    ff = np.zeros((2, 5, 8, 8))
    ff[0, 4, :4, :] = 10.0 * U[4]                 # half of face 0: removes 10x the cell's Etilde -> unphysical
    ff[0, 4, 4:, :] = 0.1 * U[4]                  # other half: benign
    ff[1, 0] = 0.05 * U[0]
    got, skipped = ref.flux_correction(patches, fc, ff, [0, 1], [1, 2], 1.0, 1.0)
    assert skipped == 32
    assert np.array_equal(got[0][:, :4, :, 7], patches[0][:, :4, :, 7])          # skipped cells untouched (a = z)
    assert np.allclose(got[0][4, 4:, :, 7], 0.9 * U[4], rtol=1e-15)
    assert np.allclose(got[1][0, :, 0, :], 1.05 * U[0], rtol=1e-15)              # y-lo face: flux enters
    x = got[:, 4] / got[:, 0]
    L = x * (x + 2) - ((got[:, 1:4] / got[:, 0:1]) ** 2).sum(1)
    assert (L > EPS).all() and (got[:, 0] > 0).all() and (got[:, 4] > 0).all()


def test_ghost_interpolation_is_conservative_linear_exact_and_bounded(ref):
    rng = np.random.default_rng(5)
    par = ref.params()
    prim = wl.random_patch_groups(1, 0, seed=9, rough=0.1)[0][:, :10, :9, :8]    # (5,10,9,8) smooth + noise
    coarse = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    fine, fb, n = ref.ghost_interp(coarse, 1.5, par)
    assert n == 0 and fine.shape == (5, 16, 14, 12)
    kids = fine.reshape(5, 8, 2, 7, 2, 6, 2).transpose(0, 1, 3, 5, 2, 4, 6).reshape(5, 8, 7, 6, 8)
    parent = coarse[:, 1:-1, 1:-1, 1:-1]
    lo = np.minimum.reduce([coarse[:, 1:-1, 1:-1, 1:-1], coarse[:, :-2, 1:-1, 1:-1], coarse[:, 2:, 1:-1, 1:-1],
                            coarse[:, 1:-1, :-2, 1:-1], coarse[:, 1:-1, 2:, 1:-1], coarse[:, 1:-1, 1:-1, :-2],
                            coarse[:, 1:-1, 1:-1, 2:]])
    hi = np.maximum.reduce([coarse[:, 1:-1, 1:-1, 1:-1], coarse[:, :-2, 1:-1, 1:-1], coarse[:, 2:, 1:-1, 1:-1],
                            coarse[:, 1:-1, :-2, 1:-1], coarse[:, 1:-1, 2:, 1:-1], coarse[:, 1:-1, 1:-1, :-2],
                            coarse[:, 1:-1, 1:-1, 2:]])
    span = hi - lo
    assert np.all(np.abs(kids.mean(-1) - parent) <= 16 * EPS * (np.abs(parent) + span))    # conservative
    assert np.all(kids >= (lo - 1.5 * span)[..., None]) and np.all(kids <= (hi + 1.5 * span)[..., None])
    # linear data are reproduced exactly: child = parent -+ slope/4 per axis
    z, y, x = np.meshgrid(np.arange(6.0), np.arange(5.0), np.arange(7.0), indexing="ij")
    lin = np.stack([30 + x + 2 * y - 3 * z, 0.1 * x, 0.2 * y, -0.1 * z, 50 + x + y + z])
    fine, fb, n = ref.ghost_interp(lin, 2.0, par)
    zf, yf, xf = np.meshgrid((np.arange(8) - 0.5) / 2 + 1, (np.arange(6) - 0.5) / 2 + 1, (np.arange(10) - 0.5) / 2 + 1,
                             indexing="ij")
    want = np.stack([30 + xf + 2 * yf - 3 * zf, 0.1 * xf, 0.2 * yf, -0.1 * zf, 50 + xf + yf + zf])
    assert n == 0 and np.allclose(fine, want, rtol=1e-14, atol=1e-14)
    # a vanished coefficient copies the parent ("directly copying data from the parent patch")
    fine, fb, n = ref.ghost_interp(coarse, 0.0, par)
    assert np.array_equal(fine.reshape(5, 8, 2, 7, 2, 6, 2)[:, :, 0, :, 0, :, 0], parent)
    assert rng is not None


def test_ghost_interpolation_falls_back_to_primitives(ref):
    """"if unphysical results occur, we interpolate primitive variables instead ... Eq. 30 is always
    satisfied".  Cold gas sits ON the boundary of Eq. 30 (L = O(T)), so limiting the slopes of D, M and Etilde
    independently pushes some child off it; the fallback children are all physical.  Hot gas needs no fallback."""
    par = ref.params()
    n = 6
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    prim = np.zeros((5, n, n, n))
    prim[0] = 10.0 ** (-0.8 * x + 0.3 * y)                    # smooth exponential gradients in rho and U:
    prim[1] = 10.0 ** (1.5 - 0.3 * x + 0.1 * z)               # Lorentz factor ~ 30 down to ~ 1
    prim[2] = 10.0 ** (0.5 + 0.3 * y)
    prim[3] = 0.3 * z
    prim[4] = prim[0] * np.where(z < 3, 1.0, 1e-8)            # hot lower half, cold upper half
    prim[1:4] *= np.where(z < 3, 0.02, 1.0)                   # ... which is also slow
    coarse = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    fine, fb, nfb = ref.ghost_interp(coarse, 1.5, par)
    assert nfb > 0 and fb.sum() == nfb and fb.max() == 1          # no cell needed the parent copy (S22)
    F = fine.reshape(5, -1)
    _, _, _, bad = ref.cons2prim(F, par, diag=True)
    assert bad.sum() == 0                                           # every child passes Eq. 30
    # where no fallback happened the children still average to the parent
    kids = fine.reshape(5, 4, 2, 4, 2, 4, 2).transpose(0, 1, 3, 5, 2, 4, 6).reshape(5, 4, 4, 4, 8)
    parent = coarse[:, 1:-1, 1:-1, 1:-1]
    ok = fb == 0
    assert ok.any() and np.all(np.abs(kids.mean(-1) - parent)[:, ok] <= 16 * EPS * np.abs(parent).max())
    # fallback children: the interpolated PRIMITIVES lie between the neighbouring coarse primitives
    Wf = ref.cons2prim(F, par)[0].reshape(fine.shape)
    assert Wf[0].min() >= prim[0].min() * (1 - 1e-9) and Wf[0].max() <= prim[0].max() * (1 + 1e-9)
    assert fb[:1].sum() == 0 and fb[3:].all()                   # hot planes: conserved interpolation; cold planes: fallback


def test_ghost_interpolation_copies_the_parent_at_a_steep_3d_corner(ref):
    """Reading S22: with density 0.01 / 1 / 3.97 along ALL three axes and beta = 1.5 each quarter-slope
    is 1.5 * 0.99 / 4 = 0.371, so the child at the low corner would get rho = 1 - 3 * 0.371 < 0 from the primitive
    interpolation: "Eq. 30 is always satisfied" does not cover it.  Such a cell's children are copies of the
    parent (vanished coefficient = copy from the parent patch) and its flag is 2; every child passes Eq. 30
    and the children trivially average to the parent."""
    par = ref.params()
    prof = np.array([0.01, 1.0, 3.97])
    z, y, x = np.meshgrid(np.arange(3), np.arange(3), np.arange(3), indexing="ij")
    prim = np.zeros((5, 3, 3, 3))
    # separable would give 0.01^3 at the corner; the recipe wants the centre cell's SIX neighbours at 0.01 / 3.97
    prim[0] = 1.0
    for ax, idx in ((2, x), (1, y), (0, z)):
        prim[0] = np.where((idx != 1) & ((x == 1).astype(int) + (y == 1).astype(int) + (z == 1).astype(int) == 2),
                           prof[idx], prim[0])
    assert prim[0][1, 1, 0] == 0.01 and prim[0][1, 1, 2] == 3.97 and prim[0][0, 1, 1] == 0.01 and prim[0][1, 1, 1] == 1.0
    prim[4] = 1e-8 * prim[0]                          # cold: the conserved interpolation fails Eq. 30 first
    prim[1] = 5.0                                     # moving, so that L sits on the boundary of Eq. 30 (L = O(T))
    coarse = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    # the arithmetic of the premise, from the limiter's definition (S3): min(2|ab|/|a+b|, beta min(|a|,|b|)) / 4
    a, b = 1.0 - 0.01, 3.97 - 1.0
    q = min(2 * a * b / (a + b), 1.5 * min(a, b)) / 4
    assert 1.0 - 3 * q < 0.0
    fine, fb, nfb = ref.ghost_interp(coarse, 1.5, par)
    assert fb.shape == (1, 1, 1) and fb[0, 0, 0] == 2 and nfb == 1
    kids = fine.reshape(5, 8)
    assert np.array_equal(kids, np.repeat(coarse[:, 1, 1, 1][:, None], 8, axis=1))
    assert ref.is_physical(kids).all()
    # a milder corner (slopes sum to less than the cell value) keeps the primitive interpolation: flag 1
    prim2 = prim.copy()
    prim2[0] = np.where(prim[0] == 0.01, 0.5, prim[0])
    prim2[4] = 1e-8 * prim2[0]
    c2 = ref.prim2cons(prim2.reshape(5, -1)).reshape(prim2.shape)
    f2, fb2, n2 = ref.ghost_interp(c2, 1.5, par)
    assert fb2[0, 0, 0] in (0, 1)
    W = ref.cons2prim(f2.reshape(5, 8), par)[0]
    assert W[0].min() > 0 and W[4].min() > 0
