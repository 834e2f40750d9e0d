"""-m gpu parity of the coarse-fine hooks (csrc/srhd_amr.cu) with the oracle's."""
import numpy as np
import pytest
import torch

from paper_2012_11130_b200 import binding as B
from paper_2012_11130_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return (t if dtype is None else t.to(dtype)).cuda()


def test_flux_correction_parity_and_skip_rule(ref):
    rng = np.random.default_rng(2)
    prim = wl.random_patch_groups(2, 0, seed=31, rough=0.2)            # (2,5,16,16,16)
    cons = ref.prim2cons(prim.transpose(1, 0, 2, 3, 4).reshape(5, -1)).reshape(5, 2, 16, 16, 16).transpose(1, 0, 2, 3, 4)
    patches = np.ascontiguousarray(cons.reshape(2, 5, 2, 8, 2, 8, 2, 8).transpose(0, 2, 4, 6, 1, 3, 5, 7).reshape(16, 5, 8, 8, 8))
    faces = [(p, f) for p in range(16) for f in range(6) if rng.random() < 0.4]
    nf = len(faces)
    fc = rng.standard_normal((nf, 5, 8, 8)) * np.abs(patches).mean((0, 2, 3, 4))[None, :, None, None]
    ff = fc * (1 + 0.01 * rng.standard_normal(fc.shape))
    ff[::3, 4] += 50.0 * np.abs(patches[:, 4]).mean()                   # every third face: a draining energy flux
    fp, fi = [p for p, _ in faces], [f for _, f in faces]
    want, skipped = ref.flux_correction(patches, fc, ff, fp, fi, 0.3, 1.0)
    assert 0 < skipped < nf * 64
    for exact in (True, False):
        d = dev(patches)
        n = B.flux_correction(d, dev(fc), dev(ff), dev(np.array(fp), torch.int32), dev(np.array(fi), torch.int32), 0.3, 1.0,
                              exact=exact)
        assert int(n.cpu()) == skipped
        g = d.cpu().numpy()
        if exact:
            assert np.array_equal(g, want)
        else:                                                           # the production build contracts U - dtdh*dF into an fma
            assert (np.abs(g - want) <= 4e-16 * (np.abs(want) + 0.3 * np.abs(ff - fc).max())).all()


def test_ghost_interp_parity_with_fallback(ref):
    n = 12
    z, y, x = np.meshgrid(np.arange(n), np.arange(n + 1), np.arange(n + 3), indexing="ij")
    prim = np.zeros((5,) + x.shape)
    prim[0] = 10.0 ** (-0.4 * x + 0.15 * y)
    prim[1] = 10.0 ** (1.5 - 0.15 * x + 0.05 * z)
    prim[2] = 10.0 ** (0.5 + 0.15 * y - 0.1 * z)
    prim[3] = 0.3 * z
    prim[4] = prim[0] * np.where(z < 6, 1.0, 1e-8)
    prim[1:4] *= np.where(z < 6, 0.02, 1.0)
    coarse = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    par = ref.params()
    want, wfb, wn = ref.ghost_interp(coarse, 1.5, par)
    assert 0 < wn < wfb.size
    for exact in (True, False):
        fine, fb, cnt = B.ghost_interp(dev(coarse), 1.5, B.params(exact=exact), exact=exact)
        assert int(cnt.cpu()) == wn and np.array_equal(fb.cpu().numpy(), wfb)
        g = fine.cpu().numpy()
        if exact:
            assert np.array_equal(g, want)
        else:
            scale = np.abs(want).reshape(5, -1).max(1)
            scale[1:4] = scale[1:4].max()
            assert (np.abs(g - want) / scale[:, None, None, None]).max() <= 1e-13


def test_ghost_interp_copies_the_parent_at_a_steep_corner(ref):
    """Reading S22: where the primitive fallback would give a child rho <= 0 (density 0.01 / 1 / 3.97 along all three
    axes, beta = 1.5) the CUDA kernel, like the oracle, copies the parent and flags the cell 2; a grid holding such
    corners next to ordinary cold gradients reproduces the oracle's flags and children."""
    n = 9
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    prim = np.zeros((5, n, n, n))
    prim[0] = 1.0
    for c in ((1, 1, 1), (4, 4, 4), (7, 4, 1)):          # corners: the six neighbours of c at 0.01 (low) / 3.97 (high)
        for ax in range(3):
            lo, hi = list(c), list(c)
            lo[ax] -= 1
            hi[ax] += 1
            prim[0][tuple(lo)], prim[0][tuple(hi)] = 0.01, 3.97
    prim[4] = 1e-8 * prim[0]
    prim[1] = 5.0 + 0.1 * x
    coarse = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    par = ref.params()
    want, wfb, wn = ref.ghost_interp(coarse, 1.5, par)
    assert (wfb == 2).sum() >= 3 and (wfb == 1).sum() > 0
    for exact in (True, False):
        fine, fb, cnt = B.ghost_interp(dev(coarse), 1.5, B.params(exact=exact), exact=exact)
        assert int(cnt.cpu()) == wn and np.array_equal(fb.cpu().numpy(), wfb)
        g = fine.cpu().numpy()
        copied = np.repeat(np.repeat(np.repeat(wfb == 2, 2, 0), 2, 1), 2, 2)
        assert np.array_equal(g[:, copied], want[:, copied])            # copies of the parent: exact in every build
        if exact:
            assert np.array_equal(g, want)
        else:
            scale = np.abs(want).reshape(5, -1).max(1)
            scale[1:4] = scale[1:4].max()
            assert (np.abs(g - want) / scale[:, None, None, None]).max() <= 1e-13
