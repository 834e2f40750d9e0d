"""Pins of the oracle's refinement criteria (section 3.1; Eq. 33) against closed forms:
a linear profile has a known normalised gradient, |M|/D = h |U| (Eq. 5b), and a flag belongs to the
patch that holds the cell."""
import numpy as np
import pytest


def tiles_from_prim(ref, prim):
    """(5, nxt, nxt, nxt) primitives -> (1, 5, nxt, nxt, nxt) conserved tile."""
    return ref.prim2cons(prim.reshape(5, -1)).reshape((1,) + prim.shape)


@pytest.mark.parametrize("ghost,recon", [(2, "plm"), (3, "ppm")])
def test_eq33_on_a_linear_density_profile(ref, ghost, recon):
    par = ref.params(recon, "hllc")
    nxt = 16 + 2 * ghost
    x = np.arange(nxt) - ghost                       # interior cells 0..15
    prim = np.zeros((5, nxt, nxt, nxt))
    b = 0.05
    prim[0] = (1.0 + b * x)[None, None, :]           # rho = 1 + b i  -> Eq. 33 value = b / rho_i exactly
    prim[4] = 1e-3
    t = tiles_from_prim(ref, prim)
    val = b / (1.0 + b * np.arange(16))              # decreasing: 0.05 at i = 0 ... 0.0286 at i = 15
    for c_q in (0.0499, 0.04, 0.0355, 0.03, 0.0285):
        want_cells = val > c_q
        want = np.zeros(8, dtype=np.uint8)
        for p in range(8):
            want[p] = want_cells[8 * (p & 1):8 * (p & 1) + 8].any()
        got = ref.refine_flags(t, par, "rho", c_q)[0]
        assert np.array_equal(got, want), (c_q, got, want)
    # conserved quantity D = rho (gas at rest): identical flags without any root finding
    assert np.array_equal(ref.refine_flags(t, par, "D", 0.0355), ref.refine_flags(t, par, "rho", 0.0355))
    # the gradient along y and z is found in the same way (axis permutation of the tile)
    ty = tiles_from_prim(ref, prim.transpose(0, 1, 3, 2))
    fy = ref.refine_flags(ty, par, "rho", 0.0364)[0]      # cells 0..7 exceed it, cell 8 (0.0357) does not
    assert list(fy) == [1, 1, 0, 0, 1, 1, 0, 0]       # low-y patches (p & 2 == 0) hold the steep cells
    tz = tiles_from_prim(ref, prim.transpose(0, 3, 2, 1))
    assert list(ref.refine_flags(tz, par, "rho", 0.0364)[0]) == [1, 1, 1, 1, 0, 0, 0, 0]


def test_lorentz_factor_gradient_and_momentum_threshold(ref):
    par = ref.params("plm", "hllc")
    nxt = 20
    prim = np.zeros((5, nxt, nxt, nxt))
    prim[0], prim[4] = 1.0, 0.5                      # T = 0.5: h = 1 + 2.5 T + 2.25T^2/(1+sqrt(2.25T^2+1))
    U = np.zeros(nxt)
    U[2 + 11:] = 3.0                                  # a shear front between interior cells 10 and 11
    prim[3] = U[None, None, :]                        # U^z varies along x
    t = tiles_from_prim(ref, prim)
    # gamma jumps from 1 to sqrt(10) between i = 10 and 11: Eq. 33 = (sqrt(10)-1)/2 at i = 10, /(2 sqrt(10)) at 11
    g = np.sqrt(10.0)
    assert list(ref.refine_flags(t, par, "gamma", 0.9 * (g - 1) / (2 * g))[0]) == [0, 1] * 4
    assert list(ref.refine_flags(t, par, "gamma", 1.01 * (g - 1) / 2)[0]) == [0] * 8
    # |M|/D = h |U| (Eq. 5b): flagged where U = 3 (x-high patches) iff the threshold is below 3 h
    T = 0.5
    h = 2.5 * T + np.sqrt(2.25 * T * T + 1.0)        # Eq. 10
    assert list(ref.refine_flags(t, par, "none", 0.0, mom_over_d=3 * h * (1 - 1e-12))[0]) == [0, 1] * 4
    assert list(ref.refine_flags(t, par, "none", 0.0, mom_over_d=3 * h * (1 + 1e-12))[0]) == [0] * 8
    # both criteria are inclusive ("two inclusive refinement criteria")
    prim2 = prim.copy()
    prim2[0, :, 2 + 3, 2 + 2] = 5.0                   # one dense cell in the patch with low x, low y
    t2 = tiles_from_prim(ref, prim2)
    f = ref.refine_flags(t2, par, "rho", 0.3, mom_over_d=3 * h * (1 - 1e-12))[0]
    assert list(f) == [1, 1, 0, 1, 1, 1, 0, 1]
