"""Pins of what decides WHICH states count as unphysical in the oracle ("What's weak" #1): the
arithmetic of the conversions and of the step was pinned in rounds 1-2, but seven one-line mutants of the verdict
logic survived every test.  These tests kill them (tests/mutants.py lists them) with states constructed so that the
left-hand side of Eq. 30 is known EXACTLY (powers of two; checked below in rational arithmetic), with the S10 /
S15 / S18 readings of DESIGN.md section 4, and with hand-written 1-D index tables for the boundary map (S11).

P:267 Eq. 30:  (Etilde/D)^2 + 2 (Etilde/D) - (|M|/D)^2 > eps_machine,  eps_machine = 2^-52 for double.
"""
from fractions import Fraction

import numpy as np
import pytest

from tests import py_step
from tests.test_oracle_pins_r2 import _rough_box

EPS = 2.0 ** -52
DBL_MIN = 2.2250738585072014e-308     # smallest positive normal double (reading S10: the vacuum floor)


def _lhs_exact(D, M, E):
    """Left-hand side of Eq. 30 in exact rational arithmetic (every double is a rational)."""
    x = Fraction(E) / Fraction(D)
    return x * x + 2 * x - sum((Fraction(m) / Fraction(D)) ** 2 for m in M)


def _threshold_states():
    """(D, M, Etilde, L / eps) with L known exactly, on both sides of eps_machine and away from rounding ties."""
    out = []
    for scale in (1.0, 2.0 ** -20, 2.0 ** 30):                  # D scales out of Eq. 30: powers of two keep it exact
        for c in (0.5, 0.75, 1.5, 2.0):
            # at rest: L = 2x + x^2 with x = c eps / 2 -> L = c eps (1 + c eps / 4)
            out.append((scale, (0.0, 0.0, 0.0), scale * c * EPS / 2, c))
            # moving: |M|/D = 2^-30, x = 2^-61 + c eps / 2 -> L = c eps + x^2, x^2 ~ 2^-122: the momentum term must
            # be subtracted (without it L ~ 2^-60 << eps for every c; with the wrong sign the same)
            out.append((scale, (0.0, scale * 2.0 ** -30, 0.0), scale * (2.0 ** -61 + c * EPS / 2), c))
    return out


def test_eq30_threshold_is_eps_machine_strictly(ref):
    """Eq. 30 "> eps_machine" on updated cells (is_physical, O9) and in the verdict of cons->prim (O3):
    L = 0.5 eps and 0.75 eps fail, 1.5 eps and 2 eps pass -- a threshold of 0 or of 2 eps fails this."""
    states = _threshold_states()
    for D, M, E, c in states:                                    # the construction itself, in exact arithmetic
        L = _lhs_exact(D, M, E)
        assert abs(L / Fraction(EPS) - Fraction(c)) < Fraction(1, 10 ** 9)
    cons = np.array([[D, M[0], M[1], M[2], E] for D, M, E, _ in states]).T.copy()
    want = np.array([c > 1.0 for *_, c in states])
    assert np.array_equal(ref.is_physical(cons), want)
    _, _, _, bad = ref.cons2prim(cons, diag=True)
    assert np.array_equal(bad == 0, want)
    assert ref.cons2prim(cons)[1].n_c2p_fail == int((~want).sum())


def test_negative_reduced_energy_or_density_is_unphysical_whatever_L(ref):
    """physical iff D > 0 AND Etilde > 0 AND L > eps.  The left-hand side of Eq. 30 is even in
    the sign of D and is large for Etilde < -2 D, so the two sign conditions are separate requirements ("negative
    pressure, negative density"): each state below has L = 3 exactly and must still be rejected."""
    cons = np.array([[1.0, 0.0, 0.0, 0.0, -3.0],       # Etilde < 0, x = -3: L = 9 - 6 = 3
                     [-1.0, 0.0, 0.0, 0.0, -1.0],      # D < 0, x = 1: L = 3
                     [2.0, 0.0, 0.0, 0.0, -6.0],
                     [-1.0, 0.0, 0.0, 0.0, 3.0],       # D < 0 alone (Etilde > 0), x = -3: L = 3
                     [1.0, 0.0, 0.0, 0.0, 1.0]]).T.copy()   # the physical twin: x = 1, L = 3
    for k in range(5):
        assert _lhs_exact(cons[0, k], cons[1:4, k], cons[4, k]) == 3
    want = np.array([False, False, False, False, True])
    assert np.array_equal(ref.is_physical(cons), want)
    prim, ht, it, bad = ref.cons2prim(cons, diag=True)
    assert np.array_equal(bad == 0, want)
    assert np.all(np.isfinite(prim))                    # S10: a rejected state is still evaluated deterministically
    assert ref.cons2prim(cons)[1].n_c2p_fail == 4


def test_vacuum_floor_of_reading_s10(ref):
    """Reading S10: a state whose D is not above the smallest normal number is evaluated as vacuum at rest
    (D <- DBL_MIN, M <- 0, Etilde <- 0, L <- eps) and counted; D = 2 DBL_MIN is an ordinary state.  With a momentum
    in the input the two branches differ in U, which is what tells them apart."""
    M = 0.5 * DBL_MIN
    cons = np.array([[0.0, M, 0.0, 0.0, DBL_MIN],
                     [0.5 * DBL_MIN, M, 0.0, 0.0, DBL_MIN],          # subnormal, > 0
                     [DBL_MIN, M, 0.0, 0.0, DBL_MIN],                # the floor itself: still vacuum
                     [-1.0, M, 0.0, 0.0, DBL_MIN],
                     [2.0 * DBL_MIN, M, 0.0, 0.0, 2.0 * DBL_MIN]]).T.copy()
    prim, ht, it, bad = ref.cons2prim(cons, diag=True)
    assert list(bad) == [1, 1, 1, 1, 0]
    for k in range(4):                                               # vacuum at rest, bit for bit the same answer
        assert prim[0, k] == DBL_MIN and np.all(prim[1:4, k] == 0.0)
        assert 0.0 <= prim[4, k] <= DBL_MIN * EPS                    # p = rho T with T ~ eps / 3 (L = eps at rest)
        assert ht[k] == ht[0] and 0.8 * EPS < ht[k] < 0.9 * EPS      # htilde ~ 2.5 T = (5/6) eps
    # the ordinary state: x = 1, |M|/D = 1/4 -> moving, hot (Etilde = D), and physical
    assert prim[1, 4] > 0.0 and prim[0, 4] > 0.0 and prim[4, 4] > 0.0
    assert np.array_equal(ref.is_physical(cons), np.array([False, True, True, False, True]))
    # (is_physical is the plain Eq. 30 check of an updated cell: D > 0, Etilde > 0, L = 3 > eps for the tiny states)


def test_vl_counts_a_failing_predictor_state(ref):
    """S18 / S15: a half-step (predictor) state of the VL integrator that fails Eq. 30 is repaired by S10 and COUNTED
    in n_c2p_fail.  The Python re-assembly (tests/py_step.py) counts them independently; the case must have some."""
    found = 0
    for recon, seed, mult in (("plm", 4, 6.0), ("ppm", 4, 6.0), ("plm", 6, 8.0)):
        par = ref.params(recon, "hllc", max_retry=2, integrator="vl")
        cons = _rough_box(ref, seed, par.ghost, n=3)
        dh = 1.0 / 64
        dt = mult * 0.4 * dh / ref.max_signal_speed(cons.reshape(5, -1))
        out, passes, hf, cf, hist = py_step.ladder_vl(ref, cons, dt, dh, par)
        got, st, got_passes = ref.step_box(cons, dt, dh, par)
        assert (got_passes, st.n_c2p_fail, st.n_unphys_final) == (passes, hf, cf), (recon, seed)
        assert np.array_equal(got, out, equal_nan=True)
        found += hf
    assert found > 0, "no case has a failing predictor state: the count is not exercised"


# ---- S11: the boundary map of the uniform-grid harness, against tables written by hand -------------------------
# source index of ghost/interior position i = -g .. n+g-1 for n = 16
def _table(n, g, lo, hi):
    t = []
    for i in range(-g, n + g):
        if i < 0:
            t.append(n + i if lo == "periodic" else 0)          # wrap: -1 -> n-1, -2 -> n-2, ...; outflow: cell 0
        elif i >= n:
            t.append(i - n if hi == "periodic" else n - 1)      # wrap: n -> 0, n+1 -> 1, ...; outflow: cell n-1
        else:
            t.append(i)
    return t


HAND = {  # written out once by hand for g = 2 (n = 16) so that _table itself is pinned
    ("periodic", "periodic"): [14, 15] + list(range(16)) + [0, 1],
    ("outflow", "outflow"): [0, 0] + list(range(16)) + [15, 15],
    ("outflow", "periodic"): [0, 0] + list(range(16)) + [0, 1],
    ("periodic", "outflow"): [14, 15] + list(range(16)) + [15, 15],
}


@pytest.mark.parametrize("g", [2, 3, 4])
def test_boundary_map_against_hand_tables(ref, g):
    for key, row in HAND.items():
        assert _table(16, 2, *key) == row
    n = 16
    # a grid whose value encodes its own index per axis, so that a wrong source cell on any axis shows
    iz, iy, ix = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    grid = np.stack([(q + 1) * 1e6 + iz * 1e4 + iy * 1e2 + ix for q in range(5)]).astype(np.float64)
    for bc in (["periodic"] * 6, ["outflow"] * 6,
               ["outflow", "periodic", "periodic", "outflow", "outflow", "outflow"],
               ["periodic", "outflow", "outflow", "periodic", "periodic", "periodic"]):
        tx, ty, tz = _table(n, g, bc[0], bc[1]), _table(n, g, bc[2], bc[3]), _table(n, g, bc[4], bc[5])
        want = grid[:, tz][:, :, ty][:, :, :, tx]
        assert np.array_equal(ref.grid_pad(grid, g, bc), want), bc
        tiles = ref.grid_gather(grid, g, bc)                     # one patch group: the tile IS the padded grid
        assert tiles.shape[0] == 1 and np.array_equal(tiles[0], want), bc


# ---- the extended-precision variant of the oracle ("ext": the stand-in for the true update) --------------------
def test_extended_precision_variant_is_the_same_algorithm_evaluated_more_finely(ref):
    """oracle/build.py "ext" (long double, eps = 1.1e-19) is what tests/test_gpu_truth.py measures both the fp64 oracle
    and the CUDA build against.  Pinned here: (1) its prim->cons agrees with the 40-digit evaluation of the
    DEFINITIONS (tests/mp_defs.py) to 1e-17 where fp64 cannot do better than 1e-16; (2) the thresholds are the fp64
    algorithm's: Eq. 30 still switches at 2^-52 and the S10 floor at DBL_MIN; (3) one fluid step makes the same
    retry decisions as the fp64 oracle and differs from it by fp64 round-off only."""
    import mpmath as mp
    from paper_2012_11130_b200 import workloads as wl
    from tests import mp_defs
    from tests.gpu_util import step_err
    prim = wl.conversion_states(n=64, seed=9)
    with ref.variant("ext"):
        assert ref.rdtype() == np.longdouble and np.finfo(np.longdouble).eps < 2e-19
        cons = ref.prim2cons(prim.astype(np.longdouble))
    c64 = ref.prim2cons(prim)
    worst_ext = worst_64 = 0.0
    for k in range(prim.shape[1]):
        want = mp_defs.prim2cons([float(v) for v in prim[:, k]])
        for q in (0, 4):
            w = mp.mpf(want[q])
            worst_ext = max(worst_ext, float(abs(mp.mpf(str(np.format_float_scientific(cons[q, k], precision=25))) - w) / abs(w)))
            worst_64 = max(worst_64, float(abs(mp.mpf(float(c64[q, k])) - w) / abs(w)))
    assert worst_ext <= 2e-18 and worst_64 >= 5e-17, (worst_ext, worst_64)
    # (2) thresholds
    states = _threshold_states()
    cons = np.array([[D, M[0], M[1], M[2], E] for D, M, E, _ in states]).T.copy()
    want = np.array([c > 1.0 for *_, c in states])
    tiny = np.array([[0.5 * DBL_MIN, 0.5 * DBL_MIN, 0.0, 0.0, DBL_MIN]]).T.copy()
    with ref.variant("ext"):
        assert np.array_equal(ref.is_physical(cons.astype(np.longdouble)), want)
        prim_t, _, _, bad = ref.cons2prim(tiny.astype(np.longdouble), diag=True)
    assert bad[0] == 1 and prim_t[0, 0] == np.longdouble(DBL_MIN) and prim_t[1, 0] == 0
    # (3) one step on rough data with retries
    par = ref.params("plm", "hllc", max_retry=3)
    box = _rough_box(ref, 4, par.ghost)
    dh = 1.0 / 64
    dt = 0.4 * dh / ref.max_signal_speed(box.reshape(5, -1))
    o64, st64, p64 = ref.step_box(box, dt, dh, par)
    with ref.variant("ext"):
        oe, ste, pe = ref.step_box(box.astype(np.longdouble), dt, dh, par)
    assert pe == p64 and (ste.n_retry_pg, ste.n_unphys_final) == (st64.n_retry_pg, st64.n_unphys_final)
    e = step_err(o64.astype(np.longdouble), oe, 0)
    assert 0 < float(e.max()) <= 1e-11, float(e.max())
