"""Pins of the oracle's VL integrator ("VL (Falle 1991; van Leer 2006)"; reading S18 of DESIGN.md:
van Leer's predictor-corrector -- first-order fluxes advance the state by dt/2, its primitives are
reconstructed, the second set of fluxes does the full step) against what does not depend on the oracle:
bit-exact fixed point, no preferred axis, conservation, the paper's 3-D convergence test, the tiled and
whole-box forms, and a Python re-assembly from per-state calls (tests/py_step.py)."""
import numpy as np
import pytest

from paper_2012_11130_b200 import workloads as wl
from tests import py_step
from tests.test_oracle_pins_r2 import _diagonal_wave, _rough_box


def cons_of(ref, prim):
    return ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)


@pytest.mark.parametrize("recon", ["plm", "ppm"])
def test_vl_uniform_state_is_bit_exact_fixed_point(ref, recon):
    par = ref.params(recon, "hllc", integrator="vl")
    g = par.ghost
    assert g == (3 if recon == "plm" else 4)
    for W in ([1.0, 0.0, 0.0, 0.0, 1e-6], [0.7, 3e2, -1e2, 5e1, 1e-4], [1e-3, 0.0, 0.0, 1e6, 1e3]):
        prim = np.broadcast_to(np.array(W)[:, None, None, None], (5, 6 + 2 * g, 5 + 2 * g, 7 + 2 * g)).copy()
        cons = cons_of(ref, prim)
        out, st, passes = ref.step_box(cons, 0.3e-2, 1e-2, par)
        assert passes == 1 and st.n_unphys_final == 0
        assert np.array_equal(out, cons[:, g:-g, g:-g, g:-g])


def test_vl_axis_permutation_is_bit_identical(ref):
    par = ref.params("plm", "hllc", integrator="vl")
    res = []
    for axis in range(3):
        prim, dh, bc = wl.shock_tube(n_long=32, n_trans=16, axis=axis, left=(1.0, 0.0, 10.0), right=(0.125, 0.0, 0.1))
        cons = cons_of(ref, prim)
        dt = ref.cfl_dt(cons, 0.4, dh, par)
        for _ in range(3):
            cons, st, _ = ref.grid_step_whole(cons, dt, dh, par, bc)
        res.append(cons)
    x = res[0]
    assert np.array_equal(x, res[1].transpose(0, 1, 3, 2)[[0, 2, 1, 3, 4]])
    assert np.array_equal(x, res[2].transpose(0, 3, 2, 1)[[0, 3, 2, 1, 4]])
    assert np.abs(x[1]).max() > 0.1


def test_vl_conservation_and_tiling(ref):
    par = ref.params("plm", "hlle", integrator="vl")
    k = 2 * np.pi * (np.arange(32) + 0.5) / 32.0
    Z, Y, X = np.meshgrid(k[:16], k[:16], k, indexing="ij")
    prim = np.empty((5, 16, 16, 32))
    prim[0] = 1.0 + 0.5 * np.sin(X) * np.cos(2 * Y)
    prim[1] = 0.8 * np.sin(2 * Y + 2 * Z)
    prim[2] = -0.5 * np.cos(X - 2 * Z)
    prim[3] = 0.3 * np.sin(X + 2 * Y + 2 * Z)
    prim[4] = prim[0] * 10.0 ** (-1.0 + 0.5 * np.sin(2 * Z) * np.sin(X))
    cons = cons_of(ref, prim)
    dh = 1.0 / 32
    tot0, scale = cons.reshape(5, -1).sum(1), np.abs(cons).reshape(5, -1).sum(1)
    for _ in range(3):
        dt = ref.cfl_dt(cons, 0.4, dh, par)
        whole, st, passes = ref.grid_step_whole(cons, dt, dh, par, ["periodic"] * 6)
        tiled, st_t = ref.grid_step_tiled(cons, dt, dh, par, ["periodic"] * 6)
        assert passes == 1 and st_t.n_retry_pg == 0
        assert np.array_equal(whole, tiled)           # patch-group tiles == one box, bit for bit
        cons = whole
    assert np.all(np.abs(cons.reshape(5, -1).sum(1) - tot0) <= 64 * 2.2e-16 * scale)


@pytest.mark.parametrize("T0", [1e-10, 1e10])
def test_vl_second_order_on_the_3d_diagonal_wave(ref, T0):
    """P:301 / Fig. 3 with the VL scheme ("MUSCL-Hancock and VL schemes")."""
    par = ref.params("plm", "hllc", integrator="vl")
    errs = []
    for N in (16, 32, 64):
        prim, dh, ph, omega, cs = _diagonal_wave(ref, N, T0)
        cons = cons_of(ref, prim)
        t, t_end = 0.0, 0.5 * np.pi / omega
        while t < t_end:
            dt = min(ref.cfl_dt(cons, 0.5, dh, par), t_end - t)
            cons, st = ref.grid_step_tiled(cons, dt, dh, par, ["periodic"] * 6)
            assert st.n_retry_pg == 0
            t += dt
        rho = ref.cons2prim(cons.reshape(5, -1))[0][0].reshape(N, N, N)
        errs.append(float(np.abs(1.0 - rho / (1.0 + 1e-6 * np.sin(ph - omega * t_end))).mean()))
    o1, o2 = np.log2(errs[0] / errs[1]), np.log2(errs[1] / errs[2])
    assert errs[0] < 0.5e-6 and o1 > 1.8 and o2 > 1.8, (errs, o1, o2)


def test_vl_equals_its_python_reassembly(ref):
    seen = set()
    for recon, seed, mult in (("plm", 4, 1.0), ("plm", 12, 1.0), ("plm", 6, 2.5), ("ppm", 2, 1.0), ("ppm", 10, 1.0)):
        par = ref.params(recon, "hllc", max_retry=2, integrator="vl")
        cons = _rough_box(ref, seed, par.ghost, n=3)
        dh = 1.0 / 64
        dt = mult * 0.4 * dh / ref.max_signal_speed(cons.reshape(5, -1))
        out, passes, hf, cf, hist = py_step.ladder_vl(ref, cons, dt, dh, par)
        got, st, got_passes = ref.step_box(cons, dt, dh, par)
        assert got_passes == passes, (recon, seed, hist)
        assert np.array_equal(got, out, equal_nan=True)
        assert (st.n_retry_pg, st.n_c2p_fail, st.n_unphys_final) == (int(passes > 1), hf, cf)
        seen.add(passes)
    assert len(seen) >= 2, seen
