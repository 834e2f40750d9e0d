"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU and
exports every symbol include/srhd.h declares; argument errors are reported before any launch."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libs():
    from paper_2012_11130_b200 import build
    build.build()
    paths = [build.lib_path(False), build.lib_path(True)]
    paths += [os.path.join(os.path.dirname(paths[0]), n) for n in build.VARIANTS if os.path.join(os.path.dirname(paths[0]), n) not in paths]
    return [C.CDLL(p) for p in paths]     # production, exact, then every variant library


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "srhd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(srhd_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for n in ("srhd_prim2cons", "srhd_cons2prim", "srhd_fluid_step", "srhd_max_signal_speed"):
        assert n in names


def test_every_declared_symbol_is_exported(libs):
    names = declared_symbols()
    assert len(names) >= 10
    for L in libs:
        for n in names:
            assert hasattr(L, n), n


def test_binding_symbol_list_matches_header():
    from paper_2012_11130_b200 import binding
    assert sorted(binding.SYMBOLS) == declared_symbols()


def test_exact_flag(libs):
    assert libs[0].srhd_build_is_exact() == 0
    assert libs[1].srhd_build_is_exact() == 1


def test_defaults_and_error_strings():
    from paper_2012_11130_b200 import binding as b
    p = b.params("ppm", "hllc")
    assert (p.recon, p.riemann, p.ghost, p.max_retry, p.newton_max_iter) == (1, 1, 3, 8, 20)
    assert p.minmod_coeff == 1.5 and p.newton_rtol == 1e-15
    assert b.params("plm", "hlle").ghost == 2
    L = b.load_library()
    for code in range(-7, 1):
        assert len(L.srhd_error_string(code)) > 1
    assert L.srhd_workspace_bytes(10, C.byref(p)) == 10   # MUSCL-Hancock: one flag byte per patch group


def test_argument_errors_without_gpu():
    """Bad arguments are rejected on the host, before any CUDA call."""
    from paper_2012_11130_b200 import binding as b
    L = b.load_library()
    p = b.params("plm", "hllc")
    assert L.srhd_prim2cons(None, None, 4, 4, None) == -1
    assert L.srhd_prim2cons(16, 32, 8, 4, None) == -3
    assert L.srhd_cons2prim(16, 32, 8, 8, None, None, None) == -1
    bad = b.params("plm", "hllc")
    bad.ghost = 3
    assert L.srhd_cons2prim(16, 32, 8, 8, C.byref(bad), None, None) == -2
    assert L.srhd_fluid_step(16, 1 << 30, 1, 0.0, 1.0, C.byref(p), None, None) == -4
    assert L.srhd_fluid_step(16, 1 << 30, -1, 0.1, 1.0, C.byref(p), None, None) == -3
    assert L.srhd_fluid_step(24, 1 << 30, 1, 0.1, 1.0, C.byref(p), None, None) == -6
    assert L.srhd_fluid_step(1 << 20, (1 << 20) + 64, 1, 0.1, 1.0, C.byref(p), None, None) == -5
    # vector accesses: cons_out on an 8-byte boundary (a view one double into a buffer) is refused, not faulted on
    assert L.srhd_fluid_step(16, (1 << 30) + 8, 1, 0.1, 1.0, C.byref(p), None, None) == -6
    assert L.srhd_fluid_step_noalloc(16, (1 << 30) + 8, 1, 0.1, 1.0, C.byref(p), None, None) == -6
    # the no-allocation variant: srhd_fluid_step's checks plus its own two limits (include/srhd.h)
    assert L.srhd_fluid_step_noalloc(16, 1 << 30, 1, 0.0, 1.0, C.byref(p), None, None) == -4
    assert L.srhd_fluid_step_noalloc(24, 1 << 30, 1, 0.1, 1.0, C.byref(p), None, None) == -6
    assert L.srhd_fluid_step_noalloc(16, 1 << 44, b.NOALLOC_MAX_NPG + 1, 0.1, 1.0, C.byref(p), None, None) == -7
    assert L.srhd_fluid_step_noalloc(16, 1 << 30, 1, 0.1, 1.0, C.byref(b.params("plm", "hllc", integrator="vl")), None, None) == -2
    # device-side dt variant: needs the speed pointer and a positive Courant number
    assert L.srhd_fluid_step_cfl(16, 1 << 30, None, 1, 0.4, 1.0, None, 0.0, C.byref(p), None, None) == -1
    assert L.srhd_fluid_step_cfl(16, 1 << 30, None, 1, 0.0, 1.0, 64, 0.0, C.byref(p), None, None) == -4
    assert L.srhd_fluid_step_cfl(16, 1 << 30, None, 1, 0.4, -1.0, 64, 0.0, C.byref(p), None, None) == -4
    # refinement flags: quantity and thresholds are checked
    assert L.srhd_refine_flags(16, 1, 9, 0.3, 0.0, C.byref(p), 64, None) == -2
    assert L.srhd_refine_flags(16, 1, 3, -1.0, 0.0, C.byref(p), 64, None) == -2
    assert L.srhd_refine_flags(None, 1, 3, 0.3, 0.0, C.byref(p), 64, None) == -1
    assert L.srhd_grid_scatter_speed(16, 32, 16, 16, 16, C.byref(p), None, None) == -1
    assert L.srhd_fp64_peak_probe(None, 4, None, None) == -1
    bc = (C.c_int * 6)(0, 0, 0, 0, 0, 0)
    assert L.srhd_grid_gather(16, 32, 16, 24, 16, 2, bc, None, None, None) == -3
    assert L.srhd_grid_scatter(16, 32, 16, 16, 0, None) == -3
    # the whole-step call: pointers, extents, Courant number, in == out
    assert L.srhd_grid_step_cfl(None, 1 << 30, 1 << 31, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -1
    assert L.srhd_grid_step_cfl(16, 1 << 30, 1 << 31, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, None, None) == -1
    assert L.srhd_grid_step_cfl(16, 1 << 30, 1 << 31, None, 16, 24, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -3
    assert L.srhd_grid_step_cfl(16, 1 << 30, 1 << 31, None, 16, 16, 16, bc, None, None, 0.0, 1.0, 0.0, C.byref(p), None, 64, None) == -4
    assert L.srhd_grid_step_cfl(16, 16, 1 << 31, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -5
    assert L.srhd_grid_step_cfl(16, 1 << 30, 1 << 31, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(bad), None, 64, None) == -2
    # round 3 (ADVICE): alignment of the three state buffers, range overlap (not only pointer equality), flat-grid overflow
    assert L.srhd_grid_step_cfl(24, 1 << 30, 1 << 31, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -6
    assert L.srhd_grid_step_cfl(16, (1 << 30) + 8, 1 << 31, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -6
    assert L.srhd_grid_step_cfl(16, 1 << 30, (1 << 31) + 8, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -6
    assert L.srhd_grid_step_cfl(1 << 30, (1 << 30) + 4096, 1 << 31, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -5
    assert L.srhd_grid_step_cfl(1 << 30, 1 << 31, (1 << 30) + 4096, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -5
    assert L.srhd_grid_step_cfl(1 << 30, 1 << 31, (1 << 31) - 4096, None, 16, 16, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -5
    assert L.srhd_grid_step_cfl(1 << 30, 1 << 31, 1 << 32, None, 8192, 4096, 16, bc, None, None, 0.4, 1.0, 0.0, C.byref(p), None, 64, None) == -3
    # every variant library answers the same way and says what it is
    for key in ("gamma53", "gamma53_exact", "gamma43_exact", "orig_exact", "f32", "f32_exact", True):
        V = b.load_library(key)
        assert V.srhd_prim2cons(None, None, 4, 4, None) == -1
        assert b"eos=" in V.srhd_build_variant() and b"precision=" in V.srhd_build_variant()
    b.load_library()


def test_no_cpu_fallback():
    """The binding refuses CPU tensors instead of computing anything on the host."""
    import torch
    from paper_2012_11130_b200 import binding as b
    with pytest.raises(b.SrhdError):
        b.prim2cons(torch.ones(5, 4, dtype=torch.float64))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2012_11130_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, re.M), f
                assert not re.search(r"#include\s+\".*oracle", txt), f
                assert "srhd_ref_" not in txt and "libsrhd_ref" not in txt, f   # the oracle's symbol prefix
