"""Mutation check of the oracle's pins ("Next round" #1).

Each entry makes ONE plausible one-line mistake in a scratch copy of oracle/srhd_ref.cpp, rebuilds the
oracle there and runs the pin tests named beside it against the mutant: at least one must FAIL.  A pin
that still passes means that part of the oracle is unpinned.  Nothing here touches the real oracle/.

    python tests/mutants.py            # run all, print a table, exit 1 if any mutant survives
(tests/test_oracle_mutants.py runs the same from pytest.)
"""
import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PINS = ["tests/test_oracle_pins_r2.py", "tests/test_oracle_pins_r3.py", "tests/test_oracle_amr_hooks.py", "tests/test_oracle_vl.py", "tests/test_oracle_variants.py"]

# (name, cited passage, old text, new text, pytest node ids / -k expression that must fail)
MUTANTS = [
    ("umax: gamma_s dropped", "P:241 Eq. 26",
     "return gs * (std::fabs(W[1]) + std::fabs(W[2]) + std::fabs(W[3])) + real(3.0) * gamma * Us;",
     "return (std::fabs(W[1]) + std::fabs(W[2]) + std::fabs(W[3])) + real(3.0) * gamma * Us;",
     "test_umax"),
    ("umax: gamma dropped from 3 gamma U_s", "P:241 Eq. 26",
     "+ real(3.0) * gamma * Us;", "+ real(3.0) * Us;", "test_umax"),
    ("wave speeds: U_s^2 dropped from the denominator", "reading S6",
     "s.lam_p = (gamma * Un + Us * Q) / (g2 + Us2);\n  s.lam_m = (gamma * Un - Us * Q) / (g2 + Us2);",
     "s.lam_p = (gamma * Un + Us * Q) / (g2);\n  s.lam_m = (gamma * Un - Us * Q) / (g2);",
     "test_wave_speed_values or test_riemann_flux_values or test_hlle_satisfies"),
    ("wave-speed differences: U_t^2 dropped from lambda - v_n", "reading S6",
     "const real d_with = Us * a / (gamma * w);", "const real d_with = Us / (gamma * w);",
     "test_wave_speed_differences or test_riemann_flux"),
    ("wave-speed differences: 1 - lambda with a single factor a", "reading S6",
     "const real c_with = a * a / ((gamma + u) * (Q + Us) * w);", "const real c_with = a / ((gamma + u) * (Q + Us) * w);",
     "test_wave_speed_differences or test_riemann_flux_at_lorentz"),
    ("HLL: S_R - v_R without the other side's wave", "reading S6",
     "h.AR = R.dp + ((h.SR > real(0.5)) ? (R.cp - cpS) : (h.SR - R.lam_p));", "h.AR = R.dp;",
     "test_riemann_flux_values or test_hlle_satisfies"),
    ("HLLE: the right state's term halved", "P:225 (Mignone & Bodo 2005)",
     "    F[c] = (SR * BL * L.U[c] + SL * AR * R.U[c] + SR * L.pt[c] - SL * R.pt[c]) / den;",
     "    F[c] = (SR * BL * L.U[c] + real(0.5) * SL * AR * R.U[c] + SR * L.pt[c] - SL * R.pt[c]) / den;",
     "test_hlle_satisfies or test_riemann_flux_values"),
    ("HLLE: wave speeds swapped on the pressure terms", "P:225 (Mignone & Bodo 2005)",
     "    F[c] = (SR * BL * L.U[c] + SL * AR * R.U[c] + SR * L.pt[c] - SL * R.pt[c]) / den;",
     "    F[c] = (SR * BL * L.U[c] + SL * AR * R.U[c] + SL * L.pt[c] - SR * R.pt[c]) / den;",
     "test_hlle_satisfies or test_riemann_flux_values"),
    ("HLLC: p* term dropped from Etilde*", "reading S7",
     "Us[4] = (K.U[4] * A + ps * lam - K.p * K.vn) / dK;", "Us[4] = (K.U[4] * A - K.p * K.vn) / dK;",
     "test_riemann_flux_values"),
    ("HLLC: star momentum flux without p*", "reading S7",
     "F[1] = Us[1] * lam + ps;", "F[1] = Us[1] * lam;",
     "test_riemann_flux_values"),
    ("Hancock predictor: per-direction (split) increment", "P:225, reading S5",
     "Um[(d * 5 + q) * np + c] = Ucm[d][q] + dU[q];\n              Up[(d * 5 + q) * np + c] = Ucp[d][q] + dU[q];",
     "Um[(d * 5 + q) * np + c] = Ucm[d][q] - hdt * dF[d][q];\n              Up[(d * 5 + q) * np + c] = Ucp[d][q] - hdt * dF[d][q];",
     "test_second_order_convergence_on_the_3d_diagonal_wave"),
    ("Hancock predictor: split increment (bitwise / 40-digit pins)", "P:225, reading S5",
     "Um[(d * 5 + q) * np + c] = Ucm[d][q] + dU[q];\n              Up[(d * 5 + q) * np + c] = Ucp[d][q] + dU[q];",
     "Um[(d * 5 + q) * np + c] = Ucm[d][q] - hdt * dF[d][q];\n              Up[(d * 5 + q) * np + c] = Ucp[d][q] - hdt * dF[d][q];",
     "test_one_step_matches_40_digit or test_retry_ladder_equals"),
    ("retry ladder: factor 0.75 -> 0.5", "P:273",
     "beta = (pass <= K) ? beta * real(0.75) : real(0.0);", "beta = (pass <= K) ? beta * real(0.5) : real(0.0);",
     "test_retry_ladder_equals"),
    ("retry ladder: failing face states ignored", "reading S15",
     "if ((face_fail == 0 && cell_fail == 0) || beta == real(0.0)) break;",
     "if ((cell_fail == 0) || beta == real(0.0)) break;",
     "test_retry_ladder_equals"),
    ("VL: predictor advanced by a full step", "P:225, reading S18",
     "Uh[q] = cons_in[q * np + c] - hdt * ((dfx + dfy) + dfz);", "Uh[q] = cons_in[q * np + c] - real(2.0) * hdt * ((dfx + dfy) + dfz);",
     "test_vl_second_order or test_vl_equals"),
    ("VL: corrector reconstructs the OLD primitives (predictor ignored)", "P:225, reading S18",
     "a[m + 2] = (par.recon == 0 && (m == -2 || m == 2)) ? real(0.0) : Wh[q * np + c + (ptrdiff_t)m * stp[d]];",
     "a[m + 2] = (par.recon == 0 && (m == -2 || m == 2)) ? real(0.0) : Wc[q * np + c + (ptrdiff_t)m * stp[d]];",
     "test_vl_second_order"),
    ("update: flux difference with the wrong sign in z", "Eq. 4a, reading S12",
     "Un[q] = cons_in[q * np + c] - dtdh * ((dfx + dfy) + dfz);",
     "Un[q] = cons_in[q * np + c] - dtdh * ((dfx + dfy) - dfz);",
     "test_one_step_matches_40_digit"),
    ("polytropic EoS: Gamma dropped from the sound speed", "P:107 Eq. 11, reading S19",
     "return (kGnum * T) / (kGden * h);", "return T / h;",
     "test_gamma_law_eos_is_eq11 or test_gamma_law_sound_wave"),
    ("polytropic EoS: Gamma/(Gamma-1) inverted", "P:107 Eq. 11",
     "constexpr real kG1 = kGnum / (kGnum - kGden);", "constexpr real kG1 = (kGnum - kGden) / kGnum;",
     "test_gamma_law"),
    ("original scheme: the rest mass not subtracted in L", "P:198, P:626",
     "real L = std::fma(x, x, -musq) - real(1.0);", "real L = std::fma(x, x, -musq);",
     "test_fig16 or test_original"),
    # the seven survivors of the round-2 judge's mutation run: what decides which states count as unphysical
    ("Eq. 30 on updated cells: threshold 0 instead of eps_machine", "P:267-269 Eq. 30, O9",
     "  const real L = std::fma(x, x + real(2.0), -musq);\n#else\n  const real L = std::fma(x, x, -musq) - real(1.0);\n#endif\n  return L > kEps;",
     "  const real L = std::fma(x, x + real(2.0), -musq);\n#else\n  const real L = std::fma(x, x, -musq) - real(1.0);\n#endif\n  return L > real(0.0);",
     "test_eq30_threshold"),
    ("Eq. 30 on updated cells: Etilde > 0 not required", "SURVEY 8(c) O3, S9",
     "if (!(D > real(0.0)) || !(Et > real(0.0))) return false;", "if (!(D > real(0.0))) return false;",
     "test_negative_reduced_energy"),
    ("Eq. 30 on updated cells: D > 0 not required", "SURVEY 8(c) O3, S9",
     "if (!(D > real(0.0)) || !(Et > real(0.0))) return false;", "if (!(Et > real(0.0))) return false;",
     "test_negative_reduced_energy or test_vacuum_floor"),
    ("cons2prim verdict: Etilde > 0 not required", "SURVEY 8(c) O3",
     "bool phys = (D > real(0.0)) && (Et > real(0.0));", "bool phys = (D > real(0.0));",
     "test_negative_reduced_energy"),
    ("cons2prim: vacuum floor at 0 instead of the smallest normal number", "reading S10",
     "const bool dpos = D > kTiny;", "const bool dpos = D > real(0.0);",
     "test_vacuum_floor"),
    ("VL: a failing predictor state is not counted", "readings S18, S15",
     "&it, nullptr)) ++half_fail;   // S15", "&it, nullptr)) (void)0;   // S15",
     "test_vl_counts_a_failing_predictor"),
    ("boundary map: outflow on the high side copies cell n-2", "reading S11",
     "if (i >= n) return (bc_hi == 0) ? (i % n) : n - 1;", "if (i >= n) return (bc_hi == 0) ? (i % n) : n - 2;",
     "test_boundary_map"),
    ("boundary map: outflow on the low side copies cell 1", "reading S11",
     "if (i < 0) return (bc_lo == 0) ? ((i % n) + n) % n : 0;", "if (i < 0) return (bc_lo == 0) ? ((i % n) + n) % n : 1;",
     "test_boundary_map"),
    ("boundary map: periodic wrap off by one on the low side", "reading S11",
     "if (i < 0) return (bc_lo == 0) ? ((i % n) + n) % n : 0;", "if (i < 0) return (bc_lo == 0) ? ((i % n) + n - 1) % n : 0;",
     "test_boundary_map"),
    ("ghost interpolation: negative primitive children accepted", "reading S22, P:277",
     "if (!(v[0] > real(0.0)) || !(v[4] > real(0.0))) prim_bad = true;", "(void)prim_bad;",
     "test_ghost_interpolation_copies_the_parent"),
    ("original scheme: HLLC contact speed with D added to E", "reading S7, P:289",
     "const real Eh = Uh[4];  ", "const real Eh = Uh[4] + Uh[0];",
     "test_original_and_new"),
]


def run_mutant(m):
    name, cite, old, new, kexpr = m
    src = open(os.path.join(ROOT, "oracle", "srhd_ref.cpp")).read()
    if src.count(old) < 1:
        return name, cite, "STALE", f"pattern not found in oracle/srhd_ref.cpp: {old[:60]!r}"
    tmp = tempfile.mkdtemp(prefix="srhd_mutant_")
    try:
        shutil.copytree(os.path.join(ROOT, "oracle"), os.path.join(tmp, "oracle"),
                        ignore=shutil.ignore_patterns("*.so", "__pycache__"))
        with open(os.path.join(tmp, "oracle", "srhd_ref.cpp"), "w") as f:
            f.write(src.replace(old, new))
        env = dict(os.environ, SRHD_TEST_ORACLE_ROOT=tmp, SRHD_TEST_SKIP_CUDA_BUILD="1", OMP_NUM_THREADS="2")
        r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider"] + PINS + ["-k", kexpr],
                           cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
        tail = (r.stdout.strip().splitlines() or [""])[-1]
        if r.returncode == 1:
            return name, cite, "KILLED", tail
        return name, cite, "SURVIVED" if r.returncode == 0 else "ERROR", tail + r.stderr[-300:]
    finally:
        shutil.rmtree(tmp, ignore_errors=True)


def run_all(workers=4):
    with ThreadPoolExecutor(workers) as ex:
        return list(ex.map(run_mutant, MUTANTS))


if __name__ == "__main__":
    res = run_all()
    for name, cite, verdict, tail in res:
        print(f"{verdict:9s} {name}  [{cite}]  -- {tail}")
    sys.exit(0 if all(v == "KILLED" for _, _, v, _ in res) else 1)
