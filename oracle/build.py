"""Build the CPU oracle shared library (TEST INFRASTRUCTURE ONLY -- see srhd_ref.hpp).

g++ -O2 -ffp-contract=off: no FMA contraction, so the only fused operations are the explicit
std::fma calls of the canonical forms.  Run: python oracle/build.py
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libsrhd_ref.so")
SRC = [os.path.join(HERE, "srhd_ref.cpp")]
HDR = [os.path.join(HERE, "srhd_ref.hpp")]
# "fma": the SAME source with the compiler free to contract a*b+c into fused multiply-adds -- a second, equally
# legitimate IEEE rounding of the same formulas.  Tests use it to measure how far two correct fp64 evaluations
# of this algorithm drift apart (tests/test_gpu_configs.py); it is never the parity reference.
# "gamma53" / "gamma43": the polytropic EoS of P:107 Eq. 11 with Gamma = 5/3 / 4/3; "orig": the paper's "original scheme"
# (evolve the total energy E) for the A/B runs of Fig. 3 / Fig. 16 (srhd_ref.cpp header).
VARIANTS = {"": ["-ffp-contract=off"], "fma": ["-ffp-contract=fast", "-mfma"],
            "gamma53": ["-ffp-contract=off", "-DSRHD_REF_EOS=1", "-DSRHD_REF_GAMMA_NUM=5", "-DSRHD_REF_GAMMA_DEN=3"],
            "gamma43": ["-ffp-contract=off", "-DSRHD_REF_EOS=1", "-DSRHD_REF_GAMMA_NUM=4", "-DSRHD_REF_GAMMA_DEN=3"],
            "orig": ["-ffp-contract=off", "-DSRHD_REF_SCHEME=1"],
            # "f32": every array and every operation in single precision (the precision of the paper's performance runs)
            "f32": ["-ffp-contract=off", "-DSRHD_REF_F32"],
            # "ext": the fp64 algorithm (same thresholds) evaluated in x87 extended precision (long double, eps 1.1e-19):
            # the "truth" both the fp64 oracle and the fp64 CUDA build are measured against; never the parity reference
            "ext": ["-ffp-contract=off", "-DSRHD_REF_EXT"]}


def lib_path(variant=""):
    return LIB if not variant else os.path.join(HERE, f"libsrhd_ref_{variant}.so")


def build(force: bool = False, variant: str = "") -> str:
    out = lib_path(variant)
    newest = max(os.path.getmtime(p) for p in SRC + HDR + [os.path.abspath(__file__)])
    if not force and os.path.exists(out) and os.path.getmtime(out) >= newest:
        return out
    cmd = ["g++", "-std=c++17", "-O2"] + VARIANTS[variant] + ["-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", out + ".tmp"] + SRC
    subprocess.run(cmd, check=True)
    os.replace(out + ".tmp", out)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
