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


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in SRC + HDR)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB] + SRC
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
