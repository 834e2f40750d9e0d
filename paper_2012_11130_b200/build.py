"""Build the C-ABI CUDA libraries in-tree with nvcc for sm_100a (cross-compiles without a GPU).

  libsrhd_b200.so        production build (DFMA contraction on)
  libsrhd_b200_exact.so  same sources with -fmad=false -DSRHD_EXACT=1: reproduces a plain IEEE
                         evaluation of the paper's formulas bit for bit (used by the parity tests)

`python -m paper_2012_11130_b200.build` builds both; nothing here touches oracle/.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["srhd_convert.cu", "srhd_fluid.cu", "srhd_grid.cu", "srhd_refine.cu", "srhd_vl.cu", "srhd_amr.cu"]
HEADERS = ["srhd_math.cuh", "srhd_common.cuh", "srhd_uniform.cuh", os.path.join("..", "..", "include", "srhd.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-shared"]
_EXACT = ["-fmad=false", "-DSRHD_EXACT=1"]
_G53 = ["-DSRHD_EOS=1", "-DSRHD_GAMMA_NUM=5", "-DSRHD_GAMMA_DEN=3"]
_G43 = ["-DSRHD_EOS=1", "-DSRHD_GAMMA_NUM=4", "-DSRHD_GAMMA_DEN=3"]
VARIANTS = {
    "libsrhd_b200.so": [],
    "libsrhd_b200_exact.so": _EXACT,
    # SURVEY.md 8f row 4 (csrc/srhd_math.cuh header): the polytropic EoS of P:107 Eq. 11 and the paper's "original
    # scheme" (evolve E; for the A/B runs of Fig. 3 / Fig. 16).  The *_exact libraries reproduce the oracle's variants
    # bit for bit; libsrhd_b200_gamma53.so is the same polytropic path with FMA contraction (for timing).
    "libsrhd_b200_gamma53.so": _G53,
    "libsrhd_b200_gamma53_exact.so": _EXACT + _G53,
    "libsrhd_b200_gamma43_exact.so": _EXACT + _G43,
    "libsrhd_b200_orig_exact.so": _EXACT + ["-DSRHD_SCHEME=1"],
    # single precision throughout (srhd_real = float): the precision of every performance number in the paper
    # (the non-exact one with nvcc's fast single-precision division and square root: <= 2 ulp, no slow path)
    "libsrhd_b200_f32.so": ["-DSRHD_F32", "-prec-div=false", "-prec-sqrt=false"],
    "libsrhd_b200_f32_exact.so": _EXACT + ["-DSRHD_F32"],
}


def lib_path(exact=False):
    """False: the production library; True: the exact build; a string: that variant ("gamma53", "gamma53_exact",
    "gamma43_exact", "orig_exact", "f32", "f32_exact")."""
    if isinstance(exact, str):
        name = f"libsrhd_b200_{exact}.so"
        if name not in VARIANTS:
            raise ValueError(f"unknown library variant {exact!r}")
        return os.path.join(HERE, name)
    return os.path.join(HERE, "libsrhd_b200_exact.so" if exact else "libsrhd_b200.so")


def _stale(out):
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, extra=()):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    outs = []
    procs = []
    for name, flags in VARIANTS.items():
        out = os.path.join(HERE, name)
        outs.append(out)
        if not force and not _stale(out):
            continue
        cmd = [nvcc] + ARCH + COMMON + flags + list(extra) + (["-Xptxas", "-v"] if verbose else []) + \
              [os.path.join(CSRC, s) for s in SOURCES] + ["-o", out + ".tmp"]
        procs.append((out, cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for out, cmd, p in procs:
        log, _ = p.communicate()
        if p.returncode != 0:
            sys.stderr.write(log)
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        if verbose:
            sys.stderr.write(log)
        os.replace(out + ".tmp", out)
    return outs


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print("\n".join(os.path.join(HERE, n) for n in VARIANTS))
