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
VARIANTS = {
    "libsrhd_b200.so": [],
    "libsrhd_b200_exact.so": ["-fmad=false", "-DSRHD_EXACT=1"],
}


def lib_path(exact=False):
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
    print("\n".join(lib_path(e) for e in (False, True)))
