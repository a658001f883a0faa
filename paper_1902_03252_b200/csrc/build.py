"""Builds liblt_gradient.so (the C-ABI CUDA library) in-tree for sm_100a with nvcc.  No GPU needed (cross-compiles).

    python -m paper_1902_03252_b200.csrc.build [--force] [--verbose]

--fmad=false: every fused multiply-add in the kernels is written explicitly (fma()/fmaf()), so that the fp64 grid
kernel and the fp64 list kernel produce identical bits and the mixed-rule criteria round exactly like their
definition (eq. 24-28).  No fast-math.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
PKG = os.path.dirname(HERE)
LIB = os.path.join(PKG, "liblt_gradient.so")
SOURCES = ["lt_api.cu"]


def deps():
    """Every source the library is built from: all *.cu / *.cuh of this folder and the C-ABI header."""
    here = sorted(f for f in os.listdir(HERE) if f.endswith((".cu", ".cuh")))
    return here + [os.path.join("..", "..", "include", "lt_gradient.h"), "build.py"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--fmad=false",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(os.path.join(HERE, d)) <= t for d in deps())


def build(force=False, verbose=False, defines=(), out=None):
    """defines / out: an experimental build (-D<name> ...) written to another path; lt.py loads it when the environment
    variable LT_GRADIENT_LIB names it.  The default build takes neither."""
    lib = out or LIB
    if not force and not defines and out is None and up_to_date():
        return LIB
    tmp = lib + ".tmp%d" % os.getpid()
    cmd = [nvcc()] + NVCC_FLAGS + ["-D" + d for d in defines] + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + \
          [os.path.join(HERE, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
