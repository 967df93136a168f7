"""Build libgf_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension machinery).

    python -m paper_1205_0752_b200.build [--force]
"""
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libgf_b200.so")
SOURCES = ["gf_api.cu", "gf_eval.cu", "gf_contour.cu", "gf_cut.cu", "gf_grid.cu", "gf_diag.cu", "gf_tables.cpp"]
HEADERS = [os.path.join(CSRC, "gf_internal.h"), os.path.join(CSRC, "gf_routes.cuh"), os.path.join(CSRC, "gf_dd.cuh"), os.path.join(ROOT, "include", "gf.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--threads", "4"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile every CUDA source of the package into paper_1205_0752_b200/libgf_b200.so."""
    if not force and not stale():
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("GF_NVCC_EXTRA", "").split() + ["-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-lquadmath"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
