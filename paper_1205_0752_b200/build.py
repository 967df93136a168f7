"""Build libgf_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension machinery).

    python -m paper_1205_0752_b200.build [--force]
"""
import hashlib
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libgf_b200.so")
SOURCES = ["gf_api.cu", "gf_eval.cu", "gf_contour.cu", "gf_taylor.cu", "gf_cut.cu", "gf_grid.cu", "gf_diag.cu", "gf_tables.cpp"]
HEADERS = [os.path.join(CSRC, "gf_internal.h"), os.path.join(CSRC, "gf_routes.cuh"), os.path.join(CSRC, "gf_dd.cuh"), os.path.join(CSRC, "gf_geometry.cuh"), os.path.join(ROOT, "include", "gf.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--threads", "4"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def source_id():
    """Hash of every source and header the library is built from (and of the flags): compiled into the library as
    gf_build_id(), so that a binary that does not belong to the sources beside it is refused at load time (file
    times do not survive the copy to the GPU box; contents do)."""
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for d in [os.path.join(CSRC, s) for s in SOURCES] + HEADERS:
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def built_id():
    """The source hash recorded in the built library ('' if there is none or it predates gf_build_id)."""
    if not os.path.exists(LIB):
        return ""
    import ctypes
    try:
        f = ctypes.CDLL(LIB).gf_build_id
    except (OSError, AttributeError):
        return ""
    f.restype = ctypes.c_char_p
    return f().decode()


def stale():
    return built_id() != source_id()


def build(force=False, verbose=False):
    """Compile every CUDA source of the package into paper_1205_0752_b200/libgf_b200.so."""
    if not force and not stale():
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("GF_NVCC_EXTRA", "").split() + [
        "-DGF_BUILD_ID=\"%s\"" % source_id(), "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-lquadmath"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
