"""The C-ABI library loads and exports every symbol include/gf.h declares; host-only entry points
behave as the header says (no GPU, no compute kernels are launched here)."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gf.h")


@pytest.fixture(scope="module")
def gf():
    from paper_1205_0752_b200 import build
    build.build()
    import paper_1205_0752_b200 as gf
    gf.lib()
    return gf


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gf_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(gf):
    names = declared_symbols()
    assert {"gf_make_grid", "gf_make_quadrature", "gf_eval_grid", "gf_eval_grid_host"} <= set(names)
    raw = ctypes.CDLL(gf.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), "include/gf.h declares %s but libgf_b200.so does not export it" % n
    # and the binding knows every one of them
    assert set(names) == set(gf._SIGNATURES), set(names) ^ set(gf._SIGNATURES)


def test_library_is_sm100a_only(gf):
    out = subprocess.run(["cuobjdump", "-lelf", gf.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_struct_layout_matches_header(gf):
    # gf_params: 2 propagators of (int, 5 doubles) + 3 doubles + int + 2 doubles + 3 ints + 1 double, natural alignment
    assert ctypes.sizeof(gf.gf_propagator) == 48
    assert ctypes.sizeof(gf.gf_params) == 2 * 48 + 3 * 8 + 8 + 2 * 8 + 8 + 8 + 8
    assert ctypes.sizeof(gf.gf_launch_info) == 40 + 8 + 22 * 8


def test_host_quadrature_is_symmetric_and_exact(gf):
    """gf_make_quadrature_host makes no CUDA call: checked here against exact moments
    (the GPU tests compare the same tables with the oracle's)."""
    for n in (1, 2, 7, 64, 512):
        x, w = gf.make_quadrature_host("gauss_legendre", n)
        assert np.array_equal(x, -x[::-1]) and np.array_equal(w, w[::-1])
        for k in range(0, min(2 * n, 30), 2):
            assert abs(np.sum(w * x ** k) - 2.0 / (k + 1)) < 2e-14
    z, w = gf.make_quadrature_host("gauss_cheb2", 33, measure="sqrt1mz2")
    assert abs(np.sum(w) - np.pi / 2) < 1e-14 and abs(np.sum(w * z * z) - np.pi / 8) < 1e-14
    z, w = gf.make_quadrature_host("tanh_sinh", 49, measure="sqrt1mz2")
    assert abs(np.sum(w) - np.pi / 2) < 1e-11


def test_host_rules_of_the_d_dimensional_measure(gf):
    """gf_make_quadrature_dim_host (no CUDA call): exact moments B(k+1/2, (d-1)/2) for the Gauss rule of each measure
    (Chebyshev-1 d = 2, Legendre d = 3, Chebyshev-2 d = 4: PAPER.md:138), d = 3 / 4 identical to the fixed measures,
    exactly mirrored tables, argument errors.  The GPU tests compare the same tables with the oracle's."""
    from math import gamma, pi
    for kind, dim in (("gauss_cheb1", 2.0), ("gauss_legendre", 3.0), ("gauss_cheb2", 4.0), ("gauss_cheb1", 6.0)):
        z, w = gf.make_quadrature_dim_host(kind, 24, dim)
        assert np.array_equal(z, -z[::-1]) and np.array_equal(w, w[::-1]) and np.all(np.diff(z) > 0)
        for k in range(8):
            ref = gamma(k + 0.5) * gamma((dim - 1) / 2) / gamma(k + dim / 2)
            assert abs(np.sum(w * z ** (2 * k)) - ref) < 4e-15 * ref * 4, (kind, dim, k)
    z, w = gf.make_quadrature_dim_host("gauss_cheb1", 5, 2.0)
    assert np.allclose(w, pi / 5, rtol=1e-15) and abs(z[-1] - np.cos(pi / 10)) < 2e-16
    for kind in ("gauss_legendre", "gauss_cheb2", "tanh_sinh"):
        for dim, meas in ((3.0, "plain"), (4.0, "sqrt1mz2")):
            a, b = gf.make_quadrature_dim_host(kind, 33, dim), gf.make_quadrature_host(kind, 33, measure=meas)
            assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    for bad in (0.5, 9.0, float("nan")):
        with pytest.raises(gf.GfError) as e:
            gf.make_quadrature_dim_host("gauss_legendre", 8, bad)
        assert e.value.status == 2


def test_argument_errors_without_gpu(gf):
    L = gf.lib()
    bub = {"kind": "massive", "m2": 1.0}
    P = gf.make_params(bub, bub, 1e4)
    info = gf.gf_launch_info()
    assert L.gf_eval_launch_info(ctypes.byref(P), 64, 32, 4096, ctypes.byref(info)) == 0
    assert info.evals == 4096 * 64 * 32 and info.block_threads > 0 and info.grid_blocks > 0
    assert L.gf_eval_launch_info(None, 64, 32, 4096, ctypes.byref(info)) == 1          # GF_ERR_NULL
    assert L.gf_eval_launch_info(ctypes.byref(P), 0, 32, 4096, ctypes.byref(info)) == 2  # GF_ERR_ARG
    assert b"n_rad" in L.gf_last_error()
    P.taylor_order = 1   # eq. (13) with n = 1: its own kernel, no per-route instruction model
    assert L.gf_eval_launch_info(ctypes.byref(P), 64, 32, 4096, ctypes.byref(info)) == 0
    assert info.grid_blocks > 0 and info.series_term_dfma == 0
    P.taylor_order = 5
    assert L.gf_eval_launch_info(ctypes.byref(P), 64, 32, 4096, ctypes.byref(info)) == 3  # UNSUPPORTED
    P = gf.make_params(bub, bub, -1.0)
    assert L.gf_eval_launch_info(ctypes.byref(P), 64, 32, 4096, ctypes.byref(info)) == 2
    for bad in (dict(cutoff2=1e61), dict(cutoff2=1e4, dim=9.0), dict(cutoff2=1e4, routing=2)):
        P = gf.make_params(bub, bub, **bad)
        assert L.gf_eval_launch_info(ctypes.byref(P), 64, 32, 4096, ctypes.byref(info)) == 2, bad
    for unsupported in (dict(routing="symmetric", taylor_order=1), dict(taylor_order=1, precision=32), dict(sub=0.5)):
        P = gf.make_params(bub, bub, 1e4, **unsupported)
        assert L.gf_eval_launch_info(ctypes.byref(P), 64, 32, 4096, ctypes.byref(info)) == 3, unsupported
    assert gf.lib().gf_eval_workspace_size(ctypes.byref(gf.make_params(bub, bub, 1e4)), 64, 32) > 0
    assert gf.lib().gf_eval_workspace_size(ctypes.byref(gf.make_params(bub, bub, 1e4)), 0, 32) == -1
    assert gf.lib().gf_trim_scratch() == 0
    P = gf.make_params(bub, {"kind": "massive", "m2": 2.0}, 1e4, contour="thread")
    assert L.gf_eval_launch_info(ctypes.byref(P), 64, 32, 4096, ctypes.byref(info)) == 3
    assert L.gf_make_grid(0.0, 1.0, 4, 0.0, 1.0, 4, 0, 0.0, None, None) == 1
    assert L.gf_make_quadrature_host(9, 4, 0.0, 0, None, None) != 0
    # gf_eval_grid_static checks its arguments and the size of the workspace before any CUDA call
    P = gf.make_params(bub, bub, 1e4)
    assert L.gf_eval_grid_static(ctypes.byref(P), None, None, 64, None, None, 32, None, 0, None, None) == 1
    assert L.gf_eval_grid_static(None, None, None, 64, None, None, 32, None, 0, None, None) == 1
    buf = (ctypes.c_double * 4)()
    ptr = ctypes.addressof(buf)   # never dereferenced on the paths below
    assert L.gf_eval_grid_static(ctypes.byref(P), ptr, ptr, 0, ptr, ptr, 32, ptr, 2, ptr, None) == 2
    Pa = gf.make_params(bub, bub, 1e4, contour="auto")
    need = L.gf_eval_workspace_size(ctypes.byref(Pa), 2048, 32)
    assert need > gf.STATIC_WORKSPACE_BYTES
    assert L.gf_eval_grid_static(ctypes.byref(Pa), ptr, ptr, 2048, ptr, ptr, 32, ptr, 2, ptr, None) == 2
    assert b"GF_STATIC_WORKSPACE_BYTES" in L.gf_last_error() and str(need).encode() in L.gf_last_error()
    assert gf.radial_table_size("real", 64) == 64
    assert gf.radial_table_size("auto", 64) == 64 + 32 + 16 + 8
    assert gf.radial_table_size("auto", 63) == -1


def test_no_cpu_fallback(gf):
    """Without a CUDA device the product path raises; it never routes to the oracle."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(gf.GfError):
        gf.make_grid(0.0, 1.0, 4, 0.0, 1.0, 4)
    src = open(os.path.join(ROOT, "paper_1205_0752_b200", "__init__.py")).read()
    assert "oracle" not in src.replace("no CPU fallback", "")
