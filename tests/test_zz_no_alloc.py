"""gf_eval_grid_static: the entry point that allocates nothing (include/gf.h) against gf_eval_grid, the existing path.

Named so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide the other
tests.  Each test passes alone in a fresh process and after the rest of the suite (the static workspace keeps the
last call's tables; every call rewrites all it reads).
"""
import ctypes

import numpy as np
import pytest
import torch

import gf_workloads as W

pytestmark = pytest.mark.gpu

TOL64 = 1e-11   # the bar of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def gf():
    import paper_1205_0752_b200 as gf
    gf.lib()  # fails loudly if the extension is missing
    assert torch.cuda.is_available()
    return gf


def relerr(g, ref):
    g = g.cpu().numpy().ravel()
    ref = ref.cpu().numpy().ravel()
    both_zero = (ref == 0) & (g == 0)
    e = np.abs(g - ref) / np.where(ref == 0, 1.0, np.abs(ref))
    e[both_zero] = 0.0
    return e


def problem(gf, name, contour):
    cfg = W.CONFIGS[name]
    P = gf.make_params(cfg["line_k"], cfg["line_pk"], cfg["cutoff2"], prefactor=W.PREFACTOR, map_scale=W.MAP_SCALE,
                       contour=contour, precision=64)
    rn, rw = gf.make_radial_tables(contour, cfg["n_rad"], W.RADIAL_RULE)
    z, wz = gf.make_quadrature(W.ANGULAR_RULE, cfg["n_ang"], measure="sqrt1mz2")
    x = gf.make_grid(cfg["re"][0], cfg["re"][1], cfg["n_re"], cfg["im"][0], cfg["im"][1], cfg["n_im"],
                     spacing=cfg["spacing"], im_abs_min=cfg["im_abs_min"])
    return cfg, P, rn, rw, z, wz, x


def test_static_workspace_matches_the_existing_path_on_two_calls_in_a_row(gf):
    """Two calls in a row with different parameters, orders and contour policies (the second finds the first one's
    tables in the workspace), then the first problem again: each equals gf_eval_grid's result."""
    jobs = [("cfg1_tiny", "real"), ("cfg2_mid", "auto"), ("cfg1_tiny", "real")]
    for name, contour in jobs:
        cfg, P, rn, rw, z, wz, x = problem(gf, name, contour)
        ref = gf.eval_grid(P, rn, rw, cfg["n_rad"], z, wz, x)
        out = torch.full_like(x, complex(float("nan"), float("nan")))
        got = gf.eval_grid_static(P, rn, rw, cfg["n_rad"], z, wz, x, out=out)
        torch.cuda.synchronize()
        assert got.data_ptr() == out.data_ptr()
        assert torch.isfinite(ref.real).all() and torch.isfinite(ref.imag).all()
        e = relerr(got, ref)
        assert e.max() <= TOL64, (name, contour, e.max())


def test_same_call_twice_gives_the_same_result(gf):
    cfg, P, rn, rw, z, wz, x = problem(gf, "cfg1_tiny", "ray_arc")
    a = gf.eval_grid_static(P, rn, rw, cfg["n_rad"], z, wz, x).clone()
    b = gf.eval_grid_static(P, rn, rw, cfg["n_rad"], z, wz, x)
    torch.cuda.synchronize()
    assert torch.equal(a.view(torch.float64), b.view(torch.float64))
    ref = gf.eval_grid(P, rn, rw, cfg["n_rad"], z, wz, x)
    assert relerr(b, ref).max() <= TOL64


def test_workspace_beyond_the_limit_is_refused(gf):
    """Orders whose tables do not fit the static workspace: GF_ERR_ARG with both sizes in the message, nothing launched."""
    cfg, P, _, _, z, wz, x = problem(gf, "cfg1_tiny", "auto")
    n_rad = 2048
    P2 = gf.make_params(cfg["line_k"], cfg["line_pk"], cfg["cutoff2"], prefactor=W.PREFACTOR, map_scale=W.MAP_SCALE,
                        contour="auto", precision=64)
    need = int(gf.lib().gf_eval_workspace_size(ctypes.byref(P2), n_rad, cfg["n_ang"]))
    assert need > gf.STATIC_WORKSPACE_BYTES, need
    rn, rw = gf.make_radial_tables("auto", n_rad, W.RADIAL_RULE)
    out = torch.zeros_like(x)
    with pytest.raises(gf.GfError) as err:
        gf.eval_grid_static(P2, rn, rw, n_rad, z, wz, x, out=out)
    assert err.value.status == 2 and str(need) in str(err.value) and str(gf.STATIC_WORKSPACE_BYTES) in str(err.value)
    torch.cuda.synchronize()
    assert (out == 0).all()
    # the same orders through the existing path still work, and the static path still works afterwards
    ref = gf.eval_grid(P2, rn, rw, n_rad, z, wz, x)
    assert torch.isfinite(ref.real).all()
    cfg, P, rn, rw, z, wz, x = problem(gf, "cfg1_tiny", "real")
    assert relerr(gf.eval_grid_static(P, rn, rw, cfg["n_rad"], z, wz, x),
                  gf.eval_grid(P, rn, rw, cfg["n_rad"], z, wz, x)).max() <= TOL64
