"""paper_1205_0752_b200 -- thin Python binding of libgf_b200 (include/gf.h).

Argument marshalling only: every step of the hot path (grid fill, evaluation of the double integral,
reductions, stores) runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and
streams.  There is no CPU fallback: if the shared library is missing, importing works but the first
call raises; if no CUDA device is present the library returns GF_ERR_CUDA and the call raises.
"""
import ctypes
import os

import numpy as np
import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libgf_b200.so")

QUAD = {"gauss_legendre": 0, "gauss_cheb2": 1, "tanh_sinh": 2, "gauss_cheb1": 3}
MEASURE = {"plain": 0, "sqrt1mz2": 1}
PROP = {"massive": 0, "rational": 1}
CONTOUR = {"real": 0, "ray_arc": 1, "thread": 2, "auto": 3}
SPACING = {"uniform": 0, "log_abs_im": 1}
STATUS = {0: "GF_OK", 1: "GF_ERR_NULL", 2: "GF_ERR_ARG", 3: "GF_ERR_UNSUPPORTED", 4: "GF_ERR_CUDA"}


class GfError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (STATUS.get(status, status), message))
        self.status = status


class gf_propagator(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("m2_re", ctypes.c_double), ("m2_im", ctypes.c_double),
                ("M2", ctypes.c_double), ("a", ctypes.c_double), ("b", ctypes.c_double)]


class gf_params(ctypes.Structure):
    _fields_ = [("line_k", gf_propagator), ("line_pk", gf_propagator), ("cutoff2", ctypes.c_double),
                ("sub_re", ctypes.c_double), ("sub_im", ctypes.c_double), ("taylor_order", ctypes.c_int),
                ("prefactor", ctypes.c_double), ("map_scale", ctypes.c_double), ("contour", ctypes.c_int),
                ("precision", ctypes.c_int), ("routing", ctypes.c_int), ("dim", ctypes.c_double)]


class gf_launch_info(ctypes.Structure):
    _fields_ = [("block_threads", ctypes.c_int), ("grid_blocks", ctypes.c_longlong), ("split", ctypes.c_int),
                ("smem_bytes", ctypes.c_int), ("n_pairs", ctypes.c_int), ("n_terms", ctypes.c_int),
                ("series_terms_max", ctypes.c_int), ("evals", ctypes.c_double)] + [
        (n, ctypes.c_double) for n in (
            "near_pair_dfma", "near_pair_other", "near_pair_fp32", "series_term_dfma", "series_term_other",
            "series_term_fp32", "exact_pair_dfma", "exact_pair_other", "node_near_dfma", "node_near_other",
            "node_moment_dfma", "node_moment_other", "node_cheb_dfma", "node_cheb_other", "node_exact_dfma",
            "node_exact_other", "tail_dfma", "tail_other", "blk_series_dfma", "blk_series_other", "blk_term_dfma",
            "blk_term_other")]


COUNTER_NAMES = ("near_pairs", "series_terms", "exact_pairs", "near_nodes", "moment_nodes", "exact_nodes",
                 "cheb_nodes", "series_terms_needed", "tails", "series_terms_fp32", "block_series", "block_series_terms",
                 "block_series_leaves")


_lib = None
_vp, _dbl, _int, _ll = ctypes.c_void_p, ctypes.c_double, ctypes.c_int, ctypes.c_longlong
_SIGNATURES = {
    "gf_make_grid": [_dbl, _dbl, _int, _dbl, _dbl, _int, _int, _dbl, _vp, _vp],
    "gf_make_grid_rows": [_dbl, _dbl, _int, _dbl, _dbl, _int, _int, _dbl, _int, _int, _vp, _vp],
    "gf_make_quadrature": [_int, _int, _dbl, _int, _vp, _vp, _vp],
    "gf_make_quadrature_host": [_int, _int, _dbl, _int, _vp, _vp],
    "gf_make_quadrature_dim": [_int, _int, _dbl, _dbl, _vp, _vp, _vp],
    "gf_make_quadrature_dim_host": [_int, _int, _dbl, _dbl, _vp, _vp],
    "gf_radial_table_size": [_int, _int],
    "gf_eval_grid": [ctypes.POINTER(gf_params), _vp, _vp, _int, _vp, _vp, _int, _vp, _ll, _vp, _vp],
    "gf_eval_grid_static": [ctypes.POINTER(gf_params), _vp, _vp, _int, _vp, _vp, _int, _vp, _ll, _vp, _vp],
    "gf_eval_grid_counted": [ctypes.POINTER(gf_params), _vp, _vp, _int, _vp, _vp, _int, _vp, _ll, _vp, _vp, _vp],
    "gf_eval_grid_host": [ctypes.POINTER(gf_params), _vp, _vp, _int, _vp, _vp, _int, _vp, _ll, _vp, _vp],
    "gf_eval_workspace_size": [ctypes.POINTER(gf_params), _int, _int],
    "gf_eval_prepare": [ctypes.POINTER(gf_params), _vp, _vp, _int, _vp, _vp, _int, _vp, _vp],
    "gf_eval_grid_prepared": [ctypes.POINTER(gf_params), _int, _int, _vp, _vp, _ll, _vp, _vp, _vp],
    "gf_eval_angular": [ctypes.POINTER(gf_params), _dbl, _dbl, _vp, _vp, _int, _vp, _ll, _vp, _vp],
    "gf_cut_crossings": [ctypes.POINTER(gf_params), _vp, _ll, _int, _vp, _vp],
    "gf_eval_launch_info": [ctypes.POINTER(gf_params), _int, _int, _ll, ctypes.POINTER(gf_launch_info)],
    "gf_diag_fp64_peak": [_int, _int, _ll, _vp, _vp],
    "gf_diag_dfma_issue": [_int, _int, _int, _ll, _vp, _vp],
    "gf_diag_radial_map": [_dbl, _dbl, _vp, _int, _vp, _vp],
    "gf_diag_contour_nodes": [ctypes.POINTER(gf_params), _int, _int, _vp, _vp, _vp, _dbl, _dbl, _vp, _vp, _vp, _vp],
    "gf_trim_scratch": [],
    "gf_last_error": [],
    "gf_version": [],
    "gf_build_id": [],
}


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libgf_b200.so is missing: run `python -m paper_1205_0752_b200.build` "
                               "(nvcc, sm_100a).  There is no CPU fallback.")
        from . import build as _build
        if os.path.isdir(_build.CSRC) and _build.stale():
            raise RuntimeError("libgf_b200.so was not built from the sources beside it (build id %r, sources %r): "
                               "run `python -m paper_1205_0752_b200.build`" % (_build.built_id(), _build.source_id()))
        L = ctypes.CDLL(LIB_PATH)
        for name, args in _SIGNATURES.items():
            f = getattr(L, name)
            f.argtypes = args
            f.restype = _int
        L.gf_radial_table_size.restype = _ll
        L.gf_eval_workspace_size.restype = _ll
        L.gf_last_error.restype = ctypes.c_char_p
        L.gf_version.restype = ctypes.c_char_p
        L.gf_build_id.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise GfError(rc, lib().gf_last_error().decode())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _device(device):
    if not torch.cuda.is_available():
        raise GfError(4, "no CUDA device: the hot path runs only in the sm_100a kernels (no CPU fallback)")
    return torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)


def _prop(d):
    p = gf_propagator()
    p.kind = PROP[d["kind"]]
    m2 = complex(d.get("m2", 0.0))
    p.m2_re, p.m2_im = m2.real, m2.imag
    p.M2, p.a, p.b = float(d.get("M2", 0.0)), float(d.get("a", 0.0)), float(d.get("b", 0.0))
    return p


def make_params(line_k, line_pk, cutoff2, prefactor=2.0 / np.pi, map_scale=1.0, contour="real", sub=0.0,
                taylor_order=0, precision=64, dim=4.0, routing="paper"):
    """gf_params from plain Python values.  Propagators: {'kind': 'massive', 'm2': complex} or
    {'kind': 'rational', 'M2': .., 'a': .., 'b': ..}."""
    P = gf_params()
    P.line_k, P.line_pk = _prop(line_k), _prop(line_pk)
    P.cutoff2 = float(cutoff2)
    s = complex(sub)
    P.sub_re, P.sub_im = s.real, s.imag
    P.taylor_order = int(taylor_order)
    P.prefactor = float(prefactor)
    P.map_scale = float(map_scale)
    P.contour = CONTOUR[contour] if isinstance(contour, str) else int(contour)
    P.precision = int(precision)
    P.dim = float(dim)
    P.routing = {"paper": 0, "symmetric": 1}[routing] if isinstance(routing, str) else int(routing)
    return P


def make_grid(re_min, re_max, n_re, im_min, im_max, n_im, spacing="uniform", im_abs_min=0.0, device=None,
              stream=None, out=None):
    """gf_make_grid: complex128 tensor [n_im, n_re] on the device."""
    dev = _device(device)
    x = out if out is not None else torch.empty((n_im, n_re), dtype=torch.complex128, device=dev)
    with torch.cuda.device(dev):
        _check(lib().gf_make_grid(re_min, re_max, n_re, im_min, im_max, n_im, SPACING[spacing], im_abs_min,
                                  x.data_ptr(), _stream(stream)))
    return x


def make_grid_rows(re_min, re_max, n_re, im_min, im_max, n_im, row_first, n_rows, spacing="uniform",
                   im_abs_min=0.0, device=None, stream=None, out=None):
    """gf_make_grid_rows: rows [row_first, row_first+n_rows) of the grid, complex128 [n_rows, n_re]."""
    dev = _device(device)
    x = out if out is not None else torch.empty((n_rows, n_re), dtype=torch.complex128, device=dev)
    with torch.cuda.device(dev):
        _check(lib().gf_make_grid_rows(re_min, re_max, n_re, im_min, im_max, n_im, SPACING[spacing], im_abs_min,
                                       row_first, n_rows, x.data_ptr(), _stream(stream)))
    return x


def make_quadrature(kind, n, step=0.0, measure="plain", device=None, stream=None):
    """gf_make_quadrature: (nodes, weights) float64 tensors on the device."""
    dev = _device(device)
    nodes = torch.empty(n, dtype=torch.float64, device=dev)
    weights = torch.empty(n, dtype=torch.float64, device=dev)
    with torch.cuda.device(dev):
        _check(lib().gf_make_quadrature(QUAD[kind], n, step, MEASURE[measure], nodes.data_ptr(),
                                        weights.data_ptr(), _stream(stream)))
    return nodes, weights


def make_quadrature_host(kind, n, step=0.0, measure="plain"):
    """gf_make_quadrature_host: (nodes, weights) numpy arrays (no CUDA call)."""
    nodes = np.empty(n, dtype=np.float64)
    weights = np.empty(n, dtype=np.float64)
    _check(lib().gf_make_quadrature_host(QUAD[kind], n, step, MEASURE[measure], nodes.ctypes.data,
                                         weights.ctypes.data))
    return nodes, weights


def make_quadrature_dim(kind, n, dim, step=0.0, device=None, stream=None):
    """gf_make_quadrature_dim: the rule for the angular measure (1 - z^2)^((dim-3)/2) dz, on the device."""
    dev = _device(device)
    nodes = torch.empty(n, dtype=torch.float64, device=dev)
    weights = torch.empty(n, dtype=torch.float64, device=dev)
    with torch.cuda.device(dev):
        _check(lib().gf_make_quadrature_dim(QUAD[kind], n, step, float(dim), nodes.data_ptr(), weights.data_ptr(),
                                            _stream(stream)))
    return nodes, weights


def make_quadrature_dim_host(kind, n, dim, step=0.0):
    """gf_make_quadrature_dim_host: the same tables as numpy arrays (no CUDA call)."""
    nodes = np.empty(n, dtype=np.float64)
    weights = np.empty(n, dtype=np.float64)
    _check(lib().gf_make_quadrature_dim_host(QUAD[kind], n, step, float(dim), nodes.ctypes.data, weights.ctypes.data))
    return nodes, weights


def radial_table_size(contour, n_rad):
    c = CONTOUR[contour] if isinstance(contour, str) else int(contour)
    return int(lib().gf_radial_table_size(c, n_rad))


def _levels(contour, n_rad):
    size = radial_table_size(contour, n_rad)
    if size < 0:
        raise GfError(2, "bad contour / n_rad (deformed contours need n_rad % 8 == 0)")
    return [n_rad] if size == n_rad else [n_rad, n_rad // 2, n_rad // 4, n_rad // 8]


def make_radial_tables(contour, n_rad, kind="gauss_legendre", device=None, stream=None):
    """The radial rule(s) gf_eval_grid expects for `contour`: one gf_make_quadrature call per level."""
    dev = _device(device)
    levels = _levels(contour, n_rad)
    nodes = torch.empty(sum(levels), dtype=torch.float64, device=dev)
    weights = torch.empty(sum(levels), dtype=torch.float64, device=dev)
    off = 0
    with torch.cuda.device(dev):
        for n in levels:
            _check(lib().gf_make_quadrature(QUAD[kind], n, 0.0, MEASURE["plain"], nodes[off:].data_ptr(),
                                            weights[off:].data_ptr(), _stream(stream)))
            off += n
    return nodes, weights


def make_radial_tables_host(contour, n_rad, kind="gauss_legendre"):
    xs, ws = zip(*[make_quadrature_host(kind, n) for n in _levels(contour, n_rad)])
    return np.concatenate(xs), np.concatenate(ws)


def _eval_checks(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out):
    if not x.is_cuda:
        raise GfError(2, "eval_grid takes device tensors; use eval_grid_host for host buffers")
    assert x.dtype == torch.complex128 and x.is_contiguous()
    for t in (rad_nodes, rad_weights, ang_nodes, ang_weights):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    assert ang_nodes.numel() == ang_weights.numel()
    need = radial_table_size(params.contour, n_rad)
    assert rad_nodes.numel() >= need and rad_weights.numel() >= need, "radial tables too short for this contour"
    odt = torch.complex64 if params.precision == 32 else torch.complex128
    if out is None:
        out = torch.empty(x.shape, dtype=odt, device=x.device)
    assert out.dtype == odt and out.is_contiguous() and out.numel() == x.numel()
    return out


def eval_grid(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out=None, stream=None):
    """gf_eval_grid on device tensors.  x: complex128, any shape; returns complex128 (precision 64) or
    complex64 (precision 32) of the same shape.  Asynchronous on the current stream."""
    out = _eval_checks(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out)
    with torch.cuda.device(x.device):
        _check(lib().gf_eval_grid(ctypes.byref(params), rad_nodes.data_ptr(), rad_weights.data_ptr(), n_rad,
                                  ang_nodes.data_ptr(), ang_weights.data_ptr(), ang_nodes.numel(),
                                  x.data_ptr(), x.numel(), out.data_ptr(), _stream(stream)))
    return out


STATIC_WORKSPACE_BYTES = 32 << 20   # GF_STATIC_WORKSPACE_BYTES of include/gf.h


def eval_grid_static(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out=None, stream=None):
    """gf_eval_grid_static: gf_eval_grid with the library's static device workspace (no allocation inside the
    library; pass `out` to allocate nothing here either).  Refuses workspaces beyond STATIC_WORKSPACE_BYTES; calls that
    overlap on the GPU race on the workspace (include/gf.h)."""
    out = _eval_checks(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out)
    with torch.cuda.device(x.device):
        _check(lib().gf_eval_grid_static(ctypes.byref(params), rad_nodes.data_ptr(), rad_weights.data_ptr(), n_rad,
                                         ang_nodes.data_ptr(), ang_weights.data_ptr(), ang_nodes.numel(),
                                         x.data_ptr(), x.numel(), out.data_ptr(), _stream(stream)))
    return out


def eval_grid_counted(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out=None, stream=None):
    """gf_eval_grid_counted: (G, {route counter: value}).  Synchronises to read the counters."""
    out = _eval_checks(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out)
    counters = torch.zeros(len(COUNTER_NAMES), dtype=torch.int64, device=x.device)
    with torch.cuda.device(x.device):
        _check(lib().gf_eval_grid_counted(ctypes.byref(params), rad_nodes.data_ptr(), rad_weights.data_ptr(), n_rad,
                                          ang_nodes.data_ptr(), ang_weights.data_ptr(), ang_nodes.numel(),
                                          x.data_ptr(), x.numel(), out.data_ptr(), counters.data_ptr(),
                                          _stream(stream)))
    return out, dict(zip(COUNTER_NAMES, counters.cpu().tolist()))


def eval_prepare(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, stream=None):
    """gf_eval_prepare: the x-independent tables into a fresh device workspace (a uint8 tensor)."""
    n_ang = ang_nodes.numel()
    size = int(lib().gf_eval_workspace_size(ctypes.byref(params), n_rad, n_ang))
    if size < 0:
        raise GfError(2, lib().gf_last_error().decode())
    ws = torch.empty(size, dtype=torch.uint8, device=ang_nodes.device)
    with torch.cuda.device(ws.device):
        _check(lib().gf_eval_prepare(ctypes.byref(params), rad_nodes.data_ptr(), rad_weights.data_ptr(), n_rad,
                                     ang_nodes.data_ptr(), ang_weights.data_ptr(), n_ang, ws.data_ptr(),
                                     _stream(stream)))
    return ws


def eval_grid_prepared(params, n_rad, n_ang, workspace, x, out=None, stream=None):
    """gf_eval_grid_prepared: G at x from a workspace made by eval_prepare with the same params and orders."""
    assert x.is_cuda and x.dtype == torch.complex128 and x.is_contiguous()
    odt = torch.complex64 if params.precision == 32 else torch.complex128
    if out is None:
        out = torch.empty(x.shape, dtype=odt, device=x.device)
    assert out.dtype == odt and out.is_contiguous() and out.numel() == x.numel()
    with torch.cuda.device(x.device):
        _check(lib().gf_eval_grid_prepared(ctypes.byref(params), n_rad, n_ang, workspace.data_ptr(), x.data_ptr(),
                                           x.numel(), out.data_ptr(), None, _stream(stream)))
    return out


def eval_angular(params, x, ang_nodes, ang_weights, y, out=None, stream=None):
    """gf_eval_angular (paper Kernel 3): B(x, y) of eq. (22) for one complex x at every y (complex128 device tensor)."""
    assert y.is_cuda and y.dtype == torch.complex128 and y.is_contiguous()
    if out is None:
        out = torch.empty_like(y)
    x = complex(x)
    with torch.cuda.device(y.device):
        _check(lib().gf_eval_angular(ctypes.byref(params), x.real, x.imag, ang_nodes.data_ptr(), ang_weights.data_ptr(),
                                     ang_nodes.numel(), y.data_ptr(), y.numel(), out.data_ptr(), _stream(stream)))
    return out


def cut_crossings(params, x, n_z, out=None, stream=None):
    """gf_cut_crossings (paper Kernel 4): crossings of (0, Lambda^2] by the cut(s) of line 2, int32 per point of x."""
    assert x.is_cuda and x.dtype == torch.complex128 and x.is_contiguous()
    if out is None:
        out = torch.empty(x.shape, dtype=torch.int32, device=x.device)
    with torch.cuda.device(x.device):
        _check(lib().gf_cut_crossings(ctypes.byref(params), x.data_ptr(), x.numel(), int(n_z), out.data_ptr(),
                                      _stream(stream)))
    return out


def executed_fp64(info, counters):
    """(FP64-pipe thread-instructions, flops with FMA = 2) of one launch from its route counters."""
    units = (("near_pair", "near_pairs"), ("series_term", "series_terms"), ("exact_pair", "exact_pairs"),
             ("node_near", "near_nodes"), ("node_moment", "moment_nodes"), ("node_exact", "exact_nodes"),
             ("node_cheb", "cheb_nodes"), ("tail", "tails"), ("blk_series", "block_series"),
             ("blk_term", "block_series_terms"))
    inst = sum((info[u + "_dfma"] + info[u + "_other"]) * counters[c] for u, c in units)
    flops = sum((2 * info[u + "_dfma"] + info[u + "_other"]) * counters[c] for u, c in units)
    return float(inst), float(flops)


def _host_ptr(a):
    if isinstance(a, torch.Tensor):
        assert not a.is_cuda and a.is_contiguous()
        return a.data_ptr()
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def eval_grid_host(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, out, stream=None):
    """gf_eval_grid_host: every buffer is HOST memory (numpy arrays or CPU torch tensors, ideally pinned);
    host<->device copies happen inside the call, which returns after `out` is complete."""
    if not torch.cuda.is_available():
        raise GfError(4, "no CUDA device (no CPU fallback)")
    n_ang = int(ang_nodes.shape[0])
    n_points = int(np.prod(x.shape))
    # the library reads and writes these buffers by size alone: check what it cannot
    def _dt(a):
        return str(a.dtype).replace("torch.", "")
    need = radial_table_size(params.contour, n_rad)
    if need < 0:
        raise GfError(2, "bad contour / n_rad (deformed contours need n_rad % 8 == 0)")
    for name, t, n in (("rad_nodes", rad_nodes, need), ("rad_weights", rad_weights, need), ("ang_nodes", ang_nodes, n_ang),
                       ("ang_weights", ang_weights, n_ang)):
        if _dt(t) != "float64" or int(np.prod(t.shape)) < n:
            raise GfError(2, "eval_grid_host: %s must be float64 with at least %d entries" % (name, n))
    if int(np.prod(ang_weights.shape)) != n_ang:
        raise GfError(2, "eval_grid_host: ang_nodes and ang_weights differ in length")
    odt = "complex64" if params.precision == 32 else "complex128"
    if _dt(x) != "complex128":
        raise GfError(2, "eval_grid_host: x must be complex128")
    if _dt(out) != odt or int(np.prod(out.shape)) != n_points:
        raise GfError(2, "eval_grid_host: out must be %s with %d entries" % (odt, n_points))
    _check(lib().gf_eval_grid_host(ctypes.byref(params), _host_ptr(rad_nodes), _host_ptr(rad_weights), n_rad,
                                   _host_ptr(ang_nodes), _host_ptr(ang_weights), n_ang, _host_ptr(x),
                                   n_points, _host_ptr(out), _stream(stream)))
    return out


def launch_info(params, n_rad, n_ang, n_points):
    info = gf_launch_info()
    _check(lib().gf_eval_launch_info(ctypes.byref(params), n_rad, n_ang, n_points, ctypes.byref(info)))
    return {k: getattr(info, k) for k, _ in gf_launch_info._fields_}


def diag_fp64_peak(blocks, threads, iters, sink, stream=None):
    _check(lib().gf_diag_fp64_peak(blocks, threads, iters, sink.data_ptr(), _stream(stream)))


def diag_radial_map(cutoff2, map_scale, nodes, stream=None):
    y = torch.empty_like(nodes)
    _check(lib().gf_diag_radial_map(cutoff2, map_scale, nodes.data_ptr(), nodes.numel(), y.data_ptr(), _stream(stream)))
    return y


def diag_contour_nodes(params, n_rad, n_ang, workspace, rad_nodes, rad_weights, x, stream=None):
    """gf_diag_contour_nodes: (policy, y, wy) of the one point x under a deformed policy, from a prepared workspace."""
    x = complex(x)
    y = torch.empty(n_rad, dtype=torch.complex128, device=workspace.device)
    wy = torch.empty_like(y)
    pol = torch.zeros(1, dtype=torch.int32, device=workspace.device)
    with torch.cuda.device(workspace.device):
        _check(lib().gf_diag_contour_nodes(ctypes.byref(params), n_rad, n_ang, workspace.data_ptr(), rad_nodes.data_ptr(),
                                           rad_weights.data_ptr(), x.real, x.imag, pol.data_ptr(), y.data_ptr(),
                                           wy.data_ptr(), _stream(stream)))
    return int(pol.item()), y, wy


def diag_dfma_issue(mode, blocks, threads, iters, sink, stream=None):
    _check(lib().gf_diag_dfma_issue(mode, blocks, threads, iters, sink.data_ptr(), _stream(stream)))


def trim_scratch():
    _check(lib().gf_trim_scratch())


def version():
    return lib().gf_version().decode()
