"""ctypes wrapper of the CPU oracle (oracle/gf_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_1205_0752_b200 (the
CUDA path) and the CUDA path imports nothing from here.

Everything numerical happens in gf_oracle.cpp; this file only builds the shared
object with g++, marshals numpy arrays and mirrors the oracle's own parameter
struct.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gf_oracle.cpp")
_LIB = os.path.join(_HERE, "libgf_oracle.so")

QUAD = {"gauss_legendre": 0, "gauss_cheb2": 1, "tanh_sinh": 2, "gauss_cheb1": 3}
MEASURE = {"plain": 0, "sqrt1mz2": 1}
PROP = {"massive": 0, "rational": 1}
CONTOUR = {"real": 0, "ray_arc": 1, "thread": 2, "auto": 3}
SPACING = {"uniform": 0, "log_abs_im": 1}
# arithmetic variants of gfo_eval_grid: double terms + long double sums; all double (timed);
# long double terms and sums, binary128 for |x| < 2^-10 (parity: own rounding error << 1e-11
# everywhere, reading G18); binary128 everywhere (slow, checks "extended")
ACCUM = {"long_double": 0, "double": 1, "extended": 2, "quad": 3}


class _Prop(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("m2_re", ctypes.c_double), ("m2_im", ctypes.c_double),
                ("M2", ctypes.c_double), ("a", ctypes.c_double), ("b", ctypes.c_double)]


class _Params(ctypes.Structure):
    _fields_ = [("line_k", _Prop), ("line_pk", _Prop), ("cutoff2", ctypes.c_double),
                ("sub_re", ctypes.c_double), ("sub_im", ctypes.c_double),
                ("taylor_order", ctypes.c_int), ("prefactor", ctypes.c_double),
                ("map_scale", ctypes.c_double), ("contour", ctypes.c_int),
                ("precision", ctypes.c_int), ("routing", ctypes.c_int), ("dim", ctypes.c_double)]


def build(force=False):
    """Compile gf_oracle.cpp -> libgf_oracle.so (g++ -O2, no fast-math)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-pthread", "-o", _LIB, _SRC,
           "-lquadmath"]
    subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        assert _lib.gfo_params_size() == ctypes.sizeof(_Params)
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _prop(d):
    """d: {'kind': 'massive', 'm2': complex} or {'kind': 'rational', 'M2':.., 'a':.., 'b':..}"""
    p = _Prop()
    p.kind = PROP[d["kind"]]
    m2 = complex(d.get("m2", 0.0))
    p.m2_re, p.m2_im = m2.real, m2.imag
    p.M2, p.a, p.b = float(d.get("M2", 0.0)), float(d.get("a", 0.0)), float(d.get("b", 0.0))
    return p


def make_params(line_k, line_pk, cutoff2, prefactor=2.0 / np.pi, map_scale=1.0, contour="real",
                sub=0.0, taylor_order=0, precision=64, dim=4.0, routing="paper"):
    P = _Params()
    P.line_k, P.line_pk = _prop(line_k), _prop(line_pk)
    P.cutoff2 = float(cutoff2)
    s = complex(sub)
    P.sub_re, P.sub_im = s.real, s.imag
    P.taylor_order = int(taylor_order)
    P.prefactor = float(prefactor)
    P.map_scale = float(map_scale)
    P.contour = CONTOUR[contour]
    P.precision = int(precision)
    P.dim = float(dim)
    P.routing = {"paper": 0, "symmetric": 1}[routing]
    return P


def make_quadrature(kind, n, step=0.0, measure="plain"):
    x = np.empty(n, dtype=np.float64)
    w = np.empty(n, dtype=np.float64)
    rc = lib().gfo_make_quadrature(QUAD[kind], int(n), ctypes.c_double(step), MEASURE[measure],
                                   _dp(x), _dp(w))
    if rc:
        raise ValueError("gfo_make_quadrature failed: %d" % rc)
    return x, w


def make_quadrature_dim(kind, n, dim, step=0.0):
    """The rule for the angular measure (1 - z^2)^((dim-3)/2) dz of `dim` space-time dimensions."""
    x = np.empty(n, dtype=np.float64)
    w = np.empty(n, dtype=np.float64)
    rc = lib().gfo_make_quadrature_dim(QUAD[kind], int(n), ctypes.c_double(step), ctypes.c_double(dim), _dp(x), _dp(w))
    if rc:
        raise ValueError("gfo_make_quadrature_dim failed: %d" % rc)
    return x, w


def make_radial_pyramid(n_rad, levels=4, kind="gauss_legendre"):
    """Rules of order n_rad, n_rad/2, ... back to back ('n arrays')."""
    xs, ws = [], []
    n = n_rad
    for _ in range(levels):
        x, w = make_quadrature(kind, n)
        xs.append(x)
        ws.append(w)
        n //= 2
    return np.concatenate(xs), np.concatenate(ws)


def make_grid(re_min, re_max, n_re, im_min, im_max, n_im, spacing="uniform", im_abs_min=0.0):
    x = np.empty(n_im * n_re, dtype=np.complex128)
    rc = lib().gfo_make_grid(ctypes.c_double(re_min), ctypes.c_double(re_max), int(n_re),
                             ctypes.c_double(im_min), ctypes.c_double(im_max), int(n_im),
                             SPACING[spacing], ctypes.c_double(im_abs_min),
                             _dp(x.view(np.float64)))
    if rc:
        raise ValueError("gfo_make_grid failed: %d" % rc)
    return x.reshape(n_im, n_re)


def eval_grid(params, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, x, n_threads=0,
              accum="long_double"):
    """G at every point of x (any shape, complex128).  Returns (G, threads_used)."""
    xf = np.ascontiguousarray(np.asarray(x, dtype=np.complex128)).ravel()
    out = np.empty_like(xf)
    rn = np.ascontiguousarray(rad_nodes, dtype=np.float64)
    rw = np.ascontiguousarray(rad_weights, dtype=np.float64)
    an = np.ascontiguousarray(ang_nodes, dtype=np.float64)
    aw = np.ascontiguousarray(ang_weights, dtype=np.float64)
    used = ctypes.c_int(0)
    rc = lib().gfo_eval_grid(ctypes.byref(params), _dp(rn), _dp(rw), int(n_rad), _dp(an), _dp(aw),
                             int(an.size), _dp(xf.view(np.float64)), ctypes.c_longlong(xf.size),
                             _dp(out.view(np.float64)), int(n_threads),
                             ACCUM[accum], ctypes.byref(used))
    if rc:
        raise ValueError("gfo_eval_grid failed: %d" % rc)
    return out.reshape(np.shape(x)), used.value


def contour_nodes(params, x, rad_nodes, rad_weights, n_rad, n_ang):
    y = np.empty(2 * n_rad, dtype=np.complex128)
    wy = np.empty(2 * n_rad, dtype=np.complex128)
    n = ctypes.c_int(0)
    rn = np.ascontiguousarray(rad_nodes, dtype=np.float64)
    rw = np.ascontiguousarray(rad_weights, dtype=np.float64)
    x = complex(x)
    pol = lib().gfo_contour_nodes(ctypes.byref(params), ctypes.c_double(x.real),
                                  ctypes.c_double(x.imag), _dp(rn), _dp(rw), int(n_rad), int(n_ang),
                                  _dp(y.view(np.float64)), _dp(wy.view(np.float64)), ctypes.byref(n))
    if pol < 0:
        raise ValueError("gfo_contour_nodes failed")
    return pol, y[:n.value].copy(), wy[:n.value].copy()


def eval_angular(params, x, ang_nodes, ang_weights, y, terms="long_double"):
    """Paper Kernel 3: the angular integral B(x, y) of eq. (22) for one complex x at every complex y."""
    yf = np.ascontiguousarray(np.asarray(y, dtype=np.complex128)).ravel()
    out = np.empty_like(yf)
    an = np.ascontiguousarray(ang_nodes, dtype=np.float64)
    aw = np.ascontiguousarray(ang_weights, dtype=np.float64)
    x = complex(x)
    rc = lib().gfo_eval_angular(ctypes.byref(params), ctypes.c_double(x.real), ctypes.c_double(x.imag), _dp(an),
                                _dp(aw), int(an.size), _dp(yf.view(np.float64)), ctypes.c_longlong(yf.size),
                                _dp(out.view(np.float64)), {"double": 0, "long_double": 2, "binary128": 3}[terms])
    if rc:
        raise ValueError("gfo_eval_angular failed: %d" % rc)
    return out.reshape(np.shape(y))


def cut_crossings(params, x, n_z):
    """Paper Kernel 4: how often the cut(s) of line 2 cross (0, Lambda^2] of the real y-axis, per point of x."""
    xf = np.ascontiguousarray(np.asarray(x, dtype=np.complex128)).ravel()
    out = np.empty(xf.size, dtype=np.int32)
    rc = lib().gfo_cut_crossings(ctypes.byref(params), _dp(xf.view(np.float64)), ctypes.c_longlong(xf.size),
                                 int(n_z), out.ctypes.data_as(ctypes.POINTER(ctypes.c_int)))
    if rc:
        raise ValueError("gfo_cut_crossings failed: %d" % rc)
    return out.reshape(np.shape(x))
