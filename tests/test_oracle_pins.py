"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the plausible mistake it would catch.  Nothing here compares the
oracle with itself through the same formula: references are closed forms evaluated
with mpmath (tests/closed_forms.py), numpy's own Gauss-Legendre routine, exact
moments, and invariants.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import gf_workloads as W
from tests import closed_forms as CF
from tests import mp_reference as MPR

BUB = {"kind": "massive", "m2": 1.0}
RAT = {"kind": "rational", "M2": 2.0, "a": 0.5, "b": 1.2}
GOLD = os.path.join(os.path.dirname(__file__), "golden", "closed_form_samples.txt")


def relerr(g, ref):
    ref = np.asarray(ref, dtype=complex)
    g = np.asarray(g, dtype=complex)
    den = np.where(np.abs(ref) == 0, 1.0, np.abs(ref))
    return np.abs(g - ref) / den


def tables(O, n_rad, n_ang, ang="gauss_legendre", levels=4):
    rn, rw = O.make_radial_pyramid(n_rad, levels=levels)
    z, wz = O.make_quadrature(ang, n_ang, measure="sqrt1mz2")
    return rn, rw, z, wz


def G(O, xs, line_k=BUB, line_pk=BUB, cutoff2=1e6, n_rad=256, n_ang=128, ang="gauss_cheb2",
      contour="real", **kw):
    P = O.make_params(line_k, line_pk, cutoff2, contour=contour, **kw)
    rn, rw, z, wz = tables(O, n_rad, n_ang, ang)
    g, _ = O.eval_grid(P, rn, rw, n_rad, z, wz, np.asarray(xs, dtype=complex))
    return g


# ---------------------------------------------------------------- closed forms themselves
def test_closed_forms_match_survey_samples():
    """The mpmath closed forms reproduce the independently computed sample values."""
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        form, xr, xi, gr, gi = line.split()
        x = complex(float(xr), float(xi))
        if form == "CF1":
            v = CF.cf1(x)
        elif form == "CF2":
            v = CF.cf2_paper_eq18(x)
        else:
            v = CF.cf3_rational(x, 1.0, 2.0, 0.5, 1.2)
        assert abs(complex(v) - complex(float(gr), float(gi))) < 2e-10, (form, x)


def test_cf1_series_and_threshold():
    # small-x series -tau/6 + tau^2/60 - tau^3/420 and G(-4 m^2) = 2
    x = mp.mpf("1e-3")
    assert abs(CF.cf1(x) - (-x / 6 + x ** 2 / 60 - x ** 3 / 420)) < 1e-13
    assert abs(CF.cf1(-4) - 2) < 1e-25


# ---------------------------------------------------------------- quadrature tables (a2)
@pytest.mark.parametrize("n", [1, 2, 5, 32, 64, 255, 512])
def test_gauss_legendre_matches_numpy_and_is_exact(oracle, n):
    """Catches wrong roots/weights, ordering, asymmetry (A-S 25.4.29)."""
    x, w = oracle.make_quadrature("gauss_legendre", n)
    xr, wr = np.polynomial.legendre.leggauss(n)
    assert np.max(np.abs(x - xr)) < 4e-16
    assert np.max(np.abs(w - wr) / wr) < 1e-9   # numpy's own end weights are only ~1e-10 at n=512
    if n >= 2:  # 40-digit reference for a few nodes: weights to a few ulp
        mp40 = mp.mp.clone()
        mp40.dps = 40
        for k in sorted({0, 1, n // 3, (n - 1) // 2}):
            r = mp40.findroot(lambda t: mp40.legendre(n, t), mp40.mpf(float(x[k])), tol=1e-30)
            dpn = n * (r * mp40.legendre(n, r) - mp40.legendre(n - 1, r)) / (r * r - 1)
            wk = 2 / ((1 - r * r) * dpn * dpn)
            assert abs(r - float(x[k])) < 3e-16 and abs(wk - float(w[k])) / wk < 1e-14
    assert np.all(np.diff(x) > 0) or n == 1
    assert np.array_equal(x, -x[::-1]) and np.array_equal(w, w[::-1])
    for k in range(0, min(2 * n, 40), 2):  # exact for degree <= 2n-1
        assert abs(np.sum(w * x ** k) - 2.0 / (k + 1)) < 1e-14


@pytest.mark.parametrize("n", [3, 32, 128])
def test_cheb2_moments(oracle, n):
    """int sqrt(1-z^2) z^(2k) dz = pi (2k)! / (2^(2k+1) k! (k+1)!) exactly for 2k <= 2n-1."""
    z, w = oracle.make_quadrature("gauss_cheb2", n, measure="sqrt1mz2")
    for k in range(0, min(n, 12)):
        exact = math.pi * math.factorial(2 * k) / (2 ** (2 * k + 1) * math.factorial(k) * math.factorial(k + 1))
        assert abs(np.sum(w * z ** (2 * k)) - exact) < 1e-14
    zp, wp = oracle.make_quadrature("gauss_cheb2", n, measure="plain")
    assert np.allclose(wp * np.sqrt(1 - zp ** 2), w, rtol=1e-13)


def test_tanh_sinh_rule(oracle):
    """n = 49 (the paper's ndbl) with the default step integrates the d=4
    angular measure and a smooth integrand to ~1e-12 (reading G8)."""
    z, w = oracle.make_quadrature("tanh_sinh", 49, measure="sqrt1mz2")
    assert abs(np.sum(w) - math.pi / 2) < 1e-11
    a, b = 3.0, 1.0  # int sqrt(1-z^2)/(a - b z) dz = pi (a - sqrt(a^2-b^2)) / b^2
    assert abs(np.sum(w / (a - b * z)) - math.pi * (a - math.sqrt(a * a - b * b)) / b ** 2) < 1e-11
    zp, wp = oracle.make_quadrature("tanh_sinh", 49, measure="plain")
    assert abs(np.sum(wp * zp ** 2) - 2.0 / 3.0) < 1e-11
    assert np.array_equal(z, -z[::-1])


def test_angular_measure_of_gl(oracle):
    z, w = oracle.make_quadrature("gauss_legendre", 64, measure="sqrt1mz2")
    zp, wp = oracle.make_quadrature("gauss_legendre", 64, measure="plain")
    assert np.allclose(w, wp * np.sqrt(1 - zp ** 2), rtol=1e-14)


# ---------------------------------------------------------------- grid (a1)
def test_grid_uniform(oracle):
    """Endpoint-inclusive, re index fastest, exactly mirrored rows (reading G9)."""
    x = oracle.make_grid(-5.0, 1.0, 64, -2.0, 2.0, 64)
    assert x.shape == (64, 64)
    assert x[0, 0] == complex(-5, -2) and x[-1, -1] == complex(1, 2)
    assert np.max(np.abs(x[0].real - np.linspace(-5, 1, 64))) < 2e-15
    assert np.max(np.abs(x[:, 0].imag - np.linspace(-2, 2, 64))) < 2e-15
    assert np.array_equal(x[::-1].imag, -x.imag)          # rows j <-> N-1-j are conjugates
    assert np.all(x.imag != 0)                              # even N: Im x = 0 never occurs
    assert np.array_equal(x[3].real, x[40].real)
    one = oracle.make_grid(0.25, 9.0, 1, -1.0, 7.0, 1)
    assert one[0, 0] == complex(0.25, -1.0)


def test_grid_log_abs_im(oracle):
    """Config 5 (reading G10): ascending Im, 128 log-spaced |Im| per sign in [1e-6, 1e-3]."""
    x = oracle.make_grid(-10.0, -3.0, 16, -1e-3, 1e-3, 256, spacing="log_abs_im", im_abs_min=1e-6)
    im = x[:, 0].imag
    assert im[0] == -1e-3 and im[127] == -1e-6 and im[128] == 1e-6 and im[255] == 1e-3
    assert np.all(np.diff(im) > 0)
    assert np.array_equal(im[::-1], -im)
    ratio = im[129:] / im[128:-1]
    assert np.allclose(ratio, (1e3) ** (1 / 127), rtol=1e-12)
    with pytest.raises(ValueError):
        oracle.make_grid(-10.0, -3.0, 16, -1e-3, 1e-3, 255, spacing="log_abs_im", im_abs_min=1e-6)


# ---------------------------------------------------------------- the double sum vs closed forms
def test_cf1_tight_cheb2(oracle):
    """Pins measure (y dy, sqrt(1-z^2)), prefactor 2/pi, the shifted-log map and its Jacobian,
    the subtraction term and u = x+y-2 sqrt(x) sqrt(y) z, to 1e-10 (Chebyshev angular rule)."""
    xs = [0.5 + 0.2j, 1 + 2j, 0.3 - 0.1j, 1.5 + 0j, -0.5 + 0.5j, 1e-3 + 2e-3j, 1e-5 - 1e-5j]
    assert all(CF.in_parabola_R2(x) for x in xs)
    g = G(oracle, xs)
    ref = [complex(CF.cf1(x)) for x in xs]
    assert np.max(relerr(g, ref)) < 1e-10


def test_cf1_other_mass(oracle):
    """m^2 = 2.5 on both lines: catches a mass that is hard-wired to 1."""
    xs = [0.7 + 0.4j, 2 - 1j]
    m = {"kind": "massive", "m2": 2.5}
    g = G(oracle, xs, line_k=m, line_pk=m)
    assert np.max(relerr(g, [complex(CF.cf1(x, 2.5)) for x in xs])) < 1e-10


@pytest.mark.parametrize("name,tol", [("cfg1_tiny", 2e-4), ("cfg2_mid", 3e-6)])
def test_configs_vs_cf1_inside_parabola(oracle, name, tol):
    """Configs 1 and 2 as BASELINE.json states them (Gauss-Legendre angular rule, REAL contour)
    on the mask 'parabola R2 shrunk by 0.5' (measured: 1.03e-4 / 1.40e-6; with a shrink of 0.25
    the points next to the parabola reach 4.2e-4 / 5.3e-6); the bound is the GL angular
    quadrature error (reading G5)."""
    c = W.CONFIGS[name]
    x = oracle.make_grid(c["re"][0], c["re"][1], c["n_re"], c["im"][0], c["im"][1], c["n_im"])
    step = max(1, c["n_re"] // 48)
    xs = x[::step, ::step].ravel()
    xs = np.array([v for v in xs if CF.in_parabola_R2(v, shrink=0.5)])
    assert xs.size > 100
    g = G(oracle, xs, cutoff2=c["cutoff2"], n_rad=c["n_rad"], n_ang=c["n_ang"], ang="gauss_legendre")
    err = relerr(g, [complex(CF.cf1(v)) for v in xs])
    assert np.max(err) < tol
    assert np.max(err) > tol / 50   # the error really is the GL angular error, not something else


def test_cf2_paper_example(oracle):
    """The paper's worked example eq. (19)-(21) against its eq. (18) in
    region 1 (Re x > (Im x)^2 - 1/4).  Catches swapped lines / wrong sign of a complex mass."""
    k = {"kind": "massive", "m2": 0.5j}
    pk = {"kind": "massive", "m2": -0.5j}
    xs = [0.5 + 0.2j, 2 + 1j, 3 + 0j, 1 - 0.5j, 0.2 + 0.1j]
    assert all(x.real > x.imag ** 2 - 0.25 for x in xs)
    g = G(oracle, xs, line_k=k, line_pk=pk, cutoff2=1e8, n_rad=512)
    ref = [complex(CF.cf2_paper_eq18(x)) for x in xs]
    assert np.max(relerr(g, ref)) < 1e-10
    # a wrong sign of one mass is a different function (a line SWAP is not: invariant I4)
    g_wrong = G(oracle, xs, line_k=k, line_pk=k, cutoff2=1e8, n_rad=512)
    assert np.min(relerr(g_wrong, ref)) > 1e-2


def test_finite_cutoff_against_adaptive_integration(oracle):
    """eq. (14) at a SMALL cutoff, Lambda^2 = 50, where the two lines are
    distinguishable (O(Lambda^-4) = 1e-4): mpmath's adaptive integrator over y of the plain
    difference D1(y) [ <D2(u)> - <D2(y)> ], the angular average taken analytically,
    int sqrt(1-z^2)/(A - B z) dz = pi (A - sqrt(A^2-B^2))/B^2.  Pins which line carries which
    mass, the finite cutoff, and the radial map with its Jacobian."""
    ma, mb = 1.0, 3.0
    a, b = {"kind": "massive", "m2": ma}, {"kind": "massive", "m2": mb}
    xs = [0.5 + 0.2j, 1.0 - 0.3j]

    def direct(x, m1, m2_, lam2):
        x = mp.mpc(x)

        def f(y):
            A = x + y + m2_
            B2 = 4 * x * y
            ang_u = mp.pi * (A - A * mp.sqrt(1 - B2 / (A * A))) / B2
            ang_y = mp.pi / (2 * (y + m2_))
            return y / (y + m1) * (ang_u - ang_y)
        return 2 / mp.pi * mp.quad(f, [0, 1, 5, 20, lam2])

    g_ab = G(oracle, xs, line_k=a, line_pk=b, cutoff2=50.0, n_rad=256)
    g_ba = G(oracle, xs, line_k=b, line_pk=a, cutoff2=50.0, n_rad=256)
    ref_ab = [complex(direct(x, ma, mb, 50)) for x in xs]
    ref_ba = [complex(direct(x, mb, ma, 50)) for x in xs]
    assert np.max(relerr(g_ab, ref_ab)) < 1e-10 and np.max(relerr(g_ba, ref_ba)) < 1e-10
    assert np.min(relerr(g_ab, ref_ba)) > 1e-5      # the assignment matters at this cutoff


def test_cf3_rational_line(oracle):
    """Config 4's integrand (reading G11: line 2 rational) against the Feynman-parameter form
    on the REAL mask Re x >= 0.25, |Im x| <= 1.25."""
    xs = [0.5 + 0.2j, 1 + 1j, 2 - 1j, 0.3 + 0j]
    g = G(oracle, xs, line_pk=RAT, cutoff2=1e8, n_rad=512)
    ref = [complex(CF.cf3_rational(x, 1.0, 2.0, 0.5, 1.2)) for x in xs]
    assert np.max(relerr(g, ref)) < 1e-10
    # rational on line 1 instead (line swap): same G up to O(Lambda^-4)
    g_sw = G(oracle, xs, line_k=RAT, line_pk=BUB, cutoff2=1e8, n_rad=512)
    assert np.max(relerr(g_sw, ref)) < 1e-10


def test_cf3_unequal_real_masses(oracle):
    a, b = {"kind": "massive", "m2": 1.0}, {"kind": "massive", "m2": 3.0}
    xs = [0.5 + 0.2j, 2 + 0.5j]
    g = G(oracle, xs, line_k=a, line_pk=b, cutoff2=1e8, n_rad=512)
    ref = [complex(CF.cf3_feynman(x, 1.0, 3.0)) for x in xs]
    assert np.max(relerr(g, ref)) < 1e-10


# ---------------------------------------------------------------- invariants
def test_I1_G_of_zero_is_exactly_zero(oracle):
    for contour in ["real", "ray_arc"]:
        g = G(oracle, [0j], contour=contour, ang="gauss_legendre")
        assert g[0] == 0
    assert G(oracle, [0j], line_pk=RAT)[0] == 0


def test_I2_conjugation_symmetry_bitwise(oracle):
    """G(conj x) = conj G(x) bitwise for real-coefficient propagators (real tables, principal sqrt)."""
    xs = np.array([0.5 + 0.2j, -3 + 0.5j, 2 - 4j, -7 + 1e-3j, 1e-4 + 3j])
    for kw in [dict(), dict(line_pk=RAT), dict(contour="ray_arc"), dict(contour="auto")]:
        g = G(oracle, xs, ang="gauss_legendre", **kw)
        gc = G(oracle, np.conj(xs), ang="gauss_legendre", **kw)
        assert np.array_equal(gc, np.conj(g)), kw


def test_I2_complex_masses_swap_under_conjugation(oracle):
    k = {"kind": "massive", "m2": 0.5j}
    pk = {"kind": "massive", "m2": -0.5j}
    xs = np.array([0.5 + 0.2j, 2 + 1j])
    g = G(oracle, xs, line_k=k, line_pk=pk)
    gc = G(oracle, np.conj(xs), line_k=pk, line_pk=k)
    assert np.array_equal(gc, np.conj(g))


def test_I3_cutoff_independence(oracle):
    """BPHZ subtraction makes the result cutoff independent: error ~ Lambda^-4."""
    x = [0.5 + 0.2j]
    ref = complex(CF.cf1(x[0]))
    e4 = relerr(G(oracle, x, cutoff2=1e4), [ref])[0]
    e6 = relerr(G(oracle, x, cutoff2=1e6), [ref])[0]
    e8 = relerr(G(oracle, x, cutoff2=1e8, n_rad=512), [ref])[0]
    assert 1e-8 < e4 < 1e-7 and e6 < 2e-11 and e8 < 1e-12
    assert 5e3 < e4 / max(e6, 1e-30) < 2e4 or e6 < 5e-12  # ~ (1e6/1e4)^2 = 1e4


def test_I4_line_swap(oracle):
    """k <-> p-k (shift invariance of eq. (4)): unequal masses, O(Lambda^-4)."""
    a, b = {"kind": "massive", "m2": 1.0}, {"kind": "massive", "m2": 3.0}
    xs = [0.5 + 0.2j, 1 + 1j]
    g1 = G(oracle, xs, line_k=a, line_pk=b, cutoff2=1e8, n_rad=512)
    g2 = G(oracle, xs, line_k=b, line_pk=a, cutoff2=1e8, n_rad=512)
    assert np.max(relerr(g1, g2)) < 1e-11


def test_I5_rule_independence(oracle):
    """The paper's own check: tanh-sinh vs Gauss-Chebyshev angular integration."""
    xs = [0.5 + 0.2j, 1 + 2j]
    g_ch = G(oracle, xs, ang="gauss_cheb2", n_ang=128)
    g_ts = G(oracle, xs, ang="tanh_sinh", n_ang=49)
    g_gl = G(oracle, xs, ang="gauss_legendre", n_ang=128)
    assert np.max(relerr(g_ts, g_ch)) < 1e-10
    assert 1e-7 < np.max(relerr(g_gl, g_ch)) < 3e-6


def test_I6_brute_force_high_order(oracle):
    """2048 x 1024 Chebyshev nodes, Lambda^2 = 1e8, 8x8 grid: <= 1e-12 inside the masks."""
    re, im = np.meshgrid(np.linspace(0.1, 2.0, 8), np.linspace(-1.0, 1.0, 8))
    xs = (re + 1j * im).ravel()
    g = G(oracle, xs, cutoff2=1e8, n_rad=2048, n_ang=1024)
    ref = [complex(CF.cf1(x)) for x in xs]
    assert np.max(relerr(g, ref)) < 1e-12


def test_accum_variants_agree(oracle):
    P = oracle.make_params(BUB, BUB, 1e6)
    rn, rw, z, wz = tables(oracle, 256, 128)
    xs = np.array([0.5 + 0.2j, -3 + 0.5j, 2e-3 + 1e-3j])
    g_ld, _ = oracle.eval_grid(P, rn, rw, 256, z, wz, xs, accum="long_double")
    g_d, _ = oracle.eval_grid(P, rn, rw, 256, z, wz, xs, accum="double", n_threads=2)
    assert np.max(relerr(g_d, g_ld)) < 1e-12


@pytest.mark.parametrize("x", [5.551115123125783e-17 + 1.1102230246251565e-16j, 1e-9 - 3e-10j, -7e-4 + 2e-4j,
                               1.2e-3 + 0j, 0.3 - 0.1j, -1.3112 - 1.6986j])
def test_parity_variant_rounding_error_is_negligible(oracle, x):
    """Reading G18: the variant GPU parity is measured against carries << 1e-11 of its own error, also
    at tiny |x| (where the +-z terms cancel; binary128 below |x| = 2^-10) and next to a zero of a
    denominator (x = -1.3112 - 1.6986i, outside the parabola R2)."""
    P = oracle.make_params(BUB, BUB, 1e4)
    rn, rw = oracle.make_quadrature("gauss_legendre", 24)
    z, wz = oracle.make_quadrature("gauss_cheb2", 33, measure="sqrt1mz2")
    ref = MPR.finite_sum(oracle, P, x, rn, rw, 24, z, wz, digits=60)
    g, _ = oracle.eval_grid(P, rn, rw, 24, z, wz, np.array([x]), accum="extended")
    assert relerr(g, [ref])[0] < 2e-14
    gq, _ = oracle.eval_grid(P, rn, rw, 24, z, wz, np.array([x]), accum="quad")
    assert relerr(gq, [ref])[0] < 1e-15


@pytest.mark.parametrize("case", ["rational_real", "rational_ray_arc", "bubble_ray_arc", "bubble_thread",
                                  "bubble_ray_arc_near_axis"])
def test_parity_variants_on_rational_lines_and_deformed_contours(oracle, case):
    """The same check off the REAL contour and for a rational line 2: the `extended` and `quad` term variants share
    one template with the massive REAL case, these instances of it are pinned to the 60-digit sum of the definition
    too (complex nodes, the rational form of prop_diff)."""
    lp, contour, x = {"rational_real": (RAT, "real", -2.0 + 3.0j), "rational_ray_arc": (RAT, "ray_arc", -1.5 + 2.5j),
                      "bubble_ray_arc": (BUB, "ray_arc", 2.0 - 4.0j), "bubble_thread": (BUB, "thread", -6.0 + 1e-3j),
                      "bubble_ray_arc_near_axis": (BUB, "ray_arc", -3.0 + 0.05j)}[case]
    P = oracle.make_params(BUB, lp, 1e4, contour=contour)
    rn, rw = oracle.make_radial_pyramid(32, levels=4)
    z, wz = oracle.make_quadrature("gauss_cheb2", 33, measure="sqrt1mz2")
    ref = MPR.finite_sum(oracle, P, x, rn, rw, 32, z, wz, digits=60)
    g, _ = oracle.eval_grid(P, rn, rw, 32, z, wz, np.array([x]), accum="extended")
    assert relerr(g, [ref])[0] < 1e-13, (g, ref)
    gq, _ = oracle.eval_grid(P, rn, rw, 32, z, wz, np.array([x]), accum="quad")
    assert relerr(gq, [ref])[0] < 1e-15, (gq, ref)


# ---------------------------------------------------------------- contours (a3)
def test_real_contour_fails_outside_parabola(oracle):
    """R2: outside the parabola the REAL sum is NOT the continuation."""
    x = [2 - 4j]
    assert not CF.in_parabola_R2(x[0])
    assert relerr(G(oracle, x), [complex(CF.cf1(x[0]))])[0] > 0.03


def test_ray_arc_reaches_outside_parabola(oracle):
    """Generalised region-2/5 contour reproduces CF1 where REAL cannot."""
    xs = [2 - 4j, -3 + 2j, -8 + 4j, 0.5 + 0.2j, -1 + 3j, 4 + 6j]
    g = G(oracle, xs, contour="ray_arc")
    assert np.max(relerr(g, [complex(CF.cf1(x)) for x in xs])) < 2e-9


def test_contour_geometry(oracle):
    """Every policy connects 0 with Lambda^2: sum of (weight x dy/dt) = Lambda^2 (up to the
    quadrature error of integrating dy/dt), and the node counts follow the pyramid."""
    rn, rw = oracle.make_radial_pyramid(256)
    for contour, x in [("real", 1 + 1j), ("ray_arc", -3 + 2j), ("thread", -6 + 0.1j), ("thread", -6 - 0.1j)]:
        P = oracle.make_params(BUB, BUB, 1e6, contour=contour)
        pol, y, wy = oracle.contour_nodes(P, x, rn, rw, 256, 128)
        assert y.size == 256
        assert abs(np.sum(wy) - 1e6) / 1e6 < 1e-9
    P = oracle.make_params(BUB, BUB, 1e6, contour="ray_arc")
    _, y, _ = oracle.contour_nodes(P, -3 + 2j, rn, rw, 256, 128)
    assert np.allclose(np.angle(y[:128]), np.angle(-3 + 2j))        # the ray
    assert np.allclose(np.abs(y[128:192]), np.abs(y[128]))          # the arc
    assert np.all(y[192:].imag == 0) and y[-1].real < 1e6           # the real tail


def test_auto_policy_regions(oracle):
    """AUTO's four tests in their order (include/gf.h, gf_contour), on both sides of each boundary."""
    rn, rw = oracle.make_radial_pyramid(64)
    P = oracle.make_params(BUB, BUB, 1e6, contour="auto")
    pol = lambda x: oracle.contour_nodes(P, x, rn, rw, 64, 128)[0]
    assert pol(1 + 1j) == 0 and pol(2 + 2.2j) == 0         # 1. inside the half-size parabola Re x > (Im x)^2/2 - 1/2: REAL
    assert pol(2 + 2.3j) == 1 and pol(0 + 1.1j) == 1      #    just outside it: RAY_ARC
    assert pol(-0.5 + 0.001j) == 0 and pol(-0.9 - 0.01j) == 0   # 2. next to the negative axis inside the parabola: REAL
    assert pol(-0.5 + 0.7j) == 1                           #    |Im x| n_rad >= 80 |Re x|: not "next to the axis"
    assert pol(-3 + 2j) == 1                               # 4. RAY_ARC outside the wedge
    assert pol(-6 + 0.01j) == 2 and pol(-6 - 0.01j) == 2   # 3. THREAD near the cut
    assert pol(-3 + 0.01j) == 0                            #    REAL in the strip -4.1 < Re x < -1 (the limitation)
    # a line THREAD does not apply to: REAL inside the wedge
    Pr = oracle.make_params(BUB, RAT, 1e6, contour="auto")
    assert oracle.contour_nodes(Pr, -6 + 0.01j, rn, rw, 64, 128)[0] == 0


def test_auto_is_the_continuation_where_the_header_says(oracle):
    """AUTO against the closed form CF1 over the analytic region of config 2's box (no test pinned AUTO):
    REAL inside the parabola is exact to the quadrature; RAY_ARC and THREAD reproduce CF1 away from the negative
    axis; the one region that is NOT the continuation is case 3 with REAL (the strip next to the negative axis
    between the parabola and -4.1 m^2), exactly as include/gf.h states."""
    n_rad, n_ang = 256, 128
    re, im = np.linspace(-10, 2, 49), np.linspace(-4, 4, 33)
    xs = (re[None, :] + 1j * im[:, None]).ravel()
    xs = xs[xs.imag != 0]
    P = oracle.make_params(BUB, BUB, 1e6, contour="auto")
    rn, rw = oracle.make_radial_pyramid(n_rad, levels=4)
    z, wz = oracle.make_quadrature("gauss_cheb2", n_ang, measure="sqrt1mz2")
    g, _ = oracle.eval_grid(P, rn, rw, n_rad, z, wz, xs)
    err = relerr(g, [complex(CF.cf1(v)) for v in xs])
    pol = np.array([oracle.contour_nodes(P, v, rn, rw, n_rad, n_ang)[0] for v in xs])
    inside = np.array([CF.in_parabola_R2(v) for v in xs])
    assert (pol == 0).sum() > 100 and (pol == 1).sum() > 900 and (pol == 2).sum() > 300
    assert err[(pol == 0) & inside].max() < 1e-10                       # REAL where it is the continuation
    strip = (pol == 0) & ~inside                                        # the documented limitation
    assert strip.sum() > 0 and np.all((xs[strip].real < -1) & (xs[strip].real > -4.1) & (np.abs(xs[strip].imag) <= 0.5))
    assert err[strip].min() > 0.5
    far = np.abs(xs.imag) >= 0.5                                        # rays and threads away from the axis
    assert err[(pol == 1) & far].max() < 2e-3 and err[(pol == 2)].max() < 3e-2
    assert np.median(err[pol == 1]) < 1e-8
    # the three points ADVICE r1 lists (x = -0.5, -0.5 + 0.0078i, -0.5 + 0.03i: RAY_ARC was off by 2 ... 5e3 there)
    xa = np.array([-0.5 + 1e-9j, -0.5 + 0.0078j, -0.5 + 0.03j])
    ga, _ = oracle.eval_grid(P, rn, rw, n_rad, z, wz, xa)
    assert relerr(ga, [complex(CF.cf1(v)) for v in xa]).max() < 1e-9


def test_contour_ladder_and_arc(oracle):
    """The radius of a deformed contour is the smallest rung of {2^k, 1.5 2^k} above 1.5 (sqrt|x| + sqrt(|x|+sc))^2
    (Lambda^2/2 beyond the ladder), the ray runs along x/|x|, and the rational arc ends where the ray ends and on
    the real axis, at the angles 4 atan(tau v) (compared with the angle form it replaces)."""
    rn, rw = oracle.make_radial_pyramid(256)
    P = oracle.make_params(BUB, BUB, 1e6, contour="ray_arc")
    rungs = sorted([2.0 ** k for k in range(-4, 22)] + [1.5 * 2.0 ** k for k in range(-4, 22)])
    for x in [-3 + 2j, 1e-3 + 1e-3j, 40 - 90j, -7 + 1e-7j, 0.2 - 0.1j, 2500 + 1j]:
        _, y, wy = oracle.contour_nodes(P, x, rn, rw, 256, 128)
        q = math.sqrt(abs(x)) + math.sqrt(abs(x) + 1.0)
        want = min(r for r in rungs if r >= 1.5 * q * q * (1 - 1e-15))
        R = abs(y[128])
        assert abs(R - want) <= 2e-15 * want, (x, R, want)
        assert np.max(np.abs(y[:128] / np.abs(y[:128]) - x / abs(x))) < 4e-16          # the ray's direction
        th = np.angle(y[128:192])
        u = 0.5 * (rn[256 + 128:256 + 192] + 1.0)
        tau = math.tan(np.angle(x) / 4)
        assert np.max(np.abs(th - 4 * np.arctan(tau * (1 - u)))) < 1e-14               # arc: theta = 4 atan(tau v), v = 1 - u
        dth = -4 * tau / (1 + (tau * (1 - u)) ** 2)                                     # d theta/du
        assert np.max(np.abs(wy[128:192] / (1j * y[128:192] * dth * 0.5 * rw[256 + 128:256 + 192]) - 1)) < 1e-14
        assert np.max(np.abs(np.abs(y[128:192]) / want - 1)) < 2e-15
        assert y[192].real > want and np.all(np.diff(y[192:].real) > 0)                    # real tail starts at R
        assert abs(np.sum(wy) - 1e6) / 1e6 < 1e-9
    # beyond the ladder / the cutoff: Lambda^2/2
    P2 = oracle.make_params(BUB, BUB, 30.0, contour="ray_arc")
    _, y, _ = oracle.contour_nodes(P2, -6 + 2j, rn, rw, 256, 128)
    assert abs(abs(y[128]) - 15.0) < 1e-14


def test_thread_contour_and_discontinuity(oracle):
    """Analogue of the paper's region-3/4 polylines.  Moderately close to the
    cut it matches CF1; very close it reproduces the discontinuity -2 pi i sqrt(1-4/s) within 20%."""
    g = G(oracle, [-6 + 1j, -8 + 0.5j], contour="thread", n_rad=1024, n_ang=512, ang="gauss_legendre")
    ref = [complex(CF.cf1(-6 + 1j)), complex(CF.cf1(-8 + 0.5j))]
    assert np.max(relerr(g, ref)) < 1e-4
    for s in [5.0, 7.0, 10.0]:
        gp, gm = G(oracle, [-s + 1e-4j, -s - 1e-4j], contour="thread", n_rad=1024, n_ang=512,
                   ang="gauss_legendre")
        exact = math.pi * math.sqrt(1 - 4 / s)
        assert gp.imag < 0 < gm.imag                       # sign of Im G opposite to sign of Im x
        assert abs(-gp.imag / exact - 1) < 0.2 and abs(gm.imag / exact - 1) < 0.2
    # under REAL the strip shows no cut at all
    gp, gm = G(oracle, [-6 + 1e-4j, -6 - 1e-4j], contour="real", n_rad=1024, n_ang=512, ang="gauss_legendre")
    assert abs(gp.imag) < 1e-2


# ---------------------------------------------------------------- argument checks
def test_oracle_rejects_unsupported(oracle):
    rn, rw, z, wz = tables(oracle, 64, 32)
    xs = np.array([1 + 1j])
    with pytest.raises(ValueError):
        oracle.eval_grid(oracle.make_params(BUB, BUB, 1e6, taylor_order=5), rn, rw, 64, z, wz, xs)
    with pytest.raises(ValueError):
        oracle.eval_grid(oracle.make_params(BUB, BUB, -1.0), rn, rw, 64, z, wz, xs)
    with pytest.raises(ValueError):
        oracle.eval_grid(oracle.make_params(BUB, RAT, 1e6, contour="thread"), rn, rw, 64, z, wz, xs)
    g, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e6), rn, rw, 64, z, wz, np.zeros(0, dtype=complex))
    assert g.size == 0


# ---------------------------------------------------------------- paper Kernels 3 and 4
@pytest.mark.parametrize("mu", [1.0, -0.5j])
def test_kernel3_angular_integral_closed_form(oracle, mu):
    """B(x, y) of eq. (22) with the Gauss rule of the measure against the textbook angular integral,
    for the bubble and for the paper's line 2 (mass^2 -i/2), at complex y off the cut.  Catches a wrong sign of d,
    a missing factor (y + mu), a wrong branch of sqrt(y)."""
    P = oracle.make_params({"kind": "massive", "m2": 1.0}, {"kind": "massive", "m2": mu}, 1e6)
    z, wz = oracle.make_quadrature("gauss_cheb2", 256, measure="sqrt1mz2")
    for x in (1.0 + 2.0j, 0.3 - 0.2j, 2.5):
        ys = np.array([0.3 + 0.2j, 2.0 - 1.0j, 5.0 + 0.5j, -2 + 6j, 10.0, 0.01, -4 - 4j])
        B = oracle.eval_angular(P, x, z, wz, ys)
        ref = np.array([complex(CF.angular_B_massive(x, y, mu)) for y in ys])
        assert relerr(B, ref).max() < 1e-12, (x, relerr(B, ref))
    # x = 0: the integrand vanishes identically (the factor d of eq. (20))
    assert np.all(oracle.eval_angular(P, 0.0, z, wz, np.array([1.0 + 1j, 3.0])) == 0)


def test_kernel3_binary128_variant_at_large_ratio(oracle):
    """The binary128 term variant (the reference Kernel 3's GPU parity uses) where the other variants run out of digits:
    |y/x| = 1e6 and 1e-6, where the +-z terms cancel by 2 sqrt(|y/x|) and the leading moment by another 1e7.  Against
    the definition sum_j w'_j [D2(u_j) - D2(y)]/D2(y) on the same tables at 60 digits, and (looser: the tables are
    rounded to double, which moves a sum that cancels by 1e12) against the textbook angular integral."""
    P = oracle.make_params(BUB, BUB, 1e6)
    z, wz = oracle.make_quadrature("gauss_cheb2", 512, measure="sqrt1mz2")
    for x, ys in ((1.0 + 0.5j, np.array([1e6 + 2e5j, -3e5 + 1e6j])), (2e5 - 1e6j, np.array([1.0 + 0.3j, 0.2 - 0.9j]))):
        B = oracle.eval_angular(P, x, z, wz, ys, terms="binary128")
        with mp.workdps(60):
            ref, cf = [], []
            for y in ys:
                xm, ym = mp.mpc(x), mp.mpc(complex(y))
                b2 = 2 * mp.sqrt(xm) * mp.sqrt(ym)
                D2 = lambda u: 1 / (u + 1)
                ref.append(complex(mp.fsum(mp.mpf(float(w)) * (D2(xm + ym - b2 * mp.mpf(float(t))) - D2(ym)) / D2(ym)
                                           for t, w in zip(z, wz))))
                cf.append(complex(CF.angular_B_massive(x, y, 1.0)))
        assert relerr(B, ref).max() < 1e-15, (x, relerr(B, ref))
        assert relerr(B, cf).max() < 1e-8, (x, relerr(B, cf))
        if abs(x) < 10:   # |y/x| = 1e6: the double variant is not good enough there, which is why binary128 exists
            Bd = oracle.eval_angular(P, x, z, wz, ys, terms="double")
            assert relerr(Bd, ref).max() > 1e-9


def test_kernel3_is_the_inner_sum_of_the_scan(oracle):
    """G(x) = c0 sum_i Wr_i y_i D1(y_i) D2(y_i) B(x, y_i): the scan rebuilt from Kernel 3 on the nodes of its own
    contour (deformed ones included) -- ties B's normalisation to the pinned G, for a massive and a rational line 2."""
    n_rad, n_ang = 64, 32
    for lpk, contour in ((BUB, "real"), (RAT, "real"), (BUB, "ray_arc")):
        P = oracle.make_params(BUB, lpk, 1e4, contour=contour)
        rn, rw, z, wz = tables(oracle, n_rad, n_ang, "gauss_legendre")
        for x in (0.5 + 0.2j, -3.0 + 1.5j):
            _, y, wy = oracle.contour_nodes(P, x, rn, rw, n_rad, n_ang)
            B = oracle.eval_angular(P, x, z, wz, y)
            d1 = 1.0 / (y + 1.0)
            d2 = 1.0 / (y + 1.0) if lpk is BUB else (y + RAT["M2"]) / (y * y + RAT["a"] * y + RAT["b"])
            g = P.prefactor * np.sum(wy * y * d1 * d2 * B)
            ref, _ = oracle.eval_grid(P, rn, rw, n_rad, z, wz, np.array([x]))
            assert abs(g - ref[0]) <= 1e-13 * abs(ref[0])


def test_kernel4_obstruction_is_the_parabola(oracle):
    """The set where the cut leaves the positive real y-axis free is 'a parabola-shaped region on the right'
    (PAPER.md:270): Re x > (Im x)^2/(4 m^2) - m^2 for a real mass (reading R2, from eq. (23)), and
    Re x > (Im x)^2 - 1/4 for the paper's line 2 with mass^2 -i/2.  Away from the boundary by 1e-9 every point of
    a grid must agree.  Catches a wrong branch continuation of eq. (25), a wrong sign test, an off-by-one in z."""
    re, im = np.linspace(-6, 3, 91), np.linspace(-4, 4, 81)
    X = re[None, :] + 1j * im[:, None]
    for m2 in (1.0, 0.25, 2.5):
        P = oracle.make_params(BUB, {"kind": "massive", "m2": m2}, 1e6)
        c = oracle.cut_crossings(P, X, 2001)
        margin = X.real - (X.imag ** 2 / (4 * m2) - m2)
        far = np.abs(margin) > 1e-9
        assert np.array_equal((c == 0)[far], (margin > 0)[far])
        assert set(np.unique(c)) <= {0, 1}
    P = oracle.make_params({"kind": "massive", "m2": 0.5j}, {"kind": "massive", "m2": -0.5j}, 1e6)
    c = oracle.cut_crossings(P, X, 2001)
    margin = X.real - (X.imag ** 2 - 0.25)
    far = np.abs(margin) > 1e-9
    assert np.array_equal((c == 0)[far], (margin > 0)[far])


def test_kernel4_respects_the_cutoff_and_counts_both_poles(oracle):
    """A crossing beyond Lambda^2 does not obstruct [0, Lambda^2]; a rational line 2 has one cut per pole."""
    x = np.array([-5.0 + 1.0j])
    big = oracle.make_params(BUB, BUB, 1e6)
    assert oracle.cut_crossings(big, x, 4001)[0] == 1
    # where it crosses: y0 real with (x + y0 + 1)^2 = 4 x y0 t, some t in [0,1]; locate it by bisection on the count
    lo, hi = 1e-3, 1e6
    for _ in range(60):
        mid = math.sqrt(lo * hi)
        if oracle.cut_crossings(oracle.make_params(BUB, BUB, mid), x, 4001)[0]:
            hi = mid
        else:
            lo = mid
    y0 = hi
    A = x[0] + y0 + 1.0
    t = A * A / (4 * x[0] * y0)          # zeta at the crossing must lie on [0, 1]
    assert abs(t.imag) < 1e-3 and -1e-3 < t.real < 1 + 1e-3
    P = oracle.make_params(BUB, RAT, 1e6)
    for xx in (-3.0 + 0.3j, 1.0 + 3.0j, 2.0 + 0.1j):
        total = oracle.cut_crossings(P, np.array([xx]), 4001)[0]
        parts = 0
        for u, _ in CF.rational_poles(RAT["M2"], RAT["a"], RAT["b"]):
            Pm = oracle.make_params(BUB, {"kind": "massive", "m2": complex(-u)}, 1e6)
            parts += oracle.cut_crossings(Pm, np.array([xx]), 4001)[0]
        assert total == parts


# ---------------------------------------------------------------- other dimensions
def test_dimension_3_bubble_closed_form(oracle):
    """d = 3: radial measure dy y^(1/2), angular measure dz (plain Gauss-Legendre), c0 = 1/(8 pi^2), against
    arctan(sqrt(x)/2m)/(4 pi sqrt(x)) - 1/(8 pi m) inside the parabola R2.  The sqrt(y) end-point behaviour makes the
    log-mapped Gauss-Legendre rule converge only algebraically (measured ~ n^-2.7), hence the tolerance and the
    convergence check.  Catches a wrong power of y (d = 4's y would be off by O(1)), a wrong angular measure."""
    xs = np.array([0.5 + 0.2j, 1 + 2j, 3.0, -0.5 + 0.3j, 1e-6])
    ref = np.array([complex(CF.bubble_d3(x)) for x in xs])
    errs = []
    for cutoff2, n_rad in ((1e8, 512), (1e10, 1024)):
        P = oracle.make_params(BUB, BUB, cutoff2, prefactor=1 / (8 * np.pi ** 2), dim=3.0)
        rn, rw = oracle.make_quadrature("gauss_legendre", n_rad)
        z, wz = oracle.make_quadrature("gauss_legendre", 64, measure="plain")
        g, _ = oracle.eval_grid(P, rn, rw, n_rad, z, wz, xs)
        errs.append(relerr(g, ref).max())
        g0, _ = oracle.eval_grid(P, rn, rw, n_rad, z, wz, np.array([0.0]))
        assert g0[0] == 0
    assert errs[0] < 2e-6 and errs[1] < errs[0] / 3
    # with d = 4's measure the same call is far off: the parameter is really used
    P4 = oracle.make_params(BUB, BUB, 1e8, prefactor=1 / (8 * np.pi ** 2))
    rn, rw = oracle.make_quadrature("gauss_legendre", 512)
    z, wz = oracle.make_quadrature("gauss_legendre", 64, measure="plain")
    g4, _ = oracle.eval_grid(P4, rn, rw, 512, z, wz, xs)
    assert relerr(g4, ref).min() > 0.1


def test_dimension_3_on_the_deformed_contours(oracle):
    """y^((d-2)/2) at complex y, on the branch continued along the contour from y = 0 (reading G21): with it RAY_ARC and
    AUTO reach the d = 3 closed form outside the parabola where the REAL contour is off by 20-180 %, and THREAD reaches
    it below -4 m^2 next to the cut, where its pieces W2 -> W3 -> W4 dip under the negative real axis and arg y runs
    past pi (a principal-branch power there flips the sign of those pieces: O(1) error).  Catches a wrong branch, a
    missing power on a piece, the d = 4 measure left in a table."""
    z, wz = oracle.make_quadrature("gauss_legendre", 64, measure="plain")
    c0 = 1 / (8 * np.pi ** 2)
    xs = np.array([2 - 4j, -3 + 2j, 0.5 + 0.2j, -0.5 + 0.3j])
    ref = np.array([complex(CF.bubble_d3(x)) for x in xs])
    rn, rw = oracle.make_radial_pyramid(512, levels=4)
    for contour in ("ray_arc", "auto"):
        g, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e8, prefactor=c0, dim=3.0, contour=contour), rn, rw, 512, z, wz, xs)
        assert relerr(g, ref).max() < 1e-6, (contour, relerr(g, ref))
    g, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e8, prefactor=c0, dim=3.0), rn, rw, 512, z, wz, xs[:2])
    assert relerr(g, ref[:2]).min() > 0.1                      # REAL is not the continuation there
    zt, wzt = oracle.make_quadrature("gauss_legendre", 256, measure="plain")
    xt = np.array([-6 + 1j, -6 - 1j, -8 + 0.5j])
    reft = np.array([complex(CF.bubble_d3(x)) for x in xt])
    gt, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e8, prefactor=c0, dim=3.0, contour="thread"), rn, rw, 512, zt, wzt, xt)
    assert relerr(gt, reft).max() < 2e-3, relerr(gt, reft)
    assert np.allclose(gt[1], np.conj(gt[0]), rtol=1e-13)
    # d = 5 (p = 3/2): no closed form at hand; the contour must not matter where both are the continuation
    P5r = oracle.make_params(BUB, BUB, 1e6, prefactor=c0, dim=5.0, taylor_order=1)
    P5c = oracle.make_params(BUB, BUB, 1e6, prefactor=c0, dim=5.0, taylor_order=1, contour="ray_arc")
    z5, wz5 = oracle.make_quadrature_dim("gauss_legendre", 128, 5.0)
    xin = np.array([0.5 + 0.2j, 1.0 + 0.5j])
    a, _ = oracle.eval_grid(P5r, rn, rw, 512, z5, wz5, xin)
    b, _ = oracle.eval_grid(P5c, rn, rw, 512, z5, wz5, xin)
    assert relerr(b, a).max() < 1e-4, relerr(b, a)


def test_dimension_argument_checks(oracle):
    rn, rw, z, wz = tables(oracle, 64, 32)
    with pytest.raises(ValueError):
        oracle.eval_grid(oracle.make_params(BUB, BUB, 1e4, dim=0.5), rn, rw, 64, z, wz, np.array([1.0]))
    g4, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e4, dim=4.0), rn, rw, 64, z, wz, np.array([1.0 + 1j]))
    g0, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e4, dim=0.0), rn, rw, 64, z, wz, np.array([1.0 + 1j]))
    assert g4[0] == g0[0]


# ---------------------------------------------------------------- symmetric momentum routing
def test_symmetric_routing_reaches_the_threshold_parabola(oracle):
    """Lines carrying k + p/2 and k - p/2 (shift invariance of eq. (4)): the same G as CF1 up to
    O(x/Lambda^2), and the REAL contour is now the continuation inside the parabola through the physical threshold,
    Re x > (Im x)^2/(16 m^2) - 4 m^2 -- including points next to the negative axis between -m^2 and -4 m^2 where the
    paper's routing fails.  Catches a wrong sign of the b z terms, a missing x/4, a subtraction not at x = 0."""
    n_rad, n_ang, cutoff2 = 512, 256, 1e8
    rn, rw = oracle.make_quadrature("gauss_legendre", n_rad)
    z, wz = oracle.make_quadrature("gauss_cheb2", n_ang, measure="sqrt1mz2")
    inside = np.array([0.5 + 0.2j, 1 + 2j, -3 + 0.002j, -3.9 + 0.002j, -3.5 + 0.5j, 2 - 4j, 1e-7])
    outside = np.array([-8 + 4j, -6 + 1j])
    ref_in = np.array([complex(CF.cf1(x)) for x in inside])
    ref_out = np.array([complex(CF.cf1(x)) for x in outside])
    Ps = oracle.make_params(BUB, BUB, cutoff2, routing="symmetric")
    g, _ = oracle.eval_grid(Ps, rn, rw, n_rad, z, wz, inside)
    assert relerr(g, ref_in).max() < 2e-7            # O(x/Lambda^2) + quadrature
    g, _ = oracle.eval_grid(Ps, rn, rw, n_rad, z, wz, outside)
    assert relerr(g, ref_out).min() > 1e-2           # outside the parabola REAL is another function
    # the paper's routing fails at the points between the two parabolas
    Pp = oracle.make_params(BUB, BUB, cutoff2)
    g, _ = oracle.eval_grid(Pp, rn, rw, n_rad, z, wz, inside[2:5])
    assert relerr(g, ref_in[2:5]).min() > 1e-3
    # invariants: G(0) = 0 exactly, conjugation symmetry bitwise
    g0, _ = oracle.eval_grid(Ps, rn, rw, n_rad, z, wz, np.array([0.0]))
    assert g0[0] == 0
    a, _ = oracle.eval_grid(Ps, rn, rw, n_rad, z, wz, inside[:6])
    b, _ = oracle.eval_grid(Ps, rn, rw, n_rad, z, wz, np.conj(inside[:6]))
    assert np.array_equal(b, np.conj(a))


def test_symmetric_routing_on_the_deformed_contours(oracle):
    """The cut of the symmetric routing is the cut of the paper's routing at x/4 ((y + x/4 + m^2)^2 = x y z^2), so the
    contour policies applied to x/4 continue it: RAY_ARC and AUTO reach CF1 outside the threshold parabola
    Re x > (Im x)^2/16m^2 - 4m^2 where the REAL contour is off by 50 % and more; THREAD (for Re x/4 <= -4.1 m^2) gives
    the discontinuity across the cut.  Catches contours built from x instead of x/4, a policy test on the wrong variable."""
    rn, rw = oracle.make_radial_pyramid(512, levels=4)
    z, wz = oracle.make_quadrature("gauss_cheb2", 256, measure="sqrt1mz2")
    xs = np.array([0.5 + 0.2j, -3 + 0.5j, -8 + 4j, -6 + 1j, 2 - 9j, -20 + 12j])
    ref = np.array([complex(CF.cf1(x)) for x in xs])
    for contour in ("ray_arc", "auto"):
        g, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e8, routing="symmetric", contour=contour), rn, rw, 512, z, wz, xs)
        assert relerr(g, ref).max() < 1e-7, (contour, relerr(g, ref))
    g, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e8, routing="symmetric"), rn, rw, 512, z, wz, xs[[2, 3, 5]])
    assert relerr(g, ref[[2, 3, 5]]).min() > 0.3
    # the policy is applied to x/4: the nodes of x under the symmetric routing are the nodes of x/4 under the paper's
    Ps = oracle.make_params(BUB, BUB, 1e8, routing="symmetric", contour="auto")
    Pp = oracle.make_params(BUB, BUB, 1e8, contour="auto")
    for x in (-8 + 4j, -30 + 0.5j, 0.5 + 0.2j):
        ps, ys, ws = oracle.contour_nodes(Ps, x, rn, rw, 512, 256)
        pp, yp, wp = oracle.contour_nodes(Pp, x / 4, rn, rw, 512, 256)
        assert ps == pp and np.array_equal(ys, yp) and np.array_equal(ws, wp)
    # next to the cut below the threshold: THREAD through AUTO, Im G = -+ pi sqrt(1 - 4/s) within its accuracy
    gp, gm = oracle.eval_grid(Ps, rn, rw, 512, z, wz, np.array([-30 + 0.05j, -30 - 0.05j]))[0]
    disc = math.pi * math.sqrt(1 - 4 / 30)
    assert abs(gp.imag / -disc - 1) < 0.2 and abs(gm.imag / disc - 1) < 0.2 and gm == np.conj(gp)


def test_symmetric_routing_argument_checks(oracle):
    rn, rw, z, wz = tables(oracle, 64, 32)
    for kw in (dict(line_pk={"kind": "massive", "m2": 2.0}), dict(line_pk=RAT), dict(taylor_order=1)):
        args = dict(line_k=BUB, line_pk=BUB, cutoff2=1e4, routing="symmetric")
        args.update(kw)
        with pytest.raises(ValueError):
            oracle.eval_grid(oracle.make_params(**args), rn, rw, 64, z, wz, np.array([1.0]))


# ---------------------------------------------------------------- rules of other dimensions
def _angular_moment(alpha, k):
    """int_-1^1 (1-z^2)^alpha z^(2k) dz = B(k + 1/2, alpha + 1)."""
    return float(mp.beta(mp.mpf(k) + mp.mpf(1) / 2, mp.mpf(alpha) + 1))


@pytest.mark.parametrize("n", [1, 2, 7, 32, 129])
def test_cheb1_is_the_gauss_rule_of_d2(oracle, n):
    """Gauss-Chebyshev of the first kind (A-S 25.4.38): z_j = cos((2j-1) pi/2n), weights pi/n, exact for
    int (1-z^2)^(-1/2) z^(2k) dz = pi (2k)!/(4^k k!^2) up to degree 2n-1.  Catches second-kind nodes, a wrong weight."""
    z, w = oracle.make_quadrature_dim("gauss_cheb1", n, 2.0)
    assert np.allclose(w, math.pi / n, rtol=2e-15)
    assert np.array_equal(z, -z[::-1]) and (np.all(np.diff(z) > 0) or n == 1)
    assert abs(z[-1] - math.cos(math.pi / (2 * n))) < 2e-16
    for k in range(0, min(n, 12)):
        exact = math.pi * math.factorial(2 * k) / (4 ** k * math.factorial(k) ** 2)
        assert abs(np.sum(w * z ** (2 * k)) - exact) < 4e-15 * exact * max(1, n / 8)
    if 2 <= n <= 32:   # a Gauss rule of n nodes: degree 2n is off by exactly -pi 2^(1-2n) (sum_j T_2n(z_j) pi/n = -pi)
        exact = math.pi * math.factorial(2 * n) / (4 ** n * math.factorial(n) ** 2)
        assert abs((np.sum(w * z ** (2 * n)) - exact) / (-math.pi * 2.0 ** (1 - 2 * n)) - 1) < 1e-3 * 4.0 ** max(0, n - 20)


@pytest.mark.parametrize("dim", [2.0, 3.0, 3.5, 4.0, 5.0, 6.0])
@pytest.mark.parametrize("kind", ["gauss_legendre", "gauss_cheb1", "gauss_cheb2", "tanh_sinh"])
def test_rules_of_the_d_dimensional_angular_measure(oracle, kind, dim):
    """make_quadrature_dim integrates (1-z^2)^((d-3)/2) z^(2k) dz = B(k+1/2, (d-1)/2): exactly (to rounding) for the
    Gauss rule of that measure (Legendre d=3, Chebyshev-1 d=2, Chebyshev-2 d=4), within the rule's error otherwise.
    d = 3 and d = 4 reproduce the tables of make_quadrature bit for bit."""
    alpha = (dim - 3) / 2
    n = 97 if kind == "tanh_sinh" else 64
    z, w = oracle.make_quadrature_dim(kind, n, dim)
    # the Gauss rule of the measure, and the Chebyshev rules wherever the remaining power of sin(theta) is even (the
    # midpoint / trapezoid rule in theta is then exact for the cosine polynomial; Chebyshev-2 has no end nodes, so it
    # needs at least sin^2)
    exact_rule = {("gauss_legendre", 3.0), ("gauss_cheb1", 2.0), ("gauss_cheb1", 4.0), ("gauss_cheb1", 6.0),
                  ("gauss_cheb2", 4.0), ("gauss_cheb2", 6.0)}
    for k in range(6):
        ref = _angular_moment(alpha, k)
        err = abs(np.sum(w * z ** (2 * k)) - ref) / ref
        if (kind, dim) in exact_rule:
            assert err < 1e-14, (k, err)          # polynomial x natural weight: exact
        elif kind == "tanh_sinh":
            assert err < (1e-10 if alpha >= 0 else 2e-5), (k, err)   # end-point singularity z^2-1 at d = 2
        else:
            assert err < (0.1 if alpha < 0 else 5e-3), (k, err)   # algebraic convergence where the weight is not smooth
    if dim in (3.0, 4.0) and kind != "gauss_cheb1":
        z0, w0 = oracle.make_quadrature(kind, n, measure="plain" if dim == 3.0 else "sqrt1mz2")
        assert np.array_equal(z, z0) and np.array_equal(w, w0)
    assert np.allclose(z, -z[::-1], rtol=0, atol=3e-16) and np.allclose(w, w[::-1], rtol=1e-14, atol=0)


def test_dimension_2_bubble_with_the_cheb1_rule(oracle):
    """d = 2 through the rule of its own measure: the angular integral int (1-z^2)^(-1/2)/(A - b z) dz = pi/sqrt(A^2-b^2)
    is reproduced by Chebyshev-1 to rounding where Gauss-Legendre with the weight folded in is off by 1e-3 (the rule,
    not the measure, is what the dimension changes: PAPER.md:138)."""
    A, b = 3.0, 1.0
    z, w = oracle.make_quadrature_dim("gauss_cheb1", 32, 2.0)
    assert abs(np.sum(w / (A - b * z)) - math.pi / math.sqrt(A * A - b * b)) < 1e-14
    zg, wg = oracle.make_quadrature_dim("gauss_legendre", 32, 2.0)
    assert 1e-4 < abs(np.sum(wg / (A - b * zg)) - math.pi / math.sqrt(A * A - b * b)) < 1e-1


# ---------------------------------------------------------------- Taylor subtraction of order n (eq. (12),(13))
@pytest.mark.parametrize("n", [1, 2, 3])
@pytest.mark.parametrize("lines", ["bubble", "unequal_complex", "rational"])
def test_taylor_order_matches_the_definition(oracle, n, lines):
    """(1 - t^n) F with t^n of eq. (13) read as the Taylor operator in p (reading G20): the oracle's
    combined form against the definition itself -- F minus its Taylor polynomial, differentiated numerically at 100+
    digits (tests/mp_reference.py) -- on small rules.  Catches a wrong binomial, a dropped or extra term of the
    polynomial, a wrong remainder, for massive and rational lines."""
    lk, lp = {"bubble": (BUB, BUB), "unequal_complex": ({"kind": "massive", "m2": 0.5j}, {"kind": "massive", "m2": 2 - 0.5j}),
              "rational": (BUB, RAT)}[lines]
    P = oracle.make_params(lk, lp, 1e4, taylor_order=n)
    rn, rw = oracle.make_quadrature("gauss_legendre", 12)
    z, wz = oracle.make_quadrature("gauss_cheb2", 9, measure="sqrt1mz2")
    for x in (0.5 + 0.2j, -2.0 + 1.5j, 3e-3 - 1e-3j, 40.0 + 9j, -2.8e4 + 9.4e3j):   # the last: |x| >> y, m^2
        ref = MPR.finite_sum(oracle, P, x, rn, rw, 12, z, wz, digits=60)
        g, _ = oracle.eval_grid(P, rn, rw, 12, z, wz, np.array([x]), accum="quad")
        assert relerr(g, [ref])[0] < 1e-15, (x, g, ref)
        g, _ = oracle.eval_grid(P, rn, rw, 12, z, wz, np.array([x]), accum="extended")
        assert relerr(g, [ref])[0] < 2e-13, (x, g, ref)


@pytest.mark.parametrize("n", [1, 2])
def test_taylor_order_closed_form_of_the_bubble(oracle, n):
    """Subtracting t^n under the integral removes the first n Taylor coefficients of G: with CF1's series
    -tau/6 + tau^2/60 - ..., G_1 = CF1 + x/(6 m^2), G_2 = G_1 - x^2/(60 m^4).  Catches a wrong sign or
    order of the subtracted terms; the tight tolerance needs the Gauss rule of the measure."""
    xs = [0.5 + 0.2j, 1 + 2j, 3.0, -0.5 + 0.3j, 0.05 - 0.02j]
    g = G(oracle, xs, cutoff2=1e6, n_rad=256, n_ang=128, taylor_order=n)
    with mp.workdps(40):
        ref = [CF.cf1(x) + mp.mpc(x) / 6 - (mp.mpc(x) ** 2 / 60 if n == 2 else 0) for x in xs]
        ref = [complex(r) for r in ref]
    assert np.max(relerr(g, ref)) < 3e-12


def test_taylor_order_rational_line_against_cf3(oracle):
    """Config 4's lines: G_1(x) = CF3(x) - x CF3'(0), the derivative of the Feynman-parameter form taken numerically."""
    xs = [0.5 + 0.2j, 1 + 1j]
    g = G(oracle, xs, line_k=BUB, line_pk=RAT, cutoff2=1e6, n_rad=256, n_ang=128, taylor_order=1)
    with mp.workdps(30):
        d0 = mp.diff(lambda t: CF.cf3_rational(t, 1.0, 2.0, 0.5, 1.2), 0, h=mp.mpf("1e-8"))
        ref = [complex(CF.cf3_rational(x, 1.0, 2.0, 0.5, 1.2) - mp.mpc(x) * d0) for x in xs]
    assert np.max(relerr(g, ref)) < 1e-10


def test_taylor_order_invariants_and_cutoff(oracle):
    """G_n(0) = 0 exactly and G_n = O(x^(n+1)) (G_1/x^2 -> 1/60 m^4); conjugation symmetry bitwise; the cutoff error of
    G_1 falls at least as fast as order 0's Lambda^-4 (BPHZ ensures cut-off independence)."""
    rn, rw, z, wz = tables(oracle, 256, 128, ang="gauss_cheb2", levels=1)
    P1 = oracle.make_params(BUB, BUB, 1e6, taylor_order=1)
    g, _ = oracle.eval_grid(P1, rn, rw, 256, z, wz, np.array([0.0, 1e-4, 1e-4j]), accum="extended")
    assert g[0] == 0
    assert abs(g[1] / 1e-8 - 1 / 60) < 1e-5 and abs(g[2] / -1e-8 - 1 / 60) < 1e-5
    xs = np.array([0.7 - 1.1j, -3 + 0.5j, 2e-3 + 1e-3j])
    a, _ = oracle.eval_grid(P1, rn, rw, 256, z, wz, xs)
    b, _ = oracle.eval_grid(P1, rn, rw, 256, z, wz, np.conj(xs))
    assert np.array_equal(b, np.conj(a))
    x = np.array([0.5 + 0.2j])
    ref = complex(CF.cf1(x[0])) + x[0] / 6
    err = []
    for c2 in (1e2, 1e3, 1e4):
        Pc = oracle.make_params(BUB, BUB, c2, taylor_order=1)
        gc, _ = oracle.eval_grid(Pc, rn, rw, 256, z, wz, x)
        err.append(abs(gc[0] - ref))
    p1, p2 = math.log10(err[0] / err[1]), math.log10(err[1] / err[2])
    assert p1 > 1.9 and p2 > 1.9, (err, p1, p2)   # error ~ Lambda^-4 or faster: two decades per decade of Lambda^2


def test_taylor_order_argument_checks(oracle):
    rn, rw, z, wz = tables(oracle, 64, 32)
    for kw in (dict(taylor_order=-1), dict(taylor_order=5), dict(taylor_order=1, routing="symmetric"), dict(sub=1.0)):
        args = dict(line_k=BUB, line_pk=BUB, cutoff2=1e4)
        args.update(kw)
        with pytest.raises(ValueError):
            oracle.eval_grid(oracle.make_params(**args), rn, rw, 64, z, wz, np.array([1.0]))
    # order 0 through the new code path selector is the old value, bit for bit
    g0, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e4, taylor_order=0), rn, rw, 64, z, wz, np.array([1.0 + 1j]))
    g1, _ = oracle.eval_grid(oracle.make_params(BUB, BUB, 1e4, taylor_order=1), rn, rw, 64, z, wz, np.array([1.0 + 1j]))
    assert g0[0] != g1[0] and abs(g1[0] - (g0[0] + (1 + 1j) / 6)) < 1e-3
