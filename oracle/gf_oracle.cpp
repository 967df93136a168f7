// gf_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU evaluation of the hot path of
// arXiv:1205.0752 (Windisch, Alkofer, Haase, Liebmann): for every complex
// x = p^2 of a grid, the regularised d=4 one-loop integral eq. (14)/(15)
// as a non-adaptive radial x angular quadrature (Step 5,
// PAPER.md:109-113; Kernel 2) of the Taylor-subtracted
// integrand eq. (12)/(20).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may build, load or call this file.  It shares no code, header,
// table or constant generator with paper_1205_0752_b200/csrc (the CUDA path)
// and neither includes the other.
//
// What is computed:
//
//   G(x) = c0 * sum_seg sum_i  Wr(seg,i;x) * y_i * sum_j w'_j * F_sub(x, y_i, z_j)
//
//   F     = D1(y) * D2(u),   u = x + y - 2 sqrt(x) sqrt(y) z = (p-k)^2   eq. (10),(19)
//   F_sub = (1 - t^0) F = D1(y) * [ D2(u) - D2(y) ]                      eq. (12),(13),(20)
//
// The loops run in the paper's order (sub-contour, radial node, angular node),
// every term is evaluated in std::complex<double> arithmetic in the combined
// form the paper itself prints in eq. (20) (so that G(0) = 0 exactly), and the
// sums are accumulated in long double (accum=0) or double (accum=1, the timed
// variant).  accum=2, the parity variant, runs the same loops with every term in
// std::complex<long double> as well: at the rare points where the contour passes
// within ~1e-5 of a singularity of the integrand, and at tiny |x| where the +-z
// terms cancel to O(sqrt|x|), double terms are themselves only good to ~1e-11
// (reading G18); below |x| = 2^-10 it runs them in binary128, because there the +-z
// terms cancel by a factor 2 sqrt(y/|x|).  Domain of the parity variant: x = 0 or |x| >~ 1e-30
// (below that no fixed-width type can form the plain sum; tests use tests/mp_reference.py, the
// same sum at 400 digits).  No blocking, pairing, fusion or reordering.
//
// Pins (tests/test_oracle_pins.py): closed form CF1 of the equal-mass bubble,
// the paper's eq. (18) for masses^2 = +-i/2, the Feynman-parameter form CF3 for
// the rational propagator, G(0)=0, conjugation symmetry, cutoff independence,
// line-swap symmetry, rule independence, exactness degree of the quadrature
// rules, brute-force high-order quadrature; the paper's Kernels 3 and 4 (angular integral B of eq. (22) over
// complex y; obstruction of the real y-axis by the cut) against the textbook angular integral, the scan
// itself and the parabola of PAPER.md:270; the Taylor subtraction of order n > 0 (eq. (12),(13)) against the
// definition itself (F minus its Taylor polynomial in p, differentiated numerically at 100+ digits), the closed form
// CF1 minus its first n Taylor terms, CF3 minus x CF3'(0), G_n = O(x^(n+1)); the rules of the d-dimensional angular
// measure (Gauss-Chebyshev of the first kind included) against B(k+1/2, (d-1)/2).  Unpinned: values of RAY_ARC inside
// the wedge around the negative real axis and of REAL outside the parabola R2
// (DESIGN.md "parity unpinned"), where no closed form applies.
//
// Build: g++ -O2 -std=c++17 -shared -fPIC -pthread ... -lquadmath (no -ffast-math).

#include <quadmath.h>

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

typedef std::complex<double> cplx;
typedef long double ld;

const long double kPi = 3.14159265358979323846264338327950288L;

// ---- enums (values are part of the oracle's own C interface) -------------
enum { QUAD_GAUSS_LEGENDRE = 0, QUAD_GAUSS_CHEB2 = 1, QUAD_TANH_SINH = 2, QUAD_GAUSS_CHEB1 = 3 };
enum { MEASURE_PLAIN = 0, MEASURE_SQRT1MZ2 = 1 };
enum { PROP_MASSIVE = 0, PROP_RATIONAL = 1 };
enum { CONTOUR_REAL = 0, CONTOUR_RAY_ARC = 1, CONTOUR_THREAD = 2, CONTOUR_AUTO = 3 };
enum { SPACING_UNIFORM = 0, SPACING_LOG_ABS_IM = 1 };

struct Propagator {
  int kind;
  double m2_re, m2_im;  // MASSIVE: 1/(u + m2)
  double M2, a, b;      // RATIONAL: (u + M2)/(u^2 + a u + b)
};

struct Params {
  Propagator line_k;   // D1(y), carries k        (eq. (19))
  Propagator line_pk;  // D2(u), carries p-k
  double cutoff2;      // Lambda^2
  double sub_re, sub_im;
  int taylor_order;
  double prefactor;    // c0; 2/pi reproduces eq. (21)
  double map_scale;    // s0 of the shifted-log radial map
  int contour;
  int precision;
  int routing;         // 0: the paper's eq. (19), lines carry k and p-k; 1: symmetric, lines carry k+p/2 and
                       // k-p/2 (equal massive lines, real contour)
  double dim;          // space-time dimension d ("arbitrary dimensions by trivial modifications");
                       // 0 means 4.  The radial measure is dy y^((d-2)/2) (d^dk = 1/2 y^((d-2)/2) dy dOmega_d);
                       // the angular measure (1-z^2)^((d-3)/2) is in the caller's angular weights.
};

// ---- quadrature rules on [-1,1] ----------------------------

// Gauss-Legendre: roots of P_n by Newton iteration, weights 2/((1-x^2)P_n'(x)^2)
// (Abramowitz-Stegun 25.4.29; the paper's radial rule, ref. [18]).
void gauss_legendre(int n, double* x, double* w) {
  for (int k = 0; k < (n + 1) / 2; ++k) {
    ld t = std::cos((ld)kPi * ((ld)k + 0.75L) / ((ld)n + 0.5L));
    ld dp = 0;
    for (int it = 0; it < 100; ++it) {
      ld p0 = 1, p1 = t;
      for (int l = 2; l <= n; ++l) {
        ld p2 = ((2 * l - 1) * t * p1 - (l - 1) * p0) / l;
        p0 = p1;
        p1 = p2;
      }
      if (n == 1) { p0 = 1; p1 = t; }
      dp = n * (t * p1 - p0) / (t * t - 1);
      ld dt = p1 / dp;
      t -= dt;
      if (std::fabs(dt) < 1e-19L) break;
    }
    // recompute the derivative at the converged root
    {
      ld p0 = 1, p1 = t;
      for (int l = 2; l <= n; ++l) {
        ld p2 = ((2 * l - 1) * t * p1 - (l - 1) * p0) / l;
        p0 = p1;
        p1 = p2;
      }
      dp = n * (t * p1 - p0) / (t * t - 1);
    }
    ld wt = 2 / ((1 - t * t) * dp * dp);
    // k = 0 is the largest root; store ascending
    x[n - 1 - k] = (double)t;
    x[k] = -(double)t;
    w[n - 1 - k] = (double)wt;
    w[k] = (double)wt;
  }
  if (n % 2 == 1) x[n / 2] = 0.0;
}

// Rules for the angular measure (1 - z^2)^alpha dz, alpha = (d-3)/2 in d dimensions (eq. (5),(9) for d = 4: alpha =
// 1/2; "arbitrary dimensions by trivial modifications"; Gauss-Legendre, Gauss-Chebyshev "of
// the first and second kind ... depending on the dimension", tanh-sinh).  The Gauss-Chebyshev rules are the exact Gauss
// rules of d = 2 (first kind, weight (1-z^2)^(-1/2)) and d = 4 (second kind, weight (1-z^2)^(1/2)); for another
// alpha the remaining power of (1 - z^2) = sin^2(theta) is put into the weights, as for Gauss-Legendre and tanh-sinh.
int make_quadrature_alpha(int kind, int n, double step, long double alpha, double* x, double* w) {
  if (n < 1 || !x || !w) return 1;
  if (kind == QUAD_GAUSS_LEGENDRE) {
    gauss_legendre(n, x, w);
    if (alpha == 0.5L)
      for (int j = 0; j < n; ++j) w[j] *= std::sqrt((1.0 - x[j]) * (1.0 + x[j]));
    else if (alpha != 0)
      for (int j = 0; j < n; ++j) w[j] = (double)((ld)w[j] * std::pow(((ld)1 - (ld)x[j]) * ((ld)1 + (ld)x[j]), alpha));
    return 0;
  }
  if (kind == QUAD_GAUSS_CHEB2) {
    // Gauss-Chebyshev, 2nd kind: exact Gauss rule for the weight sqrt(1-z^2)
    // (Abramowitz-Stegun 25.4.40; the paper's check rule): z_j = cos(j pi/(n+1)),
    // w_j = pi/(n+1) sin^2(theta_j); for the weight (1-z^2)^alpha: pi/(n+1) sin^(2 alpha + 1)(theta_j).
    for (int j = 0; j < n; ++j) {
      ld th = (ld)kPi * (ld)(n - j) / (ld)(n + 1);  // ascending z
      ld sn = std::sin(th);
      x[j] = (double)std::cos(th);
      ld ww = (ld)kPi / (ld)(n + 1) * sn * sn;  // includes sqrt(1-z^2)
      w[j] = (double)(alpha == 0.5L ? ww : alpha == 0 ? ww / sn : ww * std::pow(sn, 2 * alpha - 1));
    }
    if (n % 2 == 1) x[n / 2] = 0.0;
    return 0;
  }
  if (kind == QUAD_GAUSS_CHEB1) {
    // Gauss-Chebyshev, 1st kind: exact Gauss rule for the weight 1/sqrt(1-z^2) (Abramowitz-Stegun 25.4.38):
    // z_j = cos((2j-1) pi/(2n)), w_j = pi/n; for the weight (1-z^2)^alpha: pi/n sin^(2 alpha + 1)(theta_j).
    for (int j = 0; j < n; ++j) {
      ld th = (ld)kPi * (ld)(2 * (n - j) - 1) / (ld)(2 * n);  // ascending z
      ld sn = std::sin(th);
      x[j] = (double)std::cos(th);
      w[j] = (double)((ld)kPi / (ld)n * std::pow(sn, 2 * alpha + 1));
    }
    if (n % 2 == 1) x[n / 2] = 0.0;
    return 0;
  }
  if (kind == QUAD_TANH_SINH) {
    // Takahasi-Mori double exponential rule (the paper's angular rule, ref. [19]):
    // z_k = tanh(pi/2 sinh(kh)), w_k = pi/2 h cosh(kh) / cosh^2(pi/2 sinh(kh)),
    // k = -(n-1)/2 .. (n-1)/2.  Step h: reading G8, 2.9/((n-1)/2).
    ld h = step > 0 ? (ld)step : (n > 1 ? 2.9L / (((ld)n - 1) / 2) : 1.0L);
    for (int j = 0; j < n; ++j) {
      ld k = (ld)j - ((ld)n - 1) / 2;
      ld a = 0.5L * (ld)kPi * std::sinh(k * h);
      ld ch = std::cosh(a);
      x[j] = (double)std::tanh(a);
      ld ww = 0.5L * (ld)kPi * h * std::cosh(k * h) / (ch * ch);
      // 1 - tanh^2 = sech^2, computed without cancellation
      w[j] = (double)(alpha == 0.5L ? ww / ch : alpha == 0 ? ww : ww * std::pow(1 / ch, 2 * alpha));
    }
    if (n % 2 == 1) x[n / 2] = 0.0;
    return 0;
  }
  return 2;
}

int make_quadrature(int kind, int n, double step, int measure, double* x, double* w) {
  if (measure != MEASURE_PLAIN && measure != MEASURE_SQRT1MZ2) return 2;
  return make_quadrature_alpha(kind, n, step, measure == MEASURE_SQRT1MZ2 ? 0.5L : 0.0L, x, w);
}

// ---- Step 4 / Kernel 1: the grid ------------------
// Endpoint-inclusive homogeneous distribution (reading G9).  Two-sided: the
// lower half counts up from min, the upper half counts down from max, so a
// range symmetric about 0 gives exactly mirrored values.
double lin_two_sided(double lo, double hi, int n, int i) {
  if (n == 1) return lo;
  double d = (hi - lo) / (double)(n - 1);
  if (2 * i <= n - 1) return std::fma((double)i, d, lo);
  return std::fma(-(double)(n - 1 - i), d, hi);
}

int make_grid(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
              int spacing, double im_abs_min, double* x) {
  if (!x) return 1;
  if (n_re < 1 || n_im < 1) return 2;
  if (spacing == SPACING_LOG_ABS_IM) {
    // reading G10: |Im x| log-spaced in [im_abs_min, im_max], both signs, ascending Im
    if (n_im % 2 != 0 || !(im_abs_min > 0) || !(im_max > im_abs_min) || im_min != -im_max) return 2;
  } else if (spacing != SPACING_UNIFORM) {
    return 2;
  }
  for (int j = 0; j < n_im; ++j) {
    double im;
    if (spacing == SPACING_UNIFORM) {
      im = lin_two_sided(im_min, im_max, n_im, j);
    } else {
      int half = n_im / 2;
      int k = j >= half ? j - half : half - 1 - j;
      double v;
      if (k == 0) v = im_abs_min;
      else if (k == half - 1) v = im_max;
      else {
        double l0 = std::log(im_abs_min), l1 = std::log(im_max);
        v = std::exp(std::fma((double)k / (double)(half - 1), l1 - l0, l0));
      }
      im = j >= half ? v : -v;
    }
    for (int i = 0; i < n_re; ++i) {
      x[2 * ((size_t)j * n_re + i) + 0] = lin_two_sided(re_min, re_max, n_re, i);
      x[2 * ((size_t)j * n_re + i) + 1] = im;
    }
  }
  return 0;
}

// ---- propagators ---------------------------------------------------------
// R is the real type the terms are evaluated in: double, or long double for the
// variant whose own rounding error is negligible against the 1e-11 parity bar
// even where a term is nearly singular or x is tiny (reading G18).
template <typename R>
std::complex<R> prop(const Propagator& P, std::complex<R> u) {
  typedef std::complex<R> C;
  if (P.kind == PROP_MASSIVE) return C(1) / (u + C((R)P.m2_re, (R)P.m2_im));
  return (u + (R)P.M2) / (u * u + (R)P.a * u + (R)P.b);
}

// D2(u) - D2(y) with u = y + d, in the combined form of eq. (20)
// (PAPER.md:198-203): the factor d = x - 2 sqrt(x) sqrt(y) z is explicit, so
// the difference is exactly 0 at x = 0 and keeps full relative accuracy at
// small |x| (a numerical difference of two nearly equal numbers would not).
template <typename R>
std::complex<R> prop_diff(const Propagator& P, std::complex<R> y, std::complex<R> d) {
  typedef std::complex<R> C;
  C u = y + d;
  if (P.kind == PROP_MASSIVE) {
    C c = y + C((R)P.m2_re, (R)P.m2_im);
    return -d / ((c + d) * c);
  }
  // (u+M2)/Q(u) - (y+M2)/Q(y) = -d [u y + M2 (u+y) + a M2 - b] / (Q(u) Q(y))
  C Qu = u * u + (R)P.a * u + (R)P.b;
  C Qy = y * y + (R)P.a * y + (R)P.b;
  return -d * (u * y + (R)P.M2 * (u + y) + ((R)P.a * (R)P.M2 - (R)P.b)) / (Qu * Qy);
}

// ---- Taylor subtraction of order n > 0 (eq. (12),(13)) ---------------------------------------
// Reading G20: eq. (13)'s "x = 0" is p = 0 -- eq. (20) sets the scalar product sqrt(x) sqrt(y) z to zero
// together with x -- so t^n is the BPHZ Taylor operator in the external momentum p_mu, and a power x^i of eq. (13)
// is the order 2i in p.  With p -> eps p,  F(eps) = D1(y) D2(y + eps^2 x + eps bz),  bz = -2 sqrt(x) sqrt(y) z, and
//   t^n F = the Taylor polynomial of F(eps) of degree 2n, at eps = 1
//         = D1(y) sum_{m=0}^{2n} t_m sum_{l <= m, m + l <= 2n} C(m,l) x^l bz^(m-l),     t_m = D2^(m)(y)/m!
// (d^m = (x + bz)^m = sum_l C(m,l) x^l bz^(m-l) has the order m + l in p).  The odd orders are odd in z and cancel
// under a symmetric angular rule; n = 0 gives t^0 F = D1(y) D2(y), eq. (20).
//
// t_m, m = 0..M, by Leibniz' rule on Q f = N (f = D2 = N/Q):  Q t_m = N_m - Q' t_{m-1} - (Q''/2) t_{m-2},
// N_0 = N(y), N_1 = N'(y), N_m = 0 beyond (N is linear or constant).
const int kMaxTaylor = 4;
template <typename R>
void prop_taylor(const Propagator& P, std::complex<R> y, int M, std::complex<R>* t) {
  typedef std::complex<R> C;
  if (P.kind == PROP_MASSIVE) {   // N = 1, Q = y + m2
    C Q = y + C((R)P.m2_re, (R)P.m2_im);
    t[0] = C(1) / Q;
    for (int m = 1; m <= M; ++m) t[m] = -t[m - 1] / Q;
    return;
  }
  C Q = y * y + (R)P.a * y + (R)P.b, Q1 = (R)2 * y + (R)P.a;   // Q''/2 = 1
  t[0] = (y + (R)P.M2) / Q;
  if (M >= 1) t[1] = (C(1) - Q1 * t[0]) / Q;
  for (int m = 2; m <= M; ++m) t[m] = -(Q1 * t[m - 1] + t[m - 2]) / Q;
}

// squared distance from y to the nearest pole of the propagator (selects between two equal forms below)
double pole_distance2(const Propagator& P, std::complex<double> y) {
  if (P.kind == PROP_MASSIVE) return std::norm(y + std::complex<double>(P.m2_re, P.m2_im));
  std::complex<double> sq = std::sqrt(std::complex<double>(P.a * P.a - 4.0 * P.b, 0.0));
  return std::fmin(std::norm(y - 0.5 * (-P.a + sq)), std::norm(y - 0.5 * (-P.a - sq)));
}

// D2(u) - [Taylor polynomial of D2 of degree 2n in p], u = y + d, d = x + bz, in a combined form (like eq. (20) for
// n = 0: every term carries its full power of p explicitly, no difference of nearly equal numbers is formed):
//   D2(y + d) - sum_{m <= M} t_m d^m = -d^(M+1) [Q' t_M + (Q''/2)(t_{M-1} + t_M d)] / Q(u)        (M = 2n >= 2)
// (multiply by Q(u) = Q + Q' d + (Q''/2) d^2: the coefficients of d^0..d^M cancel identically, those of d^(M+1) and
// d^(M+2) remain), plus the terms of sum_{m <= M} t_m d^m whose order in p exceeds 2n, which t^n does not subtract:
//   sum_{m = n+1}^{2n} t_m sum_{l = 2n-m+1}^{m} C(m,l) x^l bz^(m-l).
template <typename R>
std::complex<R> prop_diff_taylor(const Propagator& P, std::complex<R> y, std::complex<R> x, std::complex<R> bz, int n) {
  typedef std::complex<R> C;
  const int M = 2 * n;
  C t[2 * kMaxTaylor + 1];
  prop_taylor<R>(P, y, M, t);
  C d = x + bz, u = y + d;
  // Where |d| is not small against the distance from y to the nearest pole of D2 (|c| for a massive line) the
  // polynomial is the larger part of F_sub and the definition itself, D2(u) minus the polynomial, is well
  // conditioned; the combined form below would cancel by (d/c)^(n+1) there (its pieces are of the orders 2n+1 and
  // above in d/c, the result of the order 2n).  Both are the same number; each is used where it is accurate (the
  // test only selects the form, its own accuracy plays no part).
  if ((R)4 * std::norm(d) > (R)pole_distance2(P, std::complex<double>((double)y.real(), (double)y.imag()))) {
    C poly = 0;
    for (int m = 0; m <= M; ++m) {
      R binom = 1;
      C xl = 1;
      for (int l = 0; l <= m && m + l <= M; ++l) {
        C bp = 1;
        for (int k = 0; k < m - l; ++k) bp *= bz;
        poly += t[m] * binom * xl * bp;
        binom = binom * (R)(m - l) / (R)(l + 1);
        xl *= x;
      }
    }
    return prop<R>(P, u) - poly;
  }
  C dM1 = d;
  for (int k = 0; k < M; ++k) dM1 *= d;   // d^(M+1)
  C rem;
  if (P.kind == PROP_MASSIVE) {
    rem = -dM1 * t[M] / (u + C((R)P.m2_re, (R)P.m2_im));
  } else {
    C Qu = u * u + (R)P.a * u + (R)P.b, Q1 = (R)2 * y + (R)P.a;
    rem = -dM1 * (Q1 * t[M] + t[M - 1] + t[M] * d) / Qu;
  }
  C extra = 0;
  for (int m = n + 1; m <= M; ++m) {
    R binom = 1;                         // C(m, l), starting at l = 0
    C xl = 1;                            // x^l
    for (int l = 0; l <= m; ++l) {
      if (l >= M - m + 1) {
        C bp = 1;
        for (int k = 0; k < m - l; ++k) bp *= bz;
        extra += t[m] * binom * xl * bp;
      }
      binom = binom * (R)(m - l) / (R)(l + 1);
      xl *= x;
    }
  }
  return rem + extra;
}

// Symmetric routing (shift invariance of eq. (4)): both lines 1/(q^2 + m2) with
// q = k +- p/2, (k +- p/2)^2 = y + x/4 +- sqrt(x) sqrt(y) z, so
//   F = 1/((c' + b z)(c' - b z)),  c' = y + x/4 + m2,  b = sqrt(x) sqrt(y),   F(x=0) = 1/c^2,  c = y + m2,
//   F_sub = F - F(x=0) = [c^2 - c'^2 + b^2 z^2] / ((c' + b z)(c' - b z) c^2)
//         = x [y z^2 - (2c + x/4)/4] / ((c' + b z)(c' - b z) c^2)
// (numerator combined so that x is an explicit factor, like eq. (20): exactly 0 at x = 0).
template <typename R>
std::complex<R> fsub_symmetric(const Propagator& P, std::complex<R> x, std::complex<R> y, std::complex<R> b, R z) {
  typedef std::complex<R> C;
  C m2((R)P.m2_re, (R)P.m2_im);
  C c = y + m2, cp = c + x / (R)4;
  C num = x * (y * (z * z) - ((R)2 * c + x / (R)4) / (R)4);
  return num / ((cp + b * z) * (cp - b * z) * c * c);
}

// scale of the singular structure of line 2 in the y-plane: |m2^2| for a
// massive line, the largest pole modulus sqrt(b)... of Q(u)=u^2+au+b for a
// rational one (used only to size contours).
double line2_scale(const Propagator& P) {
  if (P.kind == PROP_MASSIVE) return std::hypot(P.m2_re, P.m2_im);
  double disc = P.a * P.a - 4.0 * P.b;
  if (disc < 0) return std::sqrt(P.b);  // complex-conjugate pair, |u_r|^2 = b
  double r = std::sqrt(disc);
  return std::fmax(std::fabs(-P.a + r), std::fabs(-P.a - r)) / 2.0;
}

// ---- contours (Step 3; the IF-THEN-ELSE of Kernel 2,
//      PAPER.md:162,310).  DESIGN.md "Contour policies" states each one. -----
// node, (rule weight) x dy/dt, and arg y continued along the contour from its start at y = 0 (used only for the
// measure y^((d-2)/2) of d != 4: the branch of the power follows the contour, reading G21 of DESIGN.md)
struct RNode { cplx y; cplx wy; double arg; };

struct Rule { const double* t; const double* w; int n; };

// level l of the radial pyramid: Gauss-Legendre rule of order n_rad >> l
// ("n arrays for the radial nodes"), stored back to back.
Rule level(const double* nodes, const double* weights, int n_rad, int l) {
  int off = 0, n = n_rad;
  for (int k = 0; k < l; ++k) { off += n; n /= 2; }
  Rule r = { nodes + off, weights + off, n };
  return r;
}

// shifted-log map of a real segment [a,b] (readings G3/G4):
//   y(u) = a + (a+s0) expm1(u L),  L = ln((b+s0)/(a+s0)),  dy/du = L (y+s0)
// Node positions are evaluated in binary128 (libquadmath) and rounded once to double, like the
// quadrature tables, which are made in extended precision: where the contour passes close to a
// singularity of the integrand a 1-ulp difference of y_i (e.g. between two libm's expm1) changes
// the sum by far more than 1e-11 (reading G18), so y_i must be THE correctly rounded value.
void seg_logreal(double a, double b, double s0, cplx dir, Rule R, std::vector<RNode>& out) {
  const __float128 as = (__float128)a + (__float128)s0;
  const __float128 L = logq(((__float128)b + (__float128)s0) / as);
  for (int i = 0; i < R.n; ++i) {
    double u = 0.5 * (R.t[i] + 1.0);
    double r = (double)((__float128)a + as * expm1q((__float128)u * L));
    double dr = (double)((__float128)(0.5 * R.w[i]) * L * ((__float128)r + (__float128)s0));
    RNode nd = { dir * r, dir * dr, std::atan2(dir.imag(), dir.real()) };   // a ray from 0: arg y = arg dir
    out.push_back(nd);
  }
}

// lower: the piece dips below the negative real axis (THREAD's pieces W2 -> W3 -> W4, which pass under the inward
// tail of the cut): there arg y runs past pi, so a node with Im y < 0 has arg y = atan2 + 2 pi
void seg_line(cplx a, cplx b, Rule R, std::vector<RNode>& out, bool lower = false) {
  for (int i = 0; i < R.n; ++i) {
    double u = 0.5 * (R.t[i] + 1.0);
    cplx y = a + (b - a) * u;
    double arg = std::atan2(y.imag(), y.real());
    if (lower && y.imag() < 0) arg += 2.0 * (double)kPi;
    RNode nd = { y, (b - a) * (0.5 * R.w[i]), arg };
    out.push_back(nd);
  }
}

// Arc of the circle |y| = Rad from Rad e^{i phi} back to the real axis at Rad, tau = tan(phi/4), |tau| <= 1, in the
// rational parametrisation  y(v) = Rad ((1 + i tau v)/(1 - i tau v))^2,  v = 1 - u  (angle 4 atan(tau v), so v = 1 is
// the ray's end and v = 0 the real axis):  dy/du = -4 i tau y / (1 + tau^2 v^2).  Only + - * / occur, each rounded
// once in the order written, so the nodes are the same doubles on any IEEE machine.
void seg_arc(double Rad, double tau, Rule R, std::vector<RNode>& out) {
  for (int i = 0; i < R.n; ++i) {
    double u = 0.5 * (R.t[i] + 1.0);
    double v = 1.0 - u;
    double tv = tau * v;
    double t2 = tv * tv;
    double n2 = 1.0 + t2;
    double in2 = 1.0 / n2;                                  // the one division of the node
    double gr = (1.0 - t2) * in2, gi = (2.0 * tv) * in2;    // g = (1 + i tau v)/(1 - i tau v)
    double gr2 = gr * gr, gi2 = gi * gi;
    double Er = gr2 - gi2, Ei = 2.0 * (gr * gi);            // g^2
    double yr = Rad * Er, yi = Rad * Ei;
    double f = ((2.0 * tau) * R.w[i]) * in2;
    RNode nd = { cplx(yr, yi), cplx(f * yi, -(f * yr)), 4.0 * std::atan(tv) };   // y = Rad g^2, arg g = 2 atan(tau v)
    out.push_back(nd);
  }
}

// The radius of a deformed contour is taken from the ladder {2^k, 1.5 2^k}: the smallest rung >= v.  (The library
// keeps the radial nodes of every rung in tables made once per launch; the ladder is part of the contour's
// definition, so it is restated here.)  rung index I: value(I) = 2^(I/2) for even I, 1.5 2^((I-1)/2) for odd I.
int rung_index(double v) {
  int e;
  double m = std::frexp(v, &e);          // v = m 2^e, 0.5 <= m < 1
  if (m == 0.5) return 2 * (e - 1);
  if (m <= 0.75) return 2 * (e - 1) + 1;
  return 2 * e;
}
const int kRungs = 64;   // rungs tabulated above the one below 1.5 sc; beyond them the radius is Lambda^2/2
double contour_radius(double Rstar, double sc, double cutoff2) {
  int I = rung_index(Rstar), I_lo = rung_index(1.5 * sc) - 1;
  if (I < I_lo) I = I_lo;
  double R = (I & 1) ? std::ldexp(1.5, (I - 1) >> 1) : std::ldexp(1.0, I >> 1);
  if (I > I_lo + kRungs - 1 || !(R < 0.5 * cutoff2)) return 0.5 * cutoff2;
  return R;
}

// direction x/|x| of the ray through x, each component one correctly rounded division (no angle is formed: through
// atan2 and sincos the small component of the direction would inherit the ABSOLUTE error of the angle); x is first
// scaled by a power of two so that no square underflows.  *ax: |x|.
cplx ray_direction(cplx x, double* ax) {
  double big = std::fmax(std::fabs(x.real()), std::fabs(x.imag()));
  if (big == 0.0) { *ax = 0.0; return cplx(1.0, 0.0); }
  int e;
  std::frexp(big, &e);
  double xr = std::ldexp(x.real(), -e), xi = std::ldexp(x.imag(), -e);
  double as = std::sqrt(std::fma(xr, xr, xi * xi));
  *ax = std::ldexp(as, e);
  return cplx(xr / as, xi / as);
}

// tan(phi/4) of the direction (c, s) = (cos phi, sin phi), |phi| <= pi, by half-angle formulas without cancellation
double tan_quarter(double c, double s) {
  double ch, sh;   // cos(phi/2) >= 0, sin(phi/2)
  if (c >= 0.0) {
    ch = std::sqrt(0.5 * (1.0 + c));
    sh = (0.5 * s) / ch;
  } else {
    sh = std::copysign(std::sqrt(0.5 * (1.0 - c)), s);
    ch = (0.5 * std::fabs(s)) / std::fabs(sh);
  }
  return sh / (1.0 + ch);
}

void contour_real(const Params& P, const double* rn, const double* rw, int n_rad, std::vector<RNode>& out) {
  seg_logreal(0.0, P.cutoff2, P.map_scale, cplx(1, 0), level(rn, rw, n_rad, 0), out);
}

// RAY_ARC: generalises the paper's region-2/5 contour: ray along x, arc back to the real axis,
// real tail.
void contour_ray_arc(const Params& P, cplx x, const double* rn, const double* rw, int n_rad,
                     std::vector<RNode>& out) {
  double ax;
  cplx dir = ray_direction(x, &ax);
  double sc = line2_scale(P.line_pk);
  double q = std::sqrt(ax) + std::sqrt(ax + sc);
  double Rad = contour_radius(1.5 * q * q, sc, P.cutoff2);
  seg_logreal(0.0, Rad, P.map_scale, dir, level(rn, rw, n_rad, 1), out);
  seg_arc(Rad, tan_quarter(dir.real(), dir.imag()), level(rn, rw, n_rad, 2), out);
  seg_logreal(Rad, P.cutoff2, P.map_scale, cplx(1, 0), level(rn, rw, n_rad, 2), out);
}

// THREAD: equal real masses, Re x < -4 m^2, near the negative axis.
const double kTau5 = 0.66817863791929891999775768652308;   // tan(3 pi/16): the far waypoint sits at angle 3 pi/4
void contour_thread(const Params& P, cplx x, const double* rn, const double* rw, int n_rad,
                    std::vector<RNode>& out) {
  bool mirror = x.imag() < 0;
  cplx xx = mirror ? std::conj(x) : x;
  double m2 = P.line_pk.m2_re, m = std::sqrt(m2);
  double s;
  cplx e = ray_direction(xx, &s);
  double rs = std::sqrt(s);
  double Aa = (rs - m) * (rs - m), Bb = (rs + m) * (rs + m);
  double t = xx.real() + m2;
  double r0 = std::sqrt(std::fma(t, t, xx.imag() * xx.imag()));   // |x + m^2|
  cplx W[6];
  W[0] = 0.0;
  W[1] = cplx(-m2, 0.5 * (Aa - m2));
  double h2 = 0.5 * (Aa + m2);
  W[2] = cplx(h2 * e.real(), h2 * e.imag());
  W[3] = cplx(-0.5 * (Aa + r0), -0.5 * (r0 - Aa));
  W[4] = cplx(r0 * e.real(), r0 * e.imag());
  double Rad = contour_radius(1.5 * Bb, line2_scale(P.line_pk), P.cutoff2);
  {   // W5 = Rad e^{3 pi i/4} as the arc's own v = 1 end
    double t2 = kTau5 * kTau5, n2 = 1.0 + t2;
    double in2 = 1.0 / n2;
    double gr = (1.0 - t2) * in2, gi = (2.0 * kTau5) * in2;
    double gr2 = gr * gr, gi2 = gi * gi;
    W[5] = cplx(Rad * (gr2 - gi2), Rad * (2.0 * (gr * gi)));
  }
  size_t first = out.size();
  for (int k = 0; k < 5; ++k) seg_line(W[k], W[k + 1], level(rn, rw, n_rad, 3), out, k == 2 || k == 3);
  seg_arc(Rad, kTau5, level(rn, rw, n_rad, 3), out);
  seg_logreal(Rad, P.cutoff2, P.map_scale, cplx(1, 0), level(rn, rw, n_rad, 2), out);
  if (mirror)
    for (size_t k = first; k < out.size(); ++k) {
      out[k].y = std::conj(out[k].y);
      out[k].wy = std::conj(out[k].wy);
      out[k].arg = -out[k].arg;
    }
}

bool thread_applicable(const Params& P) {
  return P.line_k.kind == PROP_MASSIVE && P.line_pk.kind == PROP_MASSIVE && P.line_k.m2_im == 0 &&
         P.line_pk.m2_im == 0 && P.line_k.m2_re == P.line_pk.m2_re && P.line_pk.m2_re > 0;
}

// (Re sqrt(mu))^2 = (|mu| + Re mu)/2, the smallest over the poles -mu of line 2: the REAL contour is the continuation
// exactly where |Im sqrt(x)| < Re sqrt(mu) for every pole (the cut (sqrt(x) z + i sqrt(x (1-z^2) + mu))^2 of eq. (25)
// reaches the positive real y-axis when an end point (sqrt(x) +- i sqrt(mu))^2 becomes real), i.e. inside the parabola
// Re x > (Im x)^2/(4 c2) - c2 -- for a real mass m the parabola of PAPER.md:270 with c2 = m^2.
double parabola_c2(const Propagator& q) {
  auto c2 = [](double mr, double mi) { return 0.5 * (std::sqrt(std::fma(mr, mr, mi * mi)) + mr); };
  if (q.kind == PROP_MASSIVE) return c2(q.m2_re, q.m2_im);
  double disc = q.a * q.a - 4.0 * q.b;
  if (disc >= 0.0) {
    double r = std::sqrt(disc);
    return std::fmin(c2(0.5 * (q.a - r), 0.0), c2(0.5 * (q.a + r), 0.0));
  }
  return c2(0.5 * q.a, 0.5 * std::sqrt(-disc));
}
bool in_parabola(double xr, double xi, double cc) {
  double t = xr + cc;
  return t > 0.0 && xi * xi < (4.0 * cc) * t;
}

// AUTO: per-point choice, half-open tests exactly as DESIGN.md writes them.
//   1. inside the parabola of half the size (|Im sqrt x| < 0.71 Re sqrt mu): REAL, exact and the cheapest;
//   2. next to the negative real axis (|Im x| n_rad < 80 |Re x|), where the ray of RAY_ARC passes the pole of line 1
//      and the opening of the cut closer than the radial rule resolves: REAL as long as x is inside the parabola;
//   3. in the wedge {Re x < -sc, |Im x| n_ang sc < 5 |x|^2}: THREAD where it applies and Re x <= -4.1 sc, else REAL
//      (bounded and reproducible, but NOT the continuation: the documented limitation);
//   4. RAY_ARC everywhere else.
int auto_policy(const Params& P, cplx x, int n_rad, int n_ang) {
  double sc = line2_scale(P.line_pk), c2 = parabola_c2(P.line_pk);
  double xr = x.real(), xi = x.imag();
  if (in_parabola(xr, xi, 0.5 * c2)) return CONTOUR_REAL;
  bool near_axis = xr < 0.0 && std::fabs(xi) * (double)n_rad < 80.0 * std::fabs(xr);
  if (near_axis && in_parabola(xr, xi, c2)) return CONTOUR_REAL;
  double ax2 = std::fma(xr, xr, xi * xi);
  bool wedge = (xr < -sc) && (std::fabs(xi) * ((double)n_ang * sc) < 5.0 * ax2);
  if (!wedge) return CONTOUR_RAY_ARC;
  if (thread_applicable(P) && xr <= -4.1 * sc) return CONTOUR_THREAD;
  return CONTOUR_REAL;
}

// The contour of the point x under the policy of P.  Symmetric routing (lines k + p/2, k - p/2): the zeros of the
// denominators are (y + x/4 + m^2)^2 = x y z^2, i.e. the cut of the paper's routing at the external momentum x/4
// (zeta(x/4, y, m^2) in [0,1]), and the pole of the subtracted term sits at y = -m^2 as before: the policies are applied
// to x/4 (region tests, contour radius, direction and waypoints) and the integrand is taken at x.
int build_contour(const Params& P, cplx x, const double* rn, const double* rw, int n_rad, int n_ang,
                  std::vector<RNode>& nodes) {
  cplx xg = P.routing == 1 ? cplx(0.25 * x.real(), 0.25 * x.imag()) : x;
  int pol = P.contour == CONTOUR_AUTO ? auto_policy(P, xg, n_rad, n_ang) : P.contour;
  if (pol == CONTOUR_REAL) contour_real(P, rn, rw, n_rad, nodes);
  else if (pol == CONTOUR_RAY_ARC) contour_ray_arc(P, xg, rn, rw, n_rad, nodes);
  else contour_thread(P, xg, rn, rw, n_rad, nodes);
  return pol;
}

// principal square root in the term type (libstdc++ has no std::sqrt for complex<__float128>)
template <typename R>
std::complex<R> psqrt(std::complex<R> v) { return std::sqrt(v); }
template <>
std::complex<__float128> psqrt(std::complex<__float128> v) {
  __complex128 c;
  __real__ c = v.real();
  __imag__ c = v.imag();
  c = csqrtq(c);
  return std::complex<__float128>(__real__ c, __imag__ c);
}

// ---- Step 5 / Kernel 2: the double sum for one x ---------------------------
// ACC: type of the two running sums; R: type every term is evaluated in.
template <typename ACC, typename R>
cplx eval_point(const Params& P, cplx x, const double* rn, const double* rw, int n_rad,
                const double* z, const double* wz, int n_ang, std::vector<RNode>& nodes) {
  typedef std::complex<R> C;
  nodes.clear();
  build_contour(P, x, rn, rw, n_rad, n_ang, nodes);

  C xx((R)x.real(), (R)x.imag());
  C sx = psqrt<R>(xx);  // principal branch
  ACC gr = 0, gi = 0;
  for (size_t i = 0; i < nodes.size(); ++i) {
    C y((R)nodes[i].y.real(), (R)nodes[i].y.imag());
    C wy((R)nodes[i].wy.real(), (R)nodes[i].wy.imag());
    C B = (R)2 * sx * psqrt<R>(y);
    C D1 = prop<R>(P.line_k, y);
    ACC sr = 0, si = 0;
    for (int j = 0; j < n_ang; ++j) {
      C d = xx - B * (R)z[j];                                  // u - y
      C f = P.routing == 1 ? fsub_symmetric<R>(P.line_pk, xx, y, B / (R)2, (R)z[j])
            : P.taylor_order == 0 ? D1 * prop_diff<R>(P.line_pk, y, d)   // F_sub, eq. (20)
                                  : D1 * prop_diff_taylor<R>(P.line_pk, y, xx, -(B * (R)z[j]), P.taylor_order);   // eq. (12),(13)
      sr += (ACC)((R)wz[j] * f.real());
      si += (ACC)((R)wz[j] * f.imag());
    }
    C S((R)sr, (R)si);
    // dy y^((d-2)/2) (...): eq. (14) for d = 4; otherwise the power on the branch continued along the contour from
    // y = 0: |y|^p e^(i p arg y) with the node's continued argument (p real; on the real axis arg = 0)
    C term;
    if (P.dim == 0 || P.dim == 4) {
      term = wy * y * S;
    } else {
      const __float128 p = 0.5 * ((__float128)P.dim - 2);
      const __float128 mag = powq(hypotq((__float128)nodes[i].y.real(), (__float128)nodes[i].y.imag()), p);
      const __float128 ang = p * (__float128)nodes[i].arg;
      term = wy * C((R)(mag * cosq(ang)), (R)(mag * sinq(ang))) * S;
    }
    gr += (ACC)term.real();
    gi += (ACC)term.imag();
  }
  return P.prefactor * cplx((double)gr, (double)gi);
}

// ---- paper Kernel 3 (Fig. 1): the angular integral B of eq. (22) for one x at a
// complex y:  B(x, y) = sum_j w'_j [ D2(u_j) - D2(y) ] / D2(y),  u_j = x + y - 2 sqrt(x) sqrt(y) z_j.
// For the massive line of the paper's example this is eq. (22)'s
//   B = int dz sqrt(1-z^2) (-x + 2 sqrt(x) sqrt(y) z) / (x + y - 2 sqrt(x) sqrt(y) z + m2^2).
// Plain loop over the angular nodes, every term and the sum in R.
template <typename R>
cplx angular_B(const Params& P, cplx x, cplx y, const double* z, const double* wz, int n_ang) {
  typedef std::complex<R> C;
  C xx((R)x.real(), (R)x.imag()), yy((R)y.real(), (R)y.imag());
  C B2 = (R)2 * psqrt<R>(xx) * psqrt<R>(yy);
  C D2y = prop<R>(P.line_pk, yy);
  R sr = 0, si = 0;
  for (int j = 0; j < n_ang; ++j) {
    C d = xx - B2 * (R)z[j];
    C f = prop_diff<R>(P.line_pk, yy, d) / D2y;
    sr += (R)wz[j] * f.real();
    si += (R)wz[j] * f.imag();
  }
  return cplx((double)sr, (double)si);
}

// ---- paper Kernel 4 (Fig. 2): does the branch cut that the angular integral induces in
// the y-plane obstruct the original contour, the positive real y-axis up to Lambda^2?  The paper does not say
// how its kernel decides (reading G19).  Here: the cut of a pole -mu of line 2 is the curve
//   y(z) = k(z)^2,  k(z) = sqrt(x) z + i s(z),  s(z) = sqrt(x (1 - z^2) + mu),  -1 <= z <= 1       eq. (23)-(25)
// (the second sign of eq. (24) is the same curve run backwards).  It is sampled at n_z equidistant z, s(z)
// continued from sample to sample (the sign that keeps Re(s_k conj(s_{k-1})) >= 0; principal root at z = -1),
// and a crossing is counted wherever Im y changes sign between neighbours (or is zero at the later one) and
// the linearly interpolated Re y lies in (0, Lambda^2].  Every operation is a correctly rounded +, -, *, /
// or sqrt in a fixed order, so that an integer decision is the same on any IEEE machine.
struct CD { double re, im; };
inline CD csqrt_rn(CD v) {   // principal square root from real operations only
  const double m = std::sqrt(v.re * v.re + v.im * v.im);
  const double h = std::sqrt(0.5 * (m + std::fabs(v.re)));
  if (h == 0.0) return CD{0.0, 0.0};
  const double k = v.im / (2.0 * h);
  if (v.re >= 0.0) return CD{h, k};
  return CD{std::fabs(k), std::copysign(h, v.im)};
}
int cut_crossings_one(CD x, CD mu, double cutoff2, int n_z) {
  const CD sx = csqrt_rn(x);
  int count = 0;
  CD sprev{0.0, 0.0};
  double yre_prev = 0.0, yim_prev = 0.0;
  for (int k = 0; k < n_z; ++k) {
    const double z = -1.0 + 2.0 * (double)k / (double)(n_z - 1);
    const double omz2 = (1.0 - z) * (1.0 + z);
    CD s = csqrt_rn(CD{x.re * omz2 + mu.re, x.im * omz2 + mu.im});
    if (k > 0 && s.re * sprev.re + s.im * sprev.im < 0.0) { s.re = -s.re; s.im = -s.im; }
    const double kre = sx.re * z - s.im, kim = sx.im * z + s.re;   // sqrt(x) z + i s
    const double yre = kre * kre - kim * kim, yim = 2.0 * (kre * kim);
    if (k > 0) {
      const bool cross = (yim_prev < 0.0 && yim >= 0.0) || (yim_prev > 0.0 && yim <= 0.0);
      if (cross) {
        const double t = yim_prev / (yim_prev - yim);               // in (0, 1]
        const double re0 = yre_prev + t * (yre - yre_prev);
        if (re0 > 0.0 && re0 <= cutoff2) ++count;
      }
    }
    sprev = s;
    yre_prev = yre;
    yim_prev = yim;
  }
  return count;
}
// all poles of line 2: one for a massive line (mu = m2^2), two for a rational one (the roots of Q(-mu) = 0)
int cut_crossings(const Params& P, cplx x, int n_z) {
  const Propagator& q = P.line_pk;
  if (q.kind == PROP_MASSIVE) return cut_crossings_one(CD{x.real(), x.imag()}, CD{q.m2_re, q.m2_im}, P.cutoff2, n_z);
  const double disc = q.a * q.a - 4.0 * q.b;
  CD mu1, mu2;   // mu = -u_r, u_r = (-a +- sqrt(disc))/2
  if (disc >= 0.0) {
    const double r = std::sqrt(disc);
    mu1 = CD{0.5 * (q.a - r), 0.0};
    mu2 = CD{0.5 * (q.a + r), 0.0};
  } else {
    const double r = std::sqrt(-disc);
    mu1 = CD{0.5 * q.a, -0.5 * r};
    mu2 = CD{0.5 * q.a, 0.5 * r};
  }
  return cut_crossings_one(CD{x.real(), x.imag()}, mu1, P.cutoff2, n_z) +
         cut_crossings_one(CD{x.real(), x.imag()}, mu2, P.cutoff2, n_z);
}

int check_params(const Params& P, int n_rad, int n_ang) {
  if (n_rad < 1 || n_ang < 1) return 2;
  if (!(P.cutoff2 > 0) || !(P.map_scale > 0)) return 2;
  if (P.taylor_order < 0 || P.taylor_order > kMaxTaylor || P.sub_re != 0 || P.sub_im != 0) return 3;
  if (P.taylor_order != 0 && P.routing != 0) return 3;
  if (P.contour < 0 || P.contour > 3) return 2;
  if (P.contour != CONTOUR_REAL && n_rad % 8 != 0) return 2;
  if (P.contour == CONTOUR_THREAD && !thread_applicable(P)) return 3;
  if (P.routing != 0 && P.routing != 1) return 2;
  if (P.routing == 1 && !(P.line_k.kind == PROP_MASSIVE && P.line_pk.kind == PROP_MASSIVE &&
                          P.line_k.m2_re == P.line_pk.m2_re && P.line_k.m2_im == P.line_pk.m2_im))
    return 3;
  if (!(P.dim == 0 || (P.dim >= 1 && P.dim <= 8))) return 2;
  return 0;
}

}  // namespace

extern "C" {

int gfo_make_quadrature(int kind, int n, double step, int measure, double* nodes, double* weights) {
  return make_quadrature(kind, n, step, measure, nodes, weights);
}

// the rule for the angular measure (1 - z^2)^((dim-3)/2) dz of dim space-time dimensions
int gfo_make_quadrature_dim(int kind, int n, double step, double dim, double* nodes, double* weights) {
  if (!(dim >= 1 && dim <= 8)) return 2;
  return make_quadrature_alpha(kind, n, step, ((long double)dim - 3) / 2, nodes, weights);
}

int gfo_make_grid(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
                  int spacing, double im_abs_min, double* x) {
  return make_grid(re_min, re_max, n_re, im_min, im_max, n_im, spacing, im_abs_min, x);
}

// x, out: interleaved (re, im) doubles.  accum: 0 = double terms, long double sums;
// 1 = double terms and sums (the timed variant); 2 = the parity variant, whose own rounding error
// is << 1e-11 at every point (reading G18): long double terms and sums, and binary128 (libquadmath)
// terms and sums where |x| < 2^-10 -- there the +-z terms, each O(sqrt|x y|), cancel to O(|x|), which
// costs even long double a factor 2 sqrt(y/|x|) (measured against a 60-digit evaluation of the same
// sum: 7e-9 at |x| = 1e-16); with a Taylor order n > 0 below |x| = 2^-4 (the angular sum of the order-(2n+2) terms
// cancels by a further y/mu at large y: 1.7e-12 was measured at |x| = 1.5e-3, mu = 0.013 with long double terms);
// 3 = binary128 everywhere (slow; checks variant 2).
// n_threads <= 0: hardware concurrency.
// Returns 0 on success; fills *threads_used.
int gfo_eval_grid(const void* params, const double* rad_nodes, const double* rad_weights, int n_rad,
                  const double* ang_nodes, const double* ang_weights, int n_ang, const double* x,
                  long long n_points, double* out, int n_threads, int accum, int* threads_used) {
  if (!params || !rad_nodes || !rad_weights || !ang_nodes || !ang_weights || (!x && n_points) ||
      (!out && n_points))
    return 1;
  Params P;
  std::memcpy(&P, params, sizeof(Params));
  int rc = check_params(P, n_rad, n_ang);
  if (rc) return rc;
  if (n_points < 0) return 2;
  int nt = n_threads > 0 ? n_threads : (int)std::thread::hardware_concurrency();
  if (nt < 1) nt = 1;
  if ((long long)nt > n_points) nt = n_points > 0 ? (int)n_points : 1;
  if (threads_used) *threads_used = nt;
  auto work = [&](int tid) {
    std::vector<RNode> nodes;
    nodes.reserve((size_t)n_rad);
    for (long long p = tid; p < n_points; p += nt) {
      cplx xx(x[2 * p], x[2 * p + 1]);
      cplx g = accum == 0
                   ? eval_point<ld, double>(P, xx, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, n_ang, nodes)
               : accum == 1
                   ? eval_point<double, double>(P, xx, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, n_ang, nodes)
               : (accum == 2 && std::fmax(std::fabs(xx.real()), std::fabs(xx.imag())) >= (P.taylor_order > 0 ? 0x1p-4 : 0x1p-10))
                   ? eval_point<ld, ld>(P, xx, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights, n_ang, nodes)
                   : eval_point<__float128, __float128>(P, xx, rad_nodes, rad_weights, n_rad, ang_nodes, ang_weights,
                                                        n_ang, nodes);
      out[2 * p] = g.real();
      out[2 * p + 1] = g.imag();
    }
  };
  if (nt == 1) {
    work(0);
  } else {
    std::vector<std::thread> th;
    for (int t = 0; t < nt; ++t) th.emplace_back(work, t);
    for (auto& t : th) t.join();
  }
  return 0;
}

// the contour of one point, for tests and plots: fills y (2*n doubles) and
// wy (2*n doubles); returns the policy used (0..2) or a negative error.
int gfo_contour_nodes(const void* params, double x_re, double x_im, const double* rad_nodes,
                      const double* rad_weights, int n_rad, int n_ang, double* y, double* wy, int* n_out) {
  Params P;
  std::memcpy(&P, params, sizeof(Params));
  if (check_params(P, n_rad, n_ang)) return -1;
  cplx x(x_re, x_im);
  std::vector<RNode> nodes;
  int pol = build_contour(P, x, rad_nodes, rad_weights, n_rad, n_ang, nodes);
  for (size_t i = 0; i < nodes.size(); ++i) {
    y[2 * i] = nodes[i].y.real(); y[2 * i + 1] = nodes[i].y.imag();
    wy[2 * i] = nodes[i].wy.real(); wy[2 * i + 1] = nodes[i].wy.imag();
  }
  *n_out = (int)nodes.size();
  return pol;
}

// Kernel 3: B(x, y_k) for n complex y (interleaved re, im).  accum: 0 = double terms, 2 = long double terms,
// 3 = binary128 terms (the +-z terms cancel by 2 sqrt(|y/x|) or 2 sqrt(|x/y|) and the leading moment by another
// 1e7: at |y/x| = 1e6 even long double keeps only ten digits of B).
int gfo_eval_angular(const void* params, double x_re, double x_im, const double* ang_nodes, const double* ang_weights,
                     int n_ang, const double* y, long long n, double* out, int accum) {
  if (!params || !ang_nodes || !ang_weights || (!y && n) || (!out && n)) return 1;
  if (n_ang < 1 || n < 0) return 2;
  Params P;
  std::memcpy(&P, params, sizeof(Params));
  for (long long k = 0; k < n; ++k) {
    const cplx xx(x_re, x_im), yy(y[2 * k], y[2 * k + 1]);
    cplx b = accum == 0   ? angular_B<double>(P, xx, yy, ang_nodes, ang_weights, n_ang)
             : accum == 2 ? angular_B<ld>(P, xx, yy, ang_nodes, ang_weights, n_ang)
                          : angular_B<__float128>(P, xx, yy, ang_nodes, ang_weights, n_ang);
    out[2 * k] = b.real();
    out[2 * k + 1] = b.imag();
  }
  return 0;
}

// Kernel 4: crossings of (0, Lambda^2] by the cut(s) of line 2, for n points x; out: n 32-bit integers.
int gfo_cut_crossings(const void* params, const double* x, long long n, int n_z, int* out) {
  if (!params || (!x && n) || (!out && n)) return 1;
  if (n_z < 2 || n < 0) return 2;
  Params P;
  std::memcpy(&P, params, sizeof(Params));
  if (!(P.cutoff2 > 0)) return 2;
  for (long long k = 0; k < n; ++k) out[k] = cut_crossings(P, cplx(x[2 * k], x[2 * k + 1]), n_z);
  return 0;
}

int gfo_params_size(void) { return (int)sizeof(Params); }

}  // extern "C"
