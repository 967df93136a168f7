// gf_geometry.cuh -- the geometry of the point-dependent radial contours (Step 3 inside Kernel 2, PAPER.md:95-103,162,
// 233-272,310; include/gf.h gf_contour): the ladder of contour radii, the direction of the ray, AUTO's per-point choice,
// the waypoints of THREAD, the nodes of straight pieces and arcs, where node g of a point's n_rad nodes lives.  Shared by
// the evaluation kernels that walk such contours (gf_contour.cu: order 0; gf_taylor.cu: Taylor orders n > 0).  No angle
// is ever formed: every operation is a +, -, *, /, sqrt written with the _rn intrinsics in the order gf.h states, so
// the nodes are the same doubles as the oracle's on any IEEE machine.
#pragma once
#include "gf_routes.cuh"

namespace gf {
namespace {

// tan(3 pi/16): the far waypoint of THREAD sits at the angle 3 pi/4 = 4 atan(kTau5)
constexpr double kTau5 = 0.66817863791929891999775768652308;

// ln(v) for a double-double v >= 1: libm seed, one Newton step on exp in double-double
__device__ dd dd_log(dd v) {
  const double l0 = log(v.hi);
  const dd e = dd_add_d(dd_expm1(dd{l0, 0.0}), 1.0);
  const dd c = dd_div(dd_add(v, dd_neg(e)), e);
  return quick_two_sum(l0, c.hi);
}

// ---- the ladder of contour radii -------------------------------------------------------------------
__device__ __forceinline__ int rung_index_dev(double v) {
  int e;
  const double m = frexp(v, &e);   // v = m 2^e, 0.5 <= m < 1 (exact)
  if (m == 0.5) return 2 * (e - 1);
  if (m <= 0.75) return 2 * (e - 1) + 1;
  return 2 * e;
}
__device__ __forceinline__ double rung_value(int I) { return (I & 1) ? ldexp(1.5, (I - 1) >> 1) : ldexp(1.0, I >> 1); }
// smallest rung >= Rstar (not below the first tabulated one); *row: its row in the rung tables
__device__ __forceinline__ double contour_radius(const EvalArgs& a, double Rstar, int* row) {
  int I = rung_index_dev(Rstar);
  if (I < a.rung_lo) I = a.rung_lo;
  const double R = rung_value(I);
  if (I > a.rung_lo + kRungs - 1 || !(R < 0.5 * a.cutoff2)) {
    *row = kRungs;
    return 0.5 * a.cutoff2;
  }
  *row = I - a.rung_lo;
  return R;
}

// ---- the geometry of one point's contour ------------------------------------------------------------
struct Geo {
  int pol;           // GF_CONTOUR_REAL / RAY_ARC / THREAD
  int mirror;        // THREAD for Im x < 0: conjugate every node
  int row;           // row of the rung tables
  double R;          // contour radius
  double dre, dim;   // direction x/|x| of the ray (THREAD: of x mirrored into Im x >= 0)
  double tau;        // arc: tan(phi/4)
  double Aa, r0, m2; // THREAD: (sqrt|x| - m)^2, |x + m^2|, m^2
};

// x/|x| by correctly rounded operations, x scaled by a power of two first so that no square underflows; *ax = |x|
__device__ __forceinline__ void ray_direction(double xr, double xi, double* dre, double* dim, double* ax) {
  const double big = fmax(fabs(xr), fabs(xi));
  if (big == 0.0) { *ax = 0.0; *dre = 1.0; *dim = 0.0; return; }
  int e;
  frexp(big, &e);
  const double sr = ldexp(xr, -e), si = ldexp(xi, -e);
  const double as = __dsqrt_rn(__fma_rn(sr, sr, __dmul_rn(si, si)));
  *ax = ldexp(as, e);
  *dre = __ddiv_rn(sr, as);
  *dim = __ddiv_rn(si, as);
}
// tan(phi/4) of the direction (c, s) = (cos phi, sin phi), |phi| <= pi, by half-angle formulas without cancellation
__device__ __forceinline__ double tan_quarter(double c, double s) {
  double ch, sh;
  if (c >= 0.0) {
    ch = __dsqrt_rn(__dmul_rn(0.5, __dadd_rn(1.0, c)));
    sh = __ddiv_rn(__dmul_rn(0.5, s), ch);
  } else {
    sh = copysign(__dsqrt_rn(__dmul_rn(0.5, __dadd_rn(1.0, -c))), s);
    ch = __ddiv_rn(__dmul_rn(0.5, fabs(s)), fabs(sh));
  }
  return __ddiv_rn(sh, __dadd_rn(1.0, ch));
}
__device__ __forceinline__ bool in_parabola(double xr, double xi, double cc) {
  const double t = __dadd_rn(xr, cc);
  return t > 0.0 && __dmul_rn(xi, xi) < __dmul_rn(__dmul_rn(4.0, cc), t);
}

// AUTO's per-point choice; half-open tests exactly as gf.h writes them:
//   1. inside the parabola of half the size (|Im sqrt x| < 0.71 Re sqrt mu): REAL, exact and the cheapest;
//   2. next to the negative real axis (|Im x| n_rad < 80 |Re x|), where the ray of RAY_ARC passes the pole of line 1
//      and the opening of the cut closer than the radial rule resolves: REAL as long as x is inside the parabola;
//   3. in the wedge {Re x < -sc, |Im x| n_ang sc < 5 |x|^2}: THREAD where it applies and Re x <= -4.1 sc, else REAL
//      (bounded and reproducible, NOT the continuation: the documented limitation);
//   4. RAY_ARC everywhere else.
__device__ __forceinline__ int auto_policy(const EvalArgs& a, double xr, double xi) {
  const double sc = a.line2_scale, c2 = a.parab_c2;
  if (in_parabola(xr, xi, __dmul_rn(0.5, c2))) return GF_CONTOUR_REAL;
  const bool near_axis = xr < 0.0 && __dmul_rn(fabs(xi), (double)a.n_rad) < __dmul_rn(80.0, fabs(xr));
  if (near_axis && in_parabola(xr, xi, c2)) return GF_CONTOUR_REAL;
  const double ax2 = __fma_rn(xr, xr, __dmul_rn(xi, xi));
  const bool wedge = (xr < -sc) && (__dmul_rn(fabs(xi), __dmul_rn((double)a.n_ang, sc)) < __dmul_rn(5.0, ax2));
  if (!wedge) return GF_CONTOUR_RAY_ARC;
  if (a.thread_ok && xr <= __dmul_rn(-4.1, sc)) return GF_CONTOUR_THREAD;
  return GF_CONTOUR_REAL;
}

// force_pol >= 0: the policy is known to the caller at compile time (a kernel instantiated for one policy)
__device__ __forceinline__ Geo build_geo(const EvalArgs& a, double xr, double xi, int force_pol = -1) {
  Geo g = {};
  g.pol = force_pol >= 0 ? force_pol : a.contour == GF_CONTOUR_AUTO ? auto_policy(a, xr, xi) : a.contour;
  g.dre = 1.0;
  if (g.pol == GF_CONTOUR_RAY_ARC) {
    double ax;
    ray_direction(xr, xi, &g.dre, &g.dim, &ax);
    const double q = __dadd_rn(__dsqrt_rn(ax), __dsqrt_rn(__dadd_rn(ax, a.line2_scale)));
    g.R = contour_radius(a, __dmul_rn(__dmul_rn(1.5, q), q), &g.row);
    g.tau = tan_quarter(g.dre, g.dim);
  } else if (g.pol == GF_CONTOUR_THREAD) {
    g.mirror = xi < 0.0;
    const double yi = fabs(xi);
    double s;
    ray_direction(xr, yi, &g.dre, &g.dim, &s);
    g.m2 = a.term[0].mu_re;
    const double m = __dsqrt_rn(g.m2), rs = __dsqrt_rn(s);
    const double dm = __dadd_rn(rs, -m), dp = __dadd_rn(rs, m);
    g.Aa = __dmul_rn(dm, dm);
    const double Bb = __dmul_rn(dp, dp);
    const double t = __dadd_rn(xr, g.m2);
    g.r0 = __dsqrt_rn(__fma_rn(t, t, __dmul_rn(yi, yi)));   // |x + m^2|
    g.R = contour_radius(a, __dmul_rn(1.5, Bb), &g.row);
    g.tau = kTau5;
  }
  return g;
}

// the end of an arc of radius R at v = 1: R ((1 + i tau)/(1 - i tau))^2, in the arc's own arithmetic
__device__ __forceinline__ cd arc_point(double R, double tv, double* in2_out) {
  const double t2 = __dmul_rn(tv, tv);
  const double n2 = __dadd_rn(1.0, t2);
  const double in2 = __drcp_rn(n2);                                    // the one division of the node
  const double gr = __dmul_rn(__dadd_rn(1.0, -t2), in2), gi = __dmul_rn(__dmul_rn(2.0, tv), in2);
  const double gr2 = __dmul_rn(gr, gr), gi2 = __dmul_rn(gi, gi);
  const double Er = __dadd_rn(gr2, -gi2), Ei = __dmul_rn(2.0, __dmul_rn(gr, gi));
  *in2_out = in2;
  return {__dmul_rn(R, Er), __dmul_rn(R, Ei)};
}
// waypoint W_k of THREAD (Im x >= 0 side), k = 0..5
__device__ __forceinline__ cd thread_waypoint(const Geo& g, int k) {
  switch (k) {
    case 0: return {0.0, 0.0};
    case 1: return {-g.m2, __dmul_rn(0.5, __dadd_rn(g.Aa, -g.m2))};
    case 2: {
      const double h2 = __dmul_rn(0.5, __dadd_rn(g.Aa, g.m2));
      return {__dmul_rn(h2, g.dre), __dmul_rn(h2, g.dim)};
    }
    case 3: return {__dmul_rn(-0.5, __dadd_rn(g.Aa, g.r0)), __dmul_rn(-0.5, __dadd_rn(g.r0, -g.Aa))};
    case 4: return {__dmul_rn(g.r0, g.dre), __dmul_rn(g.r0, g.dim)};
    default: {
      double in2;
      return arc_point(g.R, kTau5, &in2);
    }
  }
}

// Where node g of the point's n_rad nodes lives.  type, index i inside its piece, and for LINE the piece k.
enum { SEG_TABLE = 0, SEG_RAY = 1, SEG_LINE = 2, SEG_ARC = 3, SEG_TAIL = 4 };
struct NodeAt {
  int type, i, k, rule;   // rule: offset of the piece's Gauss-Legendre rule inside the staged levels 2 and 3
};
__device__ __forceinline__ NodeAt locate(int pol, int n_rad, int g) {
  const int n2 = n_rad >> 1, n4 = n_rad >> 2, n8 = n_rad >> 3;
  if (pol == GF_CONTOUR_REAL) return {SEG_TABLE, g, 0, 0};
  if (pol == GF_CONTOUR_RAY_ARC) {
    if (g < n2) return {SEG_RAY, g, 0, 0};
    if (g < n2 + n4) return {SEG_ARC, g - n2, 0, 0};
    return {SEG_TAIL, g - n2 - n4, 0, 0};
  }
  if (g < 5 * n8) {
    const int k = (g >= n8) + (g >= 2 * n8) + (g >= 3 * n8) + (g >= 4 * n8);   // g / n8 without the division
    return {SEG_LINE, g - k * n8, k, n4};
  }
  if (g < 6 * n8) return {SEG_ARC, g - 5 * n8, 0, n4};
  return {SEG_TAIL, g - 6 * n8, 0, 0};
}
// index of the first node of the real tail piece
__device__ __forceinline__ int tail_start(int pol, int n_rad) {
  return pol == GF_CONTOUR_REAL ? 0 : n_rad - (n_rad >> 2);
}

// node of a straight piece a -> a + d and of an arc: y and (rule weight) x dy/dt
__device__ __forceinline__ void line_node(cd a, cd d, double t, double w, cd* y, cd* wy) {
  const double u = __dmul_rn(0.5, __dadd_rn(t, 1.0)), hw = __dmul_rn(0.5, w);
  *y = {__dadd_rn(a.re, __dmul_rn(d.re, u)), __dadd_rn(a.im, __dmul_rn(d.im, u))};
  *wy = {__dmul_rn(d.re, hw), __dmul_rn(d.im, hw)};
}
__device__ __forceinline__ void arc_node(double R, double tau, double t, double w, cd* y, cd* wy) {
  const double u = __dmul_rn(0.5, __dadd_rn(t, 1.0));
  const double v = __dadd_rn(1.0, -u);
  double in2;
  *y = arc_point(R, __dmul_rn(tau, v), &in2);
  const double f = __dmul_rn(__dmul_rn(__dmul_rn(2.0, tau), w), in2);
  *wy = {__dmul_rn(f, y->im), -__dmul_rn(f, y->re)};   // -i f y
}

// y + mu with mu = hi + lo: accurate to an ulp of itself next to the pole y = -mu
__device__ __forceinline__ cd y_plus_mu(cd y, const PoleTerm& t) {
  return {(y.re + t.mu_re) + t.mu_re_lo, (y.im + t.mu_im) + t.mu_im_lo};
}
// Other dimensions (gf_params.dim): the radial measure y^p, p = (d-2)/2, at complex y, on the branch continued along the
// contour from y = 0 (reading G21): |y|^p e^(i p arg y) with the continued argument of the node --
// arg dir on the ray, 4 atan(tau v) on an arc, atan2 on a straight piece, plus 2 pi below the negative real axis on
// THREAD's pieces W2 -> W3 -> W4 (which pass under the inward tail of the cut), negated for the mirrored contour.
__device__ __forceinline__ cd cpow_arg(cd y, double arg, double p) {
  const double mag = exp(0.5 * p * log(fma(y.re, y.re, y.im * y.im)));
  double sn, cs;
  sincos(p * arg, &sn, &cs);
  return {mag * cs, mag * sn};
}
// c0 (rule weight x dy/dt) y^p for a node of a straight piece (k: THREAD's piece) or of an arc, before mirroring
__device__ __forceinline__ cd measure_base(const EvalArgs& a, const Geo& geo, int seg_type, int k, double t, cd y, cd wy) {
  if (a.ypow == 1.0) return cscale(cmul(wy, y), a.c0);
  double arg;
  if (seg_type == SEG_ARC) {
    arg = 4.0 * atan(geo.tau * (1.0 - 0.5 * (t + 1.0)));
  } else {
    arg = atan2(y.im, y.re);
    if ((k == 2 || k == 3) && y.im < 0.0) arg += 6.283185307179586476925;
  }
  return cscale(cmul(wy, cpow_arg(y, arg, a.ypow)), a.c0);
}
// the direction factor of the ray's nodes: dy y^p = dir^(p+1) r^p dr
__device__ __forceinline__ cd ray_measure_dir(const EvalArgs& a, const Geo& geo) {
  if (a.ypow == 1.0) return {fma(geo.dre, geo.dre, -(geo.dim * geo.dim)), 2.0 * geo.dre * geo.dim};
  double sn, cs;
  sincos((a.ypow + 1.0) * atan2(geo.dim, geo.dre), &sn, &cs);
  return {cs, sn};
}

// D1(y) for complex y; a rational line through its factored denominator (y + nu_1)(y + nu_2), which stays accurate
// where the contour passes next to a root
__device__ __forceinline__ cd line_k_complex(const EvalArgs& a, cd y) {
  const gf_propagator& p = a.line_k;
  if (p.kind == GF_PROP_MASSIVE) return cinv_fast(cd{y.re + p.m2_re, y.im + p.m2_im});
  const cd den = cmul(y_plus_mu(y, a.kroot[0]), y_plus_mu(y, a.kroot[1]));
  return cmul(cd{y.re + p.M2, y.im}, cinv_fast(den));
}


}  // namespace
}  // namespace gf
