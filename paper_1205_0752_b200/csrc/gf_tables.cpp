// gf_tables.cpp -- host-side generation of the quadrature tables (row a2 of the hot-path table;
// the paper's "Preparation": nodes and weights are calculated on the host).
// Library code; shares nothing with oracle/.
#include <quadmath.h>

#include <algorithm>
#include <cmath>
#include <functional>
#include <thread>
#include <vector>

#include "gf_internal.h"

namespace gf {
namespace {

typedef long double real;
const real PI = 3.141592653589793238462643383279502884L;

// Legendre P_n(t) and P_{n-1}(t) by the three-term recurrence (Bonnet), extended precision.
inline void legendre_pair(int n, real t, real* pn, real* pnm1) {
  real a = 1.0L, b = t;  // P_0, P_1
  if (n == 0) { *pn = a; *pnm1 = 0; return; }
  for (int k = 1; k < n; ++k) {
    real c = ((2 * k + 1) * t * b - k * a) / (k + 1);
    a = b;
    b = c;
  }
  *pn = b;
  *pnm1 = a;
}

// The same in double with the coefficients al_k = (2k+1)/(k+1), be_k = k/(k+1) tabulated (no division in
// the loop): only used to bring Tricomi's estimate to a double-precision root quickly.
struct BonnetD {
  std::vector<double> al, be;
  explicit BonnetD(int n) : al(n + 1), be(n + 1) {
    for (int k = 0; k <= n; ++k) {
      al[k] = (2.0 * k + 1.0) / (k + 1.0);
      be[k] = (double)k / (k + 1.0);
    }
  }
  void pair(int n, double t, double* pn, double* pnm1) const {
    double a = 1, b = t;
    for (int k = 1; k < n; ++k) {
      const double c = al[k] * t * b - be[k] * a;
      a = b;
      b = c;
    }
    *pn = b;
    *pnm1 = a;
  }
};

// legendre_pair for kLanes points at once: the same operations per point in the same order (bit-identical
// results), interleaved so that the divisions of independent recurrences overlap in the pipeline.
constexpr int kLanes = 4;
inline void legendre_pair_lanes(int n, const real* t, real* pn, real* pnm1) {
  real a[kLanes], b[kLanes];
  for (int l = 0; l < kLanes; ++l) { a[l] = 1.0L; b[l] = t[l]; }
  for (int k = 1; k < n; ++k) {
    for (int l = 0; l < kLanes; ++l) {
      real c = ((2 * k + 1) * t[l] * b[l] - k * a[l]) / (k + 1);
      a[l] = b[l];
      b[l] = c;
    }
  }
  for (int l = 0; l < kLanes; ++l) { pn[l] = b[l]; pnm1[l] = a[l]; }
}

// Positive roots m0 <= m < m1 (counted from the largest) of P_n and their weights.
void gauss_legendre_roots(int n, int m0, int m1, const BonnetD& Bd, double* x, double* w) {
  for (int mb = m0; mb < m1; mb += kLanes) {
    real t[kLanes], pn[kLanes], pm[kLanes];
    bool done[kLanes];
    for (int l = 0; l < kLanes; ++l) {
      const int m = mb + l < m1 ? mb + l : m1 - 1;   // a short last group repeats its last root
      const double th = (double)(PI * (4 * (m + 1) - 1) / (4 * (real)n + 2));
      const double dn = n, sn = std::sin(th);
      double t0 = (1 - (dn - 1) / (8 * dn * dn * dn) - 1 / (384 * dn * dn * dn * dn) * (39 - 28 / (sn * sn))) * std::cos(th);
      for (int it = 0; it < 20; ++it) {
        double p, q;
        Bd.pair(n, t0, &p, &q);
        const double dt = p * (1 - t0 * t0) / (dn * (q - t0 * p));
        t0 -= dt;
        if (std::fabs(dt) <= 4e-16 * std::fabs(t0)) break;
      }
      t[l] = t0;
      done[l] = false;
    }
    for (int it = 0; it < 50; ++it) {
      legendre_pair_lanes(n, t, pn, pm);
      bool all = true;
      for (int l = 0; l < kLanes; ++l) {
        if (done[l]) continue;
        const real dpn = n * (pm[l] - t[l] * pn[l]) / (1 - t[l] * t[l]);
        const real dt = pn[l] / dpn;
        t[l] -= dt;
        done[l] = fabsl(dt) <= 1e-12L * fabsl(t[l]);  // quadratic: the next correction is below 1e-21
        all = all && done[l];
      }
      if (all) break;
    }
    legendre_pair_lanes(n, t, pn, pm);
    for (int l = 0; l < kLanes && mb + l < m1; ++l) {
      const int m = mb + l;
      const real dpn = n * (pm[l] - t[l] * pn[l]) / (1 - t[l] * t[l]);
      const real wt = 2 / ((1 - t[l] * t[l]) * dpn * dpn);
      x[n - 1 - m] = (double)t[l];
      x[m] = -(double)t[l];
      w[n - 1 - m] = w[m] = (double)wt;
    }
  }
}

// Gauss-Legendre (ref. [18]).  Positive roots: Tricomi's estimate, Newton's method in double to
// its limit, then Newton in extended precision (one step brings |dt| from ~1e-16 to ~1e-28); weights from
// w = 2 / ((1 - t^2) P_n'(t)^2) (A-S 25.4.29; the equivalent form with P_{n-1} is n times more sensitive to
// the last-bit error of the root) with P_n' from one more extended-precision evaluation at the final root.
// Mirrored, so the rule is exactly symmetric.  Roots are independent: large rules are split over up to 8 threads.
void gauss_legendre(int n, double* x, double* w) {
  const int half = n / 2;
  const BonnetD Bd(n);
  const unsigned hw = std::thread::hardware_concurrency();
  const int n_thr = half < 64 ? 1 : std::max(1, std::min({half / 32, 8, hw ? (int)hw : 4}));
  if (n_thr == 1) {
    gauss_legendre_roots(n, 0, half, Bd, x, w);
  } else {
    // roots near the ends need no more work than the others: equal blocks
    std::vector<std::thread> pool;
    for (int k = 0; k < n_thr; ++k)
      pool.emplace_back(gauss_legendre_roots, n, half * k / n_thr, half * (k + 1) / n_thr, std::cref(Bd), x, w);
    for (auto& th : pool) th.join();
  }
  if (n & 1) {
    real pn, pm;
    legendre_pair(n, 0.0L, &pn, &pm);
    x[half] = 0.0;
    w[half] = (double)(2 / ((real)n * pm * (real)n * pm));
  }
}

}  // namespace

// L = ln((b + s0)/(a + s0)) of the shifted-log map of a real segment [a, b] (readings G3/G4), in binary128,
// split into a double-double.  The map's node positions must not depend on a libm's last bit (DESIGN.md
// reading G18), so L carries ~106 bits.
void log_ratio_dd(double a, double b, double s0, double* hi, double* lo) {
  const __float128 L = logq(((__float128)b + (__float128)s0) / ((__float128)a + (__float128)s0));
  *hi = (double)L;
  *lo = (double)(L - (__float128)*hi);
}

// Rule `kind` for the angular measure (1 - z^2)^alpha dz (alpha = (d-3)/2 in d dimensions; alpha = 0 is
// the plain rule, 1/2 the d = 4 measure of eq. (9)).  Mirrored halves: exactly symmetric.
static int make_rule_alpha(int kind, int n, double step, real alpha, double* nodes, double* weights) {
  if (!nodes || !weights) { set_error("make_quadrature: null table pointer"); return GF_ERR_NULL; }
  if (n < 1 || n > (1 << 20)) { set_error("make_quadrature: n=%d out of range [1, 2^20]", n); return GF_ERR_ARG; }
  if (!(step >= 0) || !std::isfinite(step)) { set_error("make_quadrature: step must be >= 0"); return GF_ERR_ARG; }
  // sin(theta)^(2 alpha + 1 - e): the power of sin left over after the rule's own weight sin^e
  auto spow = [&](real s, real e) { const real p = 2 * alpha + 1 - e; return p == 0 ? (real)1 : p == 1 ? s : p == 2 ? s * s : powl(s, p); };
  switch (kind) {
    case GF_QUAD_GAUSS_LEGENDRE: {
      gauss_legendre(n, nodes, weights);
      if (alpha != 0)
        for (int j = 0; j < n; ++j) {
          real z = nodes[j];
          const real om = (1 - z) * (1 + z);
          weights[j] = (double)((real)weights[j] * (alpha == 0.5L ? sqrtl(om) : powl(om, alpha)));
        }
      return GF_OK;
    }
    case GF_QUAD_GAUSS_CHEB2: {
      // z_j = cos(j pi/(n+1)), w_j = pi/(n+1) sin^2(j pi/(n+1)) for the weight sqrt(1-z^2) (A-S 25.4.40)
      for (int j = 0; j < n / 2; ++j) {
        real th = PI * (real)(j + 1) / (real)(n + 1);  // largest z first
        real s = sinl(th), c = cosl(th);
        real wt = PI / (real)(n + 1) * s * spow(s, 1);
        nodes[n - 1 - j] = (double)c;
        nodes[j] = -(double)c;
        weights[n - 1 - j] = weights[j] = (double)wt;
      }
      if (n & 1) {
        nodes[n / 2] = 0.0;
        weights[n / 2] = (double)(PI / (real)(n + 1));
      }
      return GF_OK;
    }
    case GF_QUAD_GAUSS_CHEB1: {
      // z_j = cos((2j-1) pi/(2n)), w_j = pi/n for the weight 1/sqrt(1-z^2) (A-S 25.4.38): the Gauss rule of d = 2
      for (int j = 0; j < n / 2; ++j) {
        real th = PI * (real)(2 * j + 1) / (real)(2 * n);  // largest z first
        real s = sinl(th), c = cosl(th);
        real wt = PI / (real)n * spow(s, 0);
        nodes[n - 1 - j] = (double)c;
        nodes[j] = -(double)c;
        weights[n - 1 - j] = weights[j] = (double)wt;
      }
      if (n & 1) {
        nodes[n / 2] = 0.0;
        weights[n / 2] = (double)(PI / (real)n);
      }
      return GF_OK;
    }
    case GF_QUAD_TANH_SINH: {
      // Takahasi-Mori (ref. [19]); default step: reading G8 of DESIGN.md
      real h = step > 0 ? (real)step : (n > 1 ? 5.8L / (real)(n - 1) : 1.0L);
      for (int j = 0; j < (n + 1) / 2; ++j) {
        real k = (real)(n - 1) / 2 - (real)j;  // k >= 0, largest first
        real arg = 0.5L * PI * sinhl(k * h);
        real sech = 1 / coshl(arg);
        // (1 - z^2)^alpha = sech^(2 alpha)
        real wt = 0.5L * PI * h * coshl(k * h) * sech * sech * (alpha == 0 ? (real)1 : alpha == 0.5L ? sech : powl(sech, 2 * alpha));
        real z = tanhl(arg);
        nodes[n - 1 - j] = (double)z;
        nodes[j] = -(double)z;
        weights[n - 1 - j] = weights[j] = (double)wt;
      }
      if (n & 1) nodes[n / 2] = 0.0;
      return GF_OK;
    }
    default:
      set_error("make_quadrature: unknown rule kind %d", kind);
      return GF_ERR_ARG;
  }
}

int make_rule_host(int kind, int n, double step, int measure, double* nodes, double* weights) {
  if (measure != GF_MEASURE_PLAIN && measure != GF_MEASURE_SQRT1MZ2) {
    set_error("make_quadrature: unknown measure %d", measure);
    return GF_ERR_ARG;
  }
  return make_rule_alpha(kind, n, step, measure == GF_MEASURE_SQRT1MZ2 ? 0.5L : 0.0L, nodes, weights);
}

int make_rule_dim_host(int kind, int n, double step, double dim, double* nodes, double* weights) {
  if (!(dim >= 1 && dim <= 8)) { set_error("make_quadrature_dim: dim=%g outside [1, 8]", dim); return GF_ERR_ARG; }
  return make_rule_alpha(kind, n, step, ((real)dim - 3) / 2, nodes, weights);
}

}  // namespace gf
