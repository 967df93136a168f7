// gf_tables.cpp -- host-side generation of the quadrature tables (row a2 of the hot-path table;
// the paper's "Preparation": nodes and weights are calculated on the host).
// Library code; shares nothing with oracle/.
#include <quadmath.h>

#include <cmath>
#include <vector>

#include "gf_internal.h"

namespace gf {
namespace {

typedef long double real;
const real PI = 3.141592653589793238462643383279502884L;

// Legendre P_n(t) and P_{n-1}(t) by the three-term recurrence (Bonnet).
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

// Gauss-Legendre (ref. [18]).  Positive roots by Newton's method from Tricomi's
// estimate; weights from w = 2 / ((1 - t^2) P_n'(t)^2) (A-S 25.4.29; the equivalent form with P_{n-1} is n
// times more sensitive to the last-bit error of the root).  Mirrored, so the rule is exactly symmetric.
void gauss_legendre(int n, double* x, double* w) {
  const int half = n / 2;
  for (int m = 0; m < half; ++m) {
    // m-th positive root counted from the largest
    real th = PI * (4 * (m + 1) - 1) / (4 * (real)n + 2);
    real t = (1 - (real)(n - 1) / (8 * (real)n * n * n) - 1 / (384 * (real)n * n * n * n) * (39 - 28 / (sinl(th) * sinl(th)))) * cosl(th);
    real pn, pm;
    for (int it = 0; it < 50; ++it) {
      legendre_pair(n, t, &pn, &pm);
      real dpn = n * (pm - t * pn) / (1 - t * t);
      real dt = pn / dpn;
      t -= dt;
      if (fabsl(dt) <= 2e-20L * fabsl(t)) break;
    }
    legendre_pair(n, t, &pn, &pm);
    const real dpn = n * (pm - t * pn) / (1 - t * t);
    real wt = 2 / ((1 - t * t) * dpn * dpn);
    x[n - 1 - m] = (double)t;
    x[m] = -(double)t;
    w[n - 1 - m] = w[m] = (double)wt;
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

int make_rule_host(int kind, int n, double step, int measure, double* nodes, double* weights) {
  if (!nodes || !weights) { set_error("make_quadrature: null table pointer"); return GF_ERR_NULL; }
  if (n < 1 || n > (1 << 20)) { set_error("make_quadrature: n=%d out of range [1, 2^20]", n); return GF_ERR_ARG; }
  if (measure != GF_MEASURE_PLAIN && measure != GF_MEASURE_SQRT1MZ2) {
    set_error("make_quadrature: unknown measure %d", measure);
    return GF_ERR_ARG;
  }
  if (!(step >= 0) || !std::isfinite(step)) { set_error("make_quadrature: step must be >= 0"); return GF_ERR_ARG; }
  const bool ang = measure == GF_MEASURE_SQRT1MZ2;
  switch (kind) {
    case GF_QUAD_GAUSS_LEGENDRE: {
      gauss_legendre(n, nodes, weights);
      if (ang)
        for (int j = 0; j < n; ++j) {
          real z = nodes[j];
          weights[j] = (double)((real)weights[j] * sqrtl((1 - z) * (1 + z)));
        }
      return GF_OK;
    }
    case GF_QUAD_GAUSS_CHEB2: {
      // z_j = cos(j pi/(n+1)), w_j = pi/(n+1) sin^2(j pi/(n+1)) for the weight sqrt(1-z^2) (A-S 25.4.40)
      for (int j = 0; j < n / 2; ++j) {
        real th = PI * (real)(j + 1) / (real)(n + 1);  // largest z first
        real s = sinl(th), c = cosl(th);
        real wt = PI / (real)(n + 1) * s * (ang ? s : 1.0L);
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
    case GF_QUAD_TANH_SINH: {
      // Takahasi-Mori (ref. [19]); default step: reading G8 of DESIGN.md
      real h = step > 0 ? (real)step : (n > 1 ? 5.8L / (real)(n - 1) : 1.0L);
      for (int j = 0; j < (n + 1) / 2; ++j) {
        real k = (real)(n - 1) / 2 - (real)j;  // k >= 0, largest first
        real arg = 0.5L * PI * sinhl(k * h);
        real sech = 1 / coshl(arg);
        real wt = 0.5L * PI * h * coshl(k * h) * sech * sech * (ang ? sech : 1.0L);
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

}  // namespace gf
