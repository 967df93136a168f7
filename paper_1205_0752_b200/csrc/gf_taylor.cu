// gf_taylor.cu -- Step 5 / Kernel 2 with the Taylor subtraction of order n > 0 (eq. (12),(13)) on
// the REAL contour:  F_sub = (1 - t^n) F,  t^n = sum_{i<=n} x^i/i! [d^i/dx^i]_{x=0}.
//
// Reading G20: "x = 0" of eq. (13) is p = 0 (eq. (20) sets the scalar product to zero together with x),
// so t^n is the BPHZ Taylor operator in the external momentum and x^i stands for the order 2i in p; the odd orders
// are odd in z and vanish under the symmetric angular rule the kernel folds.
//
// The algebra (none of it is in the paper; the oracle evaluates F minus its Taylor polynomial term by term and knows
// none of this).  For one pole 1/(u + mu) of line 2, c = y + mu, A = x + c, t = z^2, the +-z pair
//     f(x) = 1/(A - Bz) + 1/(A + Bz) = 2A/(A^2 - 4 x y t)
// is a rational function of x, analytic at x = 0, whose Taylor coefficients are
//     f = sum_i x^i phi_i,   phi_i = (2/c^(i+1)) psi_i(T),   T = 4 y t/c,   psi_i(T) = sum_k (-1)^(i-k) C(i+k, i-k) T^k
// (psi_i(4 z^2) = U_2i(z), the Chebyshev polynomials of the second kind: psi_{i+1} = (T - 2) psi_i - psi_{i-1}).
// Multiplying the remainder by the denominator, quadratic in x, leaves two terms:
//     f - sum_{i<=n} x^i phi_i = (xi^n/(2y)) [psi_{n+1}(T) - xi psi_n(T)] / (zeta - t),   xi = x/c,  zeta = A^2/(4xy)
// (n = 0: -(2/c)(eta - t)/(zeta - t), the form of gf_eval.cu).  With the folded weights w_j (one per +-z pair):
//     sum_nodes w'_j [1/(u_j + mu) - Taylor] = (xi^n/(4y)) S_n,   S_n = sum_j w_j Pi(t_j)/(zeta - t_j),
//     Pi(t) = psi_{n+1}(kappa t) - xi psi_n(kappa t) = sum_{a<=n+1} pi_a t^a,   kappa = 4y/c.
// S_n goes through the routes of the scan (gf_routes.cuh, route_setup: chosen from zeta alone):
//   MOMENT / CHEB   S_n = g sum_a pi_a P_a(s),  P_a(s) = sum_k m^(a)_k s^k  with the moments of the measures w_j t_j^a,
//                   m^(a)_k = sum_j w_j t_j^a (t_j - 1/2)^k  resp.  sum'_j w_j t_j^a T_k(2 t_j - 1)   (n + 2 tables each,
//                   made once per launch in double-double), each P_a by the second-order (Goertzel) recurrence;
//   NEAR / EXACT    C(zeta) = sum_j w_j/(zeta - t_j) by the direct loop (EXACT: zeta and t_j in double-double), and
//                   S_n = Pi(zeta) C(zeta) - sum_a pi_a sum_{b<a} mu_b zeta^(a-1-b),  mu_b = sum_j w_j t_j^b.
// Every piece of S_n is of the size of the terms of the plain sum, so the rounding error is that of summing those
// terms; x^(n+1) is an explicit factor, so G_n(0) = 0 and small |x| keeps full accuracy.
// One thread per grid point (or 1/S of its radial nodes), no warp-collective step, no tail series: every radial node
// takes a route (far nodes need 4 to 8 series terms).
#include "gf_geometry.cuh"
#include "gf_routes.cuh"

namespace gf {
namespace {

// e_{i,k} = (-1)^(i-k) C(i+k, i-k), the coefficient of T^k in psi_i
__host__ __device__ constexpr double psi_coef(int i, int k) {
  if (k < 0 || k > i) return 0.0;
  double c = 1.0;
  const int n = i + k;
  int r = i - k;
  if (r > n - r) r = n - r;
  for (int q = 1; q <= r; ++q) c = c * (double)(n - r + q) / (double)q;   // small integers: exact
  return ((i - k) & 1) ? -c : c;
}

// The staged tables one node-term needs
struct TaylorTabs {
  Tabs<double> tb;              // a_kreq, kmc (route_setup)
  const double *st, *stlo, *sw; // folded rule
  const double *momA, *chebA;   // n + 2 series tables per family, [k][n + 2]
  int n_pairs;
};
__device__ __forceinline__ TaylorTabs make_taylor_tabs(const double* sb, const BlobLayout& L, int n_pairs) {
  TaylorTabs t = {};
  t.tb.a_kreq = smem_u32(sb + L.off_kreq);
  t.tb.kmc = L.kmc;
  t.tb.kcap = L.kmc;
  t.st = sb + L.off_t;
  t.stlo = sb + L.off_tlo;
  t.sw = sb + L.off_w;
  t.momA = sb + L.off_momA;
  t.chebA = sb + L.off_chebA;
  t.n_pairs = n_pairs;
  return t;
}

// xi^n S_n for one (point, radial node, pole): S_n = sum_j w_j Pi(t_j)/(zeta - t_j) by the route zeta selects (header).
// y may be complex (deformed contours); pole: mu = hi + lo.
template <int N>
__device__ __forceinline__ cd taylor_node(const TaylorTabs& T, cd x, cd y, cd xi, cd kap, cd zeta, const PoleTerm& pole) {
  constexpr int NA = N + 2;
  const SeriesArg o = route_setup<double>(T.tb, zeta);
  cd pi[NA];
  {
    cd kp = {1.0, 0.0};
#pragma unroll
    for (int q = 0; q < NA; ++q) {
      pi[q] = cmul(kp, cd{fma(-xi.re, psi_coef(N, q), psi_coef(N + 1, q)), -xi.im * psi_coef(N, q)});
      kp = cmul(kp, kap);
    }
  }
  cd s;
  if (o.route <= ROUTE_CHEB) {
    const double* tab = o.route == ROUTE_CHEB ? T.chebA : T.momA;
    const double rr = o.sg.re + o.sg.re, ns = o.ns;
    double p1[NA], p2[NA];
#pragma unroll
    for (int q = 0; q < NA; ++q) p1[q] = p2[q] = 0.0;
#pragma unroll 1
    for (int k = o.K - 1; k >= 0; --k) {
      const double* c = tab + k * NA;
#pragma unroll
      for (int q = 0; q < NA; ++q) {
        const double b = fma(rr, p1[q], fma(ns, p2[q], c[q]));
        p2[q] = p1[q];
        p1[q] = b;
      }
    }
    cd acc = {0.0, 0.0};
#pragma unroll
    for (int q = 0; q < NA; ++q) {
      const cd P = {fma(-p2[q], o.sg.re, p1[q]), p2[q] * o.sg.im};   // c_0 - c_1 conj(s)
      acc = cadd(acc, cmul(pi[q], P));
    }
    s = cmul(o.g, acc);
  } else {
    ZetaDD z = {zeta.re, 0.0, zeta.im, zeta.im * zeta.im};
    if (o.route == ROUTE_EXACT) z = zeta_dd(x.re, x.im, y.re, y.im, pole.mu_re, pole.mu_im, pole.mu_re_lo, pole.mu_im_lo);
    double u0 = 0.0, ua = 0.0, v0 = 0.0, va = 0.0;
    int j = 0;
#pragma unroll 1
    for (; j + 2 <= T.n_pairs; j += 2) {
      direct_step(z.re_hi, z.re_lo, z.im2, T.st[j], T.stlo[j], T.sw[j], u0, ua);
      direct_step(z.re_hi, z.re_lo, z.im2, T.st[j + 1], T.stlo[j + 1], T.sw[j + 1], v0, va);
    }
    if (j < T.n_pairs) direct_step(z.re_hi, z.re_lo, z.im2, T.st[j], T.stlo[j], T.sw[j], u0, ua);
    u0 += v0;
    ua += va;
    const cd C = {ua, -z.im * u0};                   // sum_j w_j/(zeta - t_j)
    const cd zt = {z.re_hi, z.im};
    cd Pz = pi[NA - 1], h = {T.momA[0], 0.0}, qs = cmul(pi[1], h);   // momA[q] = m^(q)_0 = sum_j w_j t_j^q
#pragma unroll
    for (int q = NA - 2; q >= 0; --q) Pz = cadd(cmul(Pz, zt), pi[q]);
#pragma unroll
    for (int q = 2; q < NA; ++q) {                   // h_q = sum_{b<q} mu_b zeta^(q-1-b)
      h = cmul(h, zt);
      h.re += T.momA[q - 1];
      qs = cadd(qs, cmul(pi[q], h));
    }
    const cd PC = cmul(Pz, C);
    s = {PC.re - qs.re, PC.im - qs.im};
  }
  cd xn = xi;
#pragma unroll
  for (int q = 1; q < N; ++q) xn = cmul(xn, xi);     // xi^n
  return cmul(xn, s);
}

// ---------------------------------------------------------------------------------------------
// Preparation (one CTA): folded rule, the n + 2 moment and Chebyshev tables, Kreq, radial nodes with 1/(y + mu_r)
// and the node prefactors pref_{r,i} = c0 Wr_i y_i^((d-2)/2) D1(y_i) R_r/(4 y_i).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) prep_taylor_kernel(const __grid_constant__ EvalArgs a,
                                                          const __grid_constant__ BlobLayout L,
                                                          double* __restrict__ blob) {
  __shared__ int bad;
  __shared__ float s_lc[kKmc];
  if (threadIdx.x == 0) bad = 0;
  __syncthreads();
  prep_angular(a, L, blob, &bad);
  check_radial_tables(a, &bad);
  __syncthreads();
  prep_series_T(a, L, blob);
  {
    const dd Llog = {a.Llog_hi, a.Llog_lo};
    for (int i = threadIdx.x; i < L.n_rad_pad; i += blockDim.x) {
      const int ii = min(i, a.n_rad - 1);
      const double y = radial_node(a.rad_nodes[ii], Llog, a.s0);
      const double Wr = i < a.n_rad ? 0.5 * a.rad_weights[ii] * a.Llog_hi * (y + a.s0) : 0.0;
      blob[L.off_y + i] = y;
      blob[L.off_q4 + i] = 0.25 / y;
      const cd d1 = cscale(line_k_real(a.line_k, y), a.c0 * Wr * (a.ypow == 1.0 ? y : pow(y, a.ypow)) * (0.25 / y));
      for (int r = 0; r < a.n_terms; ++r) {
        const cd ic = cinv(cd{y + a.term[r].mu_re, a.term[r].mu_im});
        const cd pr = cmul(d1, cd{a.term[r].R_re, a.term[r].R_im});
        blob[L.off_pref + 2 * (r * L.n_rad_pad + i)] = pr.re;
        blob[L.off_pref + 2 * (r * L.n_rad_pad + i) + 1] = pr.im;
        blob[L.off_ic + 2 * (r * L.n_rad_pad + i)] = ic.re;
        blob[L.off_ic + 2 * (r * L.n_rad_pad + i) + 1] = ic.im;
      }
    }
  }
  __syncthreads();
  prep_series_A(a, L, blob);
  __syncthreads();
  prep_series_kreq(L, blob, s_lc, blob + L.off_chebA, L.n_poly);
  if (threadIdx.x == 0) {
    blob[0] = (double)bad;
    blob[1] = a.ws_tag;
    if (bad) report_status(a.status, bad);
  }
}

// ---------------------------------------------------------------------------------------------
// Evaluation.  N = taylor order, NT = poles of line 2.
// ---------------------------------------------------------------------------------------------
template <int N, int NT>
__global__ void __launch_bounds__(kBlockThreads, 2)
    eval_taylor_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                       const double* __restrict__ blob) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
  double* sb = reinterpret_cast<double*>(smem_raw + 16);
  if (!workspace_matches(a, blob)) {   // prepared for other parameters or orders: refuse it before reading a table
    const long long pt = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> a.split_log2;
    if (pt < a.n_points) reinterpret_cast<double2*>(a.out)[pt] = make_double2(nan(""), nan(""));
    if (blockIdx.x == 0 && threadIdx.x == 0) report_status(a.status, kStatusWorkspace);
    return;
  }
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) bulk_load(sb, blob, (uint32_t)(L.n_doubles * sizeof(double)), bar);
  mbar_wait(bar, 0);

  const TaylorTabs T = make_taylor_tabs(sb, L, a.n_pairs);
  const bool bad_rule = sb[0] != 0.0;

  const int S = 1 << a.split_log2;
  const long long gtid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  const long long point = gtid >> a.split_log2;
  const int sub = (int)(gtid & (S - 1));
  const bool active = point < a.n_points;

  cd x = {1.0, 0.0};
  if (active) {
    const double2 xv = a.x[point];
    x = {xv.x, xv.y};
  }
  // G_n(0) = 0 exactly; for 0 < |x| < 2^-200: G_n(x) = G_n(x 2^k) 2^(-k (n+1)), exact to O(|x|) (G_n = O(x^(n+1)))
  const bool is_zero = (x.re == 0.0 && x.im == 0.0);
  double out_scale = 1.0;
  const double xmax = fmax(fabs(x.re), fabs(x.im));
  if (is_zero) x = {1.0, 0.0};
  else if (xmax < 0x1p-200) {
    const int k = -200 - ilogb(xmax);
    x = {scalbn(x.re, k), scalbn(x.im, k)};
    out_scale = scalbn(1.0, -k * (N + 1));
  }
  const cd xinv = cinv(x);
  // zeta = (x + mu + y)^2/(4 x y) = C1/y + C2 + C3 y, as in eval_real_kernel
  cd C1x4[NT], C2[NT];
  const cd C3 = cscale(xinv, 0.25);
#pragma unroll
  for (int r = 0; r < NT; ++r) {
    const cd xm = {x.re + a.term[r].mu_re, x.im + a.term[r].mu_im};
    C2[r] = cmul(xm, cscale(xinv, 0.5));
    C1x4[r] = cscale(cmul(xm, C2[r]), 2.0);
  }
  double g_re = 0.0, g_im = 0.0;
#pragma unroll 1
  for (int i = sub; i < a.n_rad; i += S) {
    const double y = sb[L.off_y + i], q4 = sb[L.off_q4 + i];
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      const double2 icv = reinterpret_cast<const double2*>(sb + L.off_ic)[r * L.n_rad_pad + i];
      const double2 prv = reinterpret_cast<const double2*>(sb + L.off_pref)[r * L.n_rad_pad + i];
      const cd ic = {icv.x, icv.y};
      const cd xi = cmul(x, ic);                       // x/c
      const cd kap = cscale(ic, 4.0 * y);              // 4y/c
      const cd zeta = {fma(C1x4[r].re, q4, fma(C3.re, y, C2[r].re)), fma(C1x4[r].im, q4, fma(C3.im, y, C2[r].im))};
      const cd term = cmul(cd{prv.x, prv.y}, taylor_node<N>(T, x, cd{y, 0.0}, xi, kap, zeta, a.term[r]));
      g_re += term.re;
      g_im += term.im;
    }
  }
  for (int o = 1; o < S; o <<= 1) {
    g_re += __shfl_xor_sync(0xffffffffu, g_re, o);
    g_im += __shfl_xor_sync(0xffffffffu, g_im, o);
  }
  if (active && sub == 0) {
    if (is_zero) { g_re = 0.0; g_im = 0.0; }
    g_re *= out_scale;
    g_im *= out_scale;
    if (bad_rule) { g_re = nan(""); g_im = nan(""); }
    reinterpret_cast<double2*>(a.out)[point] = make_double2(g_re, g_im);
  }
}

// ---------------------------------------------------------------------------------------------
// The same on the point-dependent contours (RAY_ARC, THREAD, AUTO; gf_geometry.cuh): the thread walks the n_rad nodes
// of its point's contour (tables of gf_contour.cu's preparation: the REAL nodes, the ray's and the real tail's nodes
// of the point's rung; lines and arcs from the staged rules) and sends every node through taylor_node with complex y.
// Node weight: c0 (rule weight x dy/dt) y D1(y) R_r/(4y).  No tail series: the real tail's nodes take a route each.
// ---------------------------------------------------------------------------------------------
template <int N, int NT>
__global__ void __launch_bounds__(kBlockThreads, 2)
    eval_taylor_contour_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                               const double* __restrict__ blob) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
  double* sb = reinterpret_cast<double*>(smem_raw + 16);
  if (!workspace_matches(a, blob)) {
    const long long pt = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> a.split_log2;
    if (pt < a.n_points) reinterpret_cast<double2*>(a.out)[pt] = make_double2(nan(""), nan(""));
    if (blockIdx.x == 0 && threadIdx.x == 0) report_status(a.status, kStatusWorkspace);
    return;
  }
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) bulk_load(sb, blob, (uint32_t)(L.n_doubles * sizeof(double)), bar);
  mbar_wait(bar, 0);
  const TaylorTabs T = make_taylor_tabs(sb, L, a.n_pairs);
  const double* srt = sb + L.off_rt;
  const double* srw = sb + L.off_rw;
  const bool bad_rule = sb[0] != 0.0;

  const int S = 1 << a.split_log2;
  const long long gtid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  const long long point = gtid >> a.split_log2;
  const int sub = (int)(gtid & (S - 1));
  const bool active = point < a.n_points;
  cd x = {1.0, 0.0};
  if (active) {
    const double2 xv = a.x[point];
    x = {xv.x, xv.y};
  }
  const bool is_zero = (x.re == 0.0 && x.im == 0.0);
  double out_scale = 1.0;
  const double xmax = fmax(fabs(x.re), fabs(x.im));
  if (is_zero) x = {1.0, 0.0};
  else if (xmax < 0x1p-200) {
    const int k = -200 - ilogb(xmax);
    x = {scalbn(x.re, k), scalbn(x.im, k)};
    out_scale = scalbn(1.0, -k * (N + 1));
  }
  const cd xinv = cinv(x);
  const Geo geo = build_geo(a, x.re, x.im);
  const cd dir2 = ray_measure_dir(a, geo);   // dir^2 in d = 4
  const double* row = blob + L.off_rung + (long long)geo.row * L.rung_stride;
  const bool real_pol = geo.pol == GF_CONTOUR_REAL;
  const double* ty = real_pol ? blob + L.off_y : row + L.rg_y;
  const double* tq4 = real_pol ? blob + L.off_q4 : row + L.rg_yq4;
  const double2* tpref = reinterpret_cast<const double2*>(real_pol ? blob + L.off_pref : row + L.rg_pref);
  const int tstride = real_pol ? L.n_rad_pad : L.n4p;

  double g_re = 0.0, g_im = 0.0;
#pragma unroll 1
  for (int g = sub; g < a.n_rad; g += S) {
    const NodeAt at = locate(geo.pol, a.n_rad, g);
    const bool table = at.type == SEG_TABLE || at.type == SEG_TAIL;
    cd y, q4, W = {0.0, 0.0};
    if (table) {
      y = {ty[at.i], 0.0};
      q4 = {tq4[at.i], 0.0};
    } else {
      cd base;
      if (at.type == SEG_RAY) {
        const double r = row[L.rg_r + at.i], q4r = row[L.rg_q4 + at.i], rw = row[L.rg_w + at.i];
        y = {__dmul_rn(geo.dre, r), __dmul_rn(geo.dim, r)};
        q4 = {geo.dre * q4r, -geo.dim * q4r};
        base = {dir2.re * rw, dir2.im * rw};          // c0 wy y = c0 dir^2 r dr
      } else {
        const double t = srt[at.rule + at.i], w = srw[at.rule + at.i];
        cd wy;
        if (at.type == SEG_LINE) {
          const cd la = thread_waypoint(geo, at.k), lb = thread_waypoint(geo, at.k + 1);
          line_node(la, cd{__dadd_rn(lb.re, -la.re), __dadd_rn(lb.im, -la.im)}, t, w, &y, &wy);
        } else {
          arc_node(geo.R, geo.tau, t, w, &y, &wy);
        }
        base = measure_base(a, geo, at.type, at.k, t, y, wy);
        if (geo.mirror) { y.im = -y.im; wy.im = -wy.im; base.im = -base.im; }
        q4 = cscale(cinv_fast(y), 0.25);
      }
      W = cmul(cmul(base, line_k_complex(a, y)), q4);   // c0 wy y D1(y)/(4y)
    }
    const cd xq = cmul(xinv, q4);                       // 1/(4 x y)
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      const cd c = y_plus_mu(y, a.term[r]);
      const cd ic = cinv_fast(c);
      cd Wr;
      if (table) {   // the tables keep pref = c0 Wr y D1 (-R_r/(y + mu_r)):  W R_r/(4y) = -pref (y + mu_r)/(4y)
        const double2 p2 = tpref[r * tstride + at.i];
        Wr = cmul(cmul(cd{-p2.x, -p2.y}, c), q4);
      } else {
        Wr = NT == 1 ? W : cmul(W, cd{a.term[r].R_re, a.term[r].R_im});
      }
      const cd xi = cmul(x, ic);
      const cd kap = cscale(cmul(y, ic), 4.0);
      const cd xm = {x.re + a.term[r].mu_re, x.im + a.term[r].mu_im};
      const cd A = {xm.re + y.re, xm.im + y.im};
      const cd zeta = cmul(csqr(A), xq);
      const cd term = cmul(Wr, taylor_node<N>(T, x, y, xi, kap, zeta, a.term[r]));
      g_re += term.re;
      g_im += term.im;
    }
  }
  for (int o = 1; o < S; o <<= 1) {
    g_re += __shfl_xor_sync(0xffffffffu, g_re, o);
    g_im += __shfl_xor_sync(0xffffffffu, g_im, o);
  }
  if (active && sub == 0) {
    if (is_zero) { g_re = 0.0; g_im = 0.0; }
    g_re *= out_scale;
    g_im *= out_scale;
    if (bad_rule) { g_re = nan(""); g_im = nan(""); }
    reinterpret_cast<double2*>(a.out)[point] = make_double2(g_re, g_im);
  }
}

BlobLayout make_taylor_layout(int n_rad, int n_pairs, int n_terms, int order) {
  BlobLayout L = {};
  L.npad = (n_pairs + 3) & ~3;
  L.kmc = kKmc;
  L.n_poly = order + 2;
  long long o = 2;
  auto take = [&](long long n) { long long at = o; o += (n + 1) & ~1LL; return (int)at; };
  L.off_t = take(L.npad);
  L.off_tlo = take(L.npad);
  L.off_w = take(L.npad);
  L.off_kreq = take(kKreqBins / 2);
  L.off_momA = take((long long)kMomTerms * L.n_poly);
  L.off_chebA = take((long long)L.kmc * L.n_poly);
  L.n_rad_pad = (n_rad + 31) & ~31;
  L.n_pref = n_terms;
  L.off_y = take(L.n_rad_pad);
  L.off_q4 = take(L.n_rad_pad);
  L.off_pref = take(2LL * n_terms * L.n_rad_pad);
  L.off_ic = take(2LL * n_terms * L.n_rad_pad);
  L.n_doubles = (int)o;
  L.off_scratch = take((long long)L.kmc * L.npad);
  L.off_f32 = L.off_rt = L.off_rw = L.off_gam = L.off_gam2 = L.off_tail = L.off_scratch2 = L.off_scratch3 = -1;
  L.off_mom = L.off_cheb = L.off_sf = -1;
  L.n_blk = L.n_lev = L.n_blk_all = 0;
  L.off_blk = L.off_blkM = -1;
  L.off_blkS = -1;
  L.n_total = o;
  return L;
}

template <int N>
int launch_taylor_n(const EvalArgs& a, const LaunchPlan& plan, const double* blob, cudaStream_t stream) {
  auto launch = [&](auto kern) {
    if (plan.smem_bytes > 48 * 1024) {
      int rc = check_cuda(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes),
                          "cudaFuncSetAttribute(max dynamic shared memory)");
      if (rc) return rc;
    }
    kern<<<(unsigned)plan.grid_blocks, plan.block_threads, plan.smem_bytes, stream>>>(a, plan.layout, blob);
    return check_cuda(cudaGetLastError(), "taylor kernel launch");
  };
  if (!plan.shared_nodes)   // a point-dependent contour
    return a.n_terms == 1 ? launch(eval_taylor_contour_kernel<N, 1>) : launch(eval_taylor_contour_kernel<N, 2>);
  return a.n_terms == 1 ? launch(eval_taylor_kernel<N, 1>) : launch(eval_taylor_kernel<N, 2>);
}

}  // namespace

int plan_taylor(const EvalArgs& a, LaunchPlan* plan) {
  plan->block_threads = kBlockThreads;
  plan->shared_nodes = true;
  int sl = 0;
  const long long want = 148LL * 2 * kBlockThreads;
  while (sl < 5 && (a.n_points << sl) < want && (2 << sl) <= a.n_rad) ++sl;
  plan->split_log2 = sl;
  const long long threads = a.n_points << sl;
  plan->grid_blocks = (threads + kBlockThreads - 1) / kBlockThreads;
  plan->layout = make_taylor_layout(a.n_rad, a.n_pairs, a.n_terms, a.taylor_order);
  plan->smem_bytes = 16 + (size_t)plan->layout.n_doubles * sizeof(double);
  if (plan->smem_bytes > 200 * 1024) {
    set_error("eval_grid: tables need %zu bytes of shared memory (limit 200 KiB): reduce n_rad/n_ang", plan->smem_bytes);
    return GF_ERR_ARG;
  }
  if (plan->grid_blocks > 0x7fffffffLL) {
    set_error("eval_grid: too many points for one launch");
    return GF_ERR_ARG;
  }
  return GF_OK;
}

int launch_taylor_prepare(const EvalArgs& a, const LaunchPlan& plan, double* blob, cudaStream_t stream) {
  prep_taylor_kernel<<<1, 256, 0, stream>>>(a, plan.layout, blob);
  return check_cuda(cudaGetLastError(), "taylor preparation kernel launch");
}

int launch_taylor(const EvalArgs& a, const LaunchPlan& plan, const double* blob, cudaStream_t stream) {
  switch (a.taylor_order) {
    case 1: return launch_taylor_n<1>(a, plan, blob, stream);
    case 2: return launch_taylor_n<2>(a, plan, blob, stream);
    case 3: return launch_taylor_n<3>(a, plan, blob, stream);
    case 4: return launch_taylor_n<4>(a, plan, blob, stream);
    default: set_error("eval_grid: taylor_order %d out of range", a.taylor_order); return GF_ERR_UNSUPPORTED;
  }
}

}  // namespace gf
