// gf_eval.cu -- Step 5 / Kernel 2 of the paper: the double integral of
// eq. (14)/(15) for every grid point, as hand-written sm_100a CUDA.
//
// The sum that is computed:
//
//   G(x) = c0 sum_i Wr_i y_i D1(y_i) sum_j w'_j [ D2(u_ij) - D2(y_i) ],   u_ij = A_i - B_i z_j,
//   A_i = x + y_i + mu,  B_i = 2 sqrt(x) sqrt(y_i)                             eq. (10),(12),(20)
//
// How it is restructured for the FP64 pipe (none of this is in the paper):
//
//  * Line 2 is a sum of simple poles, D2(u) = sum_r R_r/(u + mu_r) (one term for 1/(u+m^2), two for the
//    rational propagator).  For one pole, with c = y + mu and A = x + c, a +-z pair of a symmetric
//    angular rule folds into
//        1/(A - Bz) + 1/(A + Bz) - 2/c = -(2/c) (eta - t)/(zeta - t),
//        t = z^2,  eta = A/(4y) = 1/4 + delta,  delta = (x + mu)/(4y),  zeta = A^2/(4xy),
//    which needs no square root of x or y.  Per (point, radial node, pole) the angular sum
//        S = sum_j w_j (eta - t_j)/(zeta - t_j)          (w_j: folded weights)
//    is the Cauchy transform of a fixed discrete measure on [0,1], analytic in zeta off [0,1].  It is
//    evaluated by one of four routes chosen from zeta alone (gf_routes.cuh, node_term):
//      MOMENT |zeta| large: geometric series in s = 1/(zeta - 1/2) with the centred moments of the rule,
//             at most 20 terms.
//      CHEB   Chebyshev series in s = 1/(w + sqrt(w^2-1)), w = 2 zeta - 1: 1/(zeta - t) = 4/sqrt(w^2-1)
//             sum'_k s^k T_k(2t-1), with the Chebyshev moments of the rule (made once per launch).  It
//             converges like rho^-k, rho = 1/|s| the parameter of the ellipse with foci 0 and 1 through
//             zeta, so a few tens of terms replace the N_a/2 pairs of the direct sum wherever the
//             radial node is not next to the image of the cut (median rho over the production scan: 3).
//             Both series have real coefficients and a complex argument and share one loop: the
//             second-order (Goertzel) recurrence, 2 DFMA per coefficient, 4 per term for the two
//             polynomials P (times delta) and N.  Cancellation free as x -> 0 and as y -> infinity.
//      NEAR   zeta close to [0,1] (rho < ~1.2): q_j = w_j/|zeta - t_j|^2 by one real reciprocal per PAIR
//             (MUFU.RCP64H seed + one cubic correction, 3 DFMA, no slow path), two real sums U0 = sum q_j,
//             U1 = sum q_j t_j, and S = mu_0 - (zeta - eta)(conj(zeta) U0 - U1).  8 FP64 instructions per pair.
//      EXACT  zeta within 2^-8 of the segment [0,1] (the radial contour passes next to a zero of a
//             denominator): zeta is recomputed in double-double and each term is formed directly with
//             a = (zeta_hi - t_hi) + (zeta_lo - t_lo), t_hi + t_lo = z^2 exactly.  Rare (a few nodes per
//             point outside the parabola where REAL is the continuation); without it such terms carry an
//             error eps/dist (reading G18).
//  * x = 0 gives exactly 0 (invariant I1); 0 < |x| < 2^-200 is rescaled (the sum is analytic at 0).
//  * A one-CTA preparation kernel makes every x-independent table once per launch (folded angular rule,
//    series coefficients, the radial map y_i in double-double so that it is correctly rounded, per-node
//    prefactors); each CTA of the evaluation kernel pulls that block into shared memory with ONE bulk copy
//    (cp.async.bulk + mbarrier, the 1-D TMA path) and reads it as warp-wide broadcasts.
//  * One thread owns one grid point (or 1/S of its radial nodes when the grid is too small to fill 148
//    SMs; the S lanes are merged with warp shuffles); the node loop is warp-synchronous (the series loop
//    of node_term runs to the warp's longest series); results leave as coalesced 16-byte stores.
#include <cstdlib>
#include <cfloat>
#include <cmath>
#include <cstdint>

#include "gf_dd.cuh"
#include "gf_internal.h"
#include "gf_routes.cuh"

namespace gf {
namespace {

__global__ void radial_map_kernel(double Lhi, double Llo, double s0, const double* __restrict__ nodes, int n,
                                  double* __restrict__ y) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) y[i] = radial_node(nodes[i], dd{Lhi, Llo}, s0);
}

// ---------------------------------------------------------------------------------------------
// Preparation: everything that does not depend on x, for the REAL contour.
//   header [0] = status bits of the tables;  t, t_lo, w (folded rule);  series coefficients mom[k], cheb[k], Kreq;
//   block tables of a split rule;  y_i, 1/(4 y_i);  pref_{r,i} = c0 Wr_i y_i D1(y_i) (-R_r/(y_i + mu_r));  the
//   tail's gamma and Rhat tables.
// Four CTAs with one role each, nothing exchanged between them (each folds the angular rule for itself: the same
// values to the same places): 0 the series tables and the checks, 1 the radial tables and the tail's Rhat, 2 the
// block tables, 3 the tail's gamma.  Their chains of dependent double-double steps run side by side instead of one
// after the other.
// ---------------------------------------------------------------------------------------------
constexpr int kPrepThreads = 1024, kPrepRoles = 4;
__global__ void __launch_bounds__(kPrepThreads) prep_real_kernel(const __grid_constant__ EvalArgs a,
                                                                 const __grid_constant__ BlobLayout L,
                                                                 double* __restrict__ blob) {
  __shared__ int bad;
  __shared__ dd s_mu[kTailN], s_nu[kTailN], s_part[8][2][kTailN];
  __shared__ float s_lc[kKmc];
  __shared__ dd s_cpart[8][2][kMomTerms];
  const int role = blockIdx.x;
  if (threadIdx.x == 0) bad = 0;
  __syncthreads();
  if (role != 1) prep_angular(a, L, blob, &bad);   // (role 1 reads nothing of the angular rule)
  if (role == 0) check_radial_tables(a, &bad);
  __syncthreads();  // t, w written by this CTA are visible to it
  if (role == 0) {
    prep_series_T(a, L, blob);
    if (L.off_rt >= 0) {  // point-dependent contours: levels 2 and 3 of the rule pyramid as given ("n arrays",
                          // PAPER.md:150; levels 0 and 1 are mapped once per launch: REAL tables, rung tables)
      const int lvl2 = a.n_rad + a.n_rad / 2;
      for (int i = threadIdx.x; i < L.n_tab; i += blockDim.x) {
        blob[L.off_rt + i] = a.rad_nodes[lvl2 + i];
        blob[L.off_rw + i] = a.rad_weights[lvl2 + i];
      }
    }
    __syncthreads();  // the T_k(s_j) matrix is complete
    prep_series_sums(a, L, blob, s_cpart);
    if (L.n_poly) prep_series_A(a, L, blob);
    __syncthreads();
    // Kreq from the tables the evaluation kernel will run: order 0's two, or the n + 2 of a Taylor order
    if (L.n_poly) prep_series_kreq(L, blob, s_lc, blob + L.off_chebA, L.n_poly);
    else prep_series_kreq(L, blob, s_lc, blob + L.off_cheb, 2);
    if (threadIdx.x == 0) {
      blob[0] = (double)bad;
      blob[1] = a.ws_tag;
      if (bad) report_status(a.status, bad);
    }
  } else if (role == 1) {
    // shifted-log map of [0, Lambda^2] (readings G3/G4): y(u) = s0 expm1(u L), dy/du = L (y + s0),
    // L = ln((Lambda^2 + s0)/s0) as a double-double from the host; y_i correctly rounded.
    const dd Llog = {a.Llog_hi, a.Llog_lo};
    for (int ip = threadIdx.x; ip < L.n_rad_pad; ip += blockDim.x) {
      const int i = min(ip, a.n_rad - 1);            // padding: the last node again, prefactor 0
      const double y = radial_node(a.rad_nodes[i], Llog, a.s0);
      const double Wr = ip < a.n_rad ? 0.5 * a.rad_weights[i] * a.Llog_hi * (y + a.s0) : 0.0;
      blob[L.off_y + ip] = y;
      blob[L.off_q4 + ip] = 0.25 / y;
      // radial measure dy y^((d-2)/2): y itself in d = 4 (eq. (14)), pow otherwise
      // symmetric routing: D1 D2 at x = 0 is 1/(y + mu)^2 for both lines together (line_k == line_pk, massive)
      const cd d1 = cscale(a.routing == 1 ? cinv(cd{y + a.term[0].mu_re, a.term[0].mu_im}) : line_k_real(a.line_k, y),
                           a.c0 * Wr * (a.ypow == 1.0 ? y : pow(y, a.ypow)));
      for (int r = 0; r < a.n_terms; ++r) {
        const cd ic = cinv(cd{y + a.term[r].mu_re, a.term[r].mu_im});
        const cd pr = cmul(cmul(d1, cd{-a.term[r].R_re, -a.term[r].R_im}), ic);
        blob[L.off_pref + 2 * (r * L.n_rad_pad + ip)] = pr.re;
        blob[L.off_pref + 2 * (r * L.n_rad_pad + ip) + 1] = pr.im;
        if (L.n_pref > a.n_terms) {   // symmetric routing, tail table 1: pref (1 + mu/y)/4
          const cd f = {0.25 + a.term[0].mu_re * (0.25 / y), a.term[0].mu_im * (0.25 / y)};
          const cd p2 = cmul(pr, f);
          blob[L.off_pref + 2 * (a.n_terms * L.n_rad_pad + ip)] = p2.re;
          blob[L.off_pref + 2 * (a.n_terms * L.n_rad_pad + ip) + 1] = p2.im;
        }
      }
    }
    __syncthreads();  // the radial tables are complete
    if (L.off_gam >= 0) {
      const TailJob J = real_tail_job(a, L, blob);
      prep_tail_powers(J);
      __syncthreads();
      prep_tail_sums(J);
    }
  } else if (role == 2) {
    prep_blocks_T(a, L, blob);
    __syncthreads();
    prep_blocks_sums(a, L, blob);
  } else if (L.off_gam >= 0) {
    prep_tail_moments(a, L, blob, s_part);
    __syncthreads();  // the monomial moments are complete
    prep_tail_gamma(L, blob, s_part, s_mu, s_nu);
  }
}

// ---------------------------------------------------------------------------------------------
// Evaluation, REAL contour.  counters (COUNT only): gf.h, gf_eval_grid_counted.
// ---------------------------------------------------------------------------------------------
#ifndef GF_MIN_BLOCKS
#define GF_MIN_BLOCKS 4
#endif
// SPLIT = false: one thread per point known at compile time (the node pointers are then warp-uniform: no lane
// registers, nothing of the node loop's bookkeeping in local memory)
template <typename T, bool COUNT, int NT, bool BLK, bool SPLIT>
__global__ void __launch_bounds__(kBlockThreads, GF_MIN_BLOCKS)
    eval_real_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                     const double* __restrict__ blob, unsigned long long* __restrict__ counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
  double* sb = reinterpret_cast<double*>(smem_raw + 16);
  if (!workspace_matches(a, blob)) {   // prepared for other parameters or orders: refuse it before reading a table
    const long long pt = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> a.split_log2;
    if (pt < a.n_points) {
      if (sizeof(T) == 8) reinterpret_cast<double2*>(a.out)[pt] = make_double2(nan(""), nan(""));
      else reinterpret_cast<float2*>(a.out)[pt] = make_float2(nanf(""), nanf(""));
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) report_status(a.status, kStatusWorkspace);
    return;
  }
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) bulk_load(sb, blob, (uint32_t)(L.n_doubles * sizeof(double)), bar);
  mbar_wait(bar, 0);

  const Tabs<T> tb = make_tabs<T>(sb, L, a.n_pairs);
  const bool bad_rule = sb[0] != 0.0;

  const int S = SPLIT ? 1 << a.split_log2 : 1;
  const long long gtid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  const long long point = SPLIT ? gtid >> a.split_log2 : gtid;
  const int sub = SPLIT ? (int)(gtid & (S - 1)) : 0;
  const bool active = point < a.n_points;

  cd x = {1.0, 0.0};
  if (active) {
    const double2 xv = a.x[point];
    x = {xv.x, xv.y};
  }
  // G(0) = 0 exactly (invariant I1); for 0 < |x| < 2^-200 use G(x) = G(x 2^k) 2^-k with |x 2^k| ~ 2^-200,
  // exact to O(|x|) because the sum is analytic at 0 and vanishes there (keeps zeta inside the FP64 range).
  const bool is_zero = (x.re == 0.0 && x.im == 0.0);
  double out_scale = 1.0;
  const double xmax = fmax(fabs(x.re), fabs(x.im));
  if (is_zero) x = {1.0, 0.0};
  else if (xmax < 0x1p-200) {
    const int k = -200 - ilogb(xmax);
    x = {scalbn(x.re, k), scalbn(x.im, k)};
    out_scale = scalbn(1.0, -k);
  }
  const cd xinv = cinv(x);
  // zeta = (x + mu + y)^2/(4 x y) = C1/y + C2 + C3 y with C1 = (x + mu)^2/(4x), C2 = (x + mu)/(2x), C3 = 1/(4x):
  // four DFMA per node-term.  Its absolute error is an ulp of the largest of the three terms, which is O(1)
  // wherever zeta is O(1) (the EXACT route recomputes zeta in double-double from x, y, mu anyway).
  // Symmetric routing (gf_params.routing = 1; lines carry k + p/2 and k - p/2, equal masses): the folded sum is
  // the same S with  zeta' = (y + x/4 + mu)^2/(x y) = zeta(x/4, y, mu)  and  eta' = 1/2 + (2 mu + x/4)/(4y),
  // and the node prefactor is -c0 Wr y/(y + mu)^2 (made in the preparation kernel).
  cd xm[NT], C1x4[NT], C2[NT], dA[NT];  // x + mu_r, 4 C1 (multiplies 1/(4y)), C2, delta = d0 + dA/(4y)
  cd C3 = cscale(xinv, 0.25);
  cd xz = x;                            // the "x" of zeta (the EXACT route recomputes zeta from it)
  double d0 = 0.0;
  if (a.routing == 1) {
    xz = cscale(x, 0.25);
    C3 = xinv;                          // 1/(4 (x/4))
    d0 = 0.25;
  }
#pragma unroll
  for (int r = 0; r < NT; ++r) {
    xm[r] = {x.re + a.term[r].mu_re, x.im + a.term[r].mu_im};
    dA[r] = xm[r];
    cd az = xm[r], izx2 = cscale(xinv, 0.5);   // a = xz + mu, 1/(2 xz)
    if (a.routing == 1) {
      az = {xz.re + a.term[r].mu_re, xz.im + a.term[r].mu_im};
      izx2 = cscale(xinv, 2.0);
      dA[r] = {xz.re + 2.0 * a.term[r].mu_re, xz.im + 2.0 * a.term[r].mu_im};
    }
    C2[r] = cmul(az, izx2);
    C1x4[r] = cscale(cmul(az, C2[r]), 2.0);
  }

  // where the tail series takes over: the first node with y_i >= Y0 = 4 (sqrt|x| + sqrt(|x| + |x + mu|))^2
  int i_end = a.n_rad;
  if (L.off_gam >= 0) {
    const double ax = sqrt(fma(x.re, x.re, x.im * x.im));
    double Y0 = 0.0;
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      // symmetric routing: zeta' = zeta(x/4, y, mu), the same bound with x/4 and a' = x/4 + mu
      const cd az = {xz.re + a.term[r].mu_re, xz.im + a.term[r].mu_im};
      const double axz = a.routing == 1 ? 0.25 * ax : ax;
      const double q = sqrt(axz) + sqrt(axz + sqrt(fma(az.re, az.re, az.im * az.im)));
      Y0 = fmax(Y0, kTailFactor * q * q);
    }
    int lo = 0, hi = a.n_rad;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (sb[L.off_y + mid] < Y0) lo = mid + 1; else hi = mid;
    }
    i_end = lo;
  }
  const int i_stop = __reduce_max_sync(0xffffffffu, i_end);

  RouteCount rc;
  double g_re = 0.0, g_im = 0.0;
  // warp-synchronous node loop: every lane makes the same number of trips (node_term is warp-collective);
  // the node tables are padded to a multiple of 32 with zero-weight copies of the last node
  const double* py = sb + L.off_y + sub;
  const double* pq4 = sb + L.off_q4 + sub;
  const double2* ppref = reinterpret_cast<const double2*>(sb + L.off_pref) + sub;
#pragma unroll 1
  for (int i0 = 0; i0 < i_stop; i0 += S, py += S, pq4 += S, ppref += S) {
    const double y = *py, q4 = *pq4;
    const bool on = i0 + sub < i_end;                // past its own i_end a lane idles with weight 0
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      const cd delta = {fma(dA[r].re, q4, d0), dA[r].im * q4};   // eta - 1/4
      const cd zeta = {fma(C1x4[r].re, q4, fma(C3.re, y, C2[r].re)), fma(C1x4[r].im, q4, fma(C3.im, y, C2[r].im))};
      // (the lo parts of a rational line's poles matter where a contour passes next to y = -mu: not on the real axis)
      const cd s = node_term<T, COUNT, BLK>(tb, xz, cd{y, 0.0}, delta, zeta, a.term[r].mu_re, a.term[r].mu_im, rc);
      const double2 pr = ppref[r * L.n_rad_pad];
      if (on) {   // (four predicated DFMA; an idle lane's s may be anything)
        g_re = fma(pr.x, s.re, fma(-pr.y, s.im, g_re));
        g_im = fma(pr.x, s.im, fma(pr.y, s.re, g_im));
      }
    }
  }
  if (L.off_gam >= 0 && __any_sync(0xffffffffu, i_end < a.n_rad)) {
    const double invy0 = 4.0 * sb[L.off_q4 + min(i_end, a.n_rad - 1)];
    const double2* R = reinterpret_cast<const double2*>(blob + L.off_tail) + (size_t)i_end * kTailN;
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      const cd az = {xz.re + a.term[r].mu_re, xz.im + a.term[r].mu_im};   // x + mu, or x/4 + mu
      cd tl = tail_series(sb + L.off_gam, R + (size_t)r * (a.n_rad + 1) * kTailN, xz, az, invy0);
      if (L.off_gam2 >= 0)   // symmetric routing: S' = S(x/4, a') + (1 + mu/y)/4 sum_j w_j/(zeta' - t_j)
        tl = cadd(tl, tail_series(sb + L.off_gam2, R + (size_t)NT * (a.n_rad + 1) * kTailN, xz, az, invy0));
      if (sub == 0) {
        g_re += tl.re;
        g_im += tl.im;
      }
      if (COUNT) ++rc.tails;
    }
  }
  // merge the S lanes that share a point
  for (int o = 1; o < S; o <<= 1) {
    g_re += __shfl_xor_sync(0xffffffffu, g_re, o);
    g_im += __shfl_xor_sync(0xffffffffu, g_im, o);
  }
  if (active && sub == 0) {
    if (is_zero) { g_re = 0.0; g_im = 0.0; }
    g_re *= out_scale;
    g_im *= out_scale;
    if (bad_rule) { g_re = nan(""); g_im = nan(""); }
    if (sizeof(T) == 8) reinterpret_cast<double2*>(a.out)[point] = make_double2(g_re, g_im);
    else reinterpret_cast<float2*>(a.out)[point] = make_float2((float)g_re, (float)g_im);
  }
  if (COUNT) flush_counters(rc, active, counters);
}

}  // namespace

// pyramid: the layout of the deformed-contour kernel (gf_contour.cu).  It stages the angular rule, the series
// tables, levels 2 and 3 of the radial pyramid and the tail's gamma table; the REAL node tables (read by the points
// AUTO sends to REAL), every Rhat table and the rung tables stay in global memory.
BlobLayout make_blob_layout(int n_rad, int n_pairs, int n_terms, bool f32, bool pyramid, bool tail, bool sym,
                            int taylor_order) {
  BlobLayout L = {};
  L.npad = (n_pairs + 3) & ~3;
  L.kmc = kKmc;
  long long o = 2;  // header
  auto take = [&](long long n) { long long at = o; o += (n + 1) & ~1LL; return at; };
  // the tables every node-term reads come first, at offsets known at compile time (kOffMom ... kOffSf: the kernels
  // address them as one base plus immediates); four entries of slack below the float2 series tables (the
  // software-pipelined loop reads them on its last trip), 2 float2 tables of kmc entries = 2 kmc doubles
  L.off_mom = (int)take(2 * L.kmc);
  L.off_cheb = (int)take(2 * L.kmc);
  L.off_kreq = (int)take(kKreqBins / 2);
  take(4);
  L.off_sf = (int)take(2 * L.kmc);
  static_assert(kOffSf % 2 == 0, "float2 tables must be 16-byte aligned");
  if (L.off_mom != kOffMom || L.off_cheb != kOffCheb || L.off_kreq != kOffKreq || L.off_sf != kOffSf) abort();
  L.off_t = (int)take(L.npad);
  L.off_tlo = (int)take(L.npad);
  L.off_w = (int)take(L.npad);
  L.n_rad_pad = (n_rad + 31) & ~31;
  L.n_pref = n_terms + (sym && tail ? 1 : 0);
  auto take_nodes = [&]() {
    L.off_y = (int)take(L.n_rad_pad);
    L.off_q4 = (int)take(L.n_rad_pad);
    L.off_pref = (int)take(2 * L.n_pref * L.n_rad_pad);
  };
  if (!pyramid) take_nodes();
  // FP32 variant: 2 float tables of npad entries = npad doubles
  L.off_f32 = f32 ? (int)take(L.npad) : -1;
  L.n_tab = pyramid ? n_rad / 4 + n_rad / 8 : 0;
  L.off_rt = pyramid ? (int)take(L.n_tab) : -1;
  L.off_rw = pyramid ? (int)take(L.n_tab) : -1;
  L.off_gam = tail ? (int)take(kTailN * (kTailN + 1) / 2) : -1;
  L.off_gam2 = tail && sym ? (int)take(kTailN * (kTailN + 1) / 2) : -1;
  // Taylor order n > 0 on a deformed contour (gf_taylor.cu): the n + 2 series tables per family, staged
  L.n_poly = taylor_order > 0 ? taylor_order + 2 : 0;
  L.off_momA = L.n_poly ? (int)take((long long)kMomTerms * L.n_poly) : -1;
  L.off_chebA = L.n_poly ? (int)take((long long)L.kmc * L.n_poly) : -1;
  L.off_ic = -1;
  L.n_blk = n_pairs >= (pyramid ? kBlkMinPairsContour : kBlkMinPairs) ? (n_pairs + kBlkPairs - 1) / kBlkPairs : 0;
  L.n_lev = 0;
  L.n_blk_all = 0;
  for (int l = 0, n = L.n_blk; l < kBlkMaxLev && n > 0; ++l) {   // levels up to the one that has a single block
    L.lev_off[l] = L.n_blk_all;
    L.n_blk_all += n;
    L.n_lev = l + 1;
    if (n == 1) break;
    n = (n + 1) / 2;
  }
  L.off_blk = L.n_blk ? (int)take(2 * L.n_blk_all) : -1;
  L.off_blkM = L.n_blk ? (int)take((long long)L.n_blk_all * kBlkTerms) : -1;
  L.n_doubles = (int)o;
  if (pyramid) take_nodes();
  L.off_tail = tail ? (int)take(2LL * L.n_pref * (n_rad + 1) * kTailN) : -1;
  L.off_scratch = (int)take((long long)L.kmc * L.npad);
  L.off_blkS = L.n_blk ? take(2LL * kBlkTerms * L.npad * L.n_lev) : -1;
  L.off_scratch2 = tail ? (int)take(2LL * kTailN * n_rad) : -1;
  L.off_scratch3 = tail ? (int)take((long long)kTailN * n_rad + 2 * kTailChunks * (2 * L.n_pref * kTailN + kTailN)) : -1;
  L.n_rungs = 0;
  if (pyramid && tail) {
    const int n2 = n_rad / 2, n4 = n_rad / 4;
    L.n4p = (n4 + 1) & ~1;
    long long ro = 0;
    auto rtake = [&](long long n) { long long at = ro; ro += (n + 1) & ~1LL; return (int)at; };
    L.rg_r = rtake(n2);
    L.rg_q4 = rtake(n2);
    L.rg_w = rtake(n2);
    L.rg_y = rtake(L.n4p);
    L.rg_yq4 = rtake(L.n4p);
    L.rg_pref = rtake(2LL * n_terms * L.n4p);
    L.rg_tail = rtake(2LL * n_terms * (n4 + 1) * kTailN);
    L.rg_s2 = rtake(2LL * kTailN * n4);
    L.rg_s3 = rtake((long long)kTailN * n4 + 2 * kTailChunks * (2 * n_terms * kTailN + kTailN));
    L.rung_stride = ro;
    L.n_rungs = kRungs + 1;
    L.off_rung = take(ro * L.n_rungs);
  }
  L.n_total = o;
  return L;
}


// ---------------------------------------------------------------------------------------------
int plan_eval(const EvalArgs& a, int precision, LaunchPlan* plan) {
  if (a.taylor_order > 0 && a.contour == GF_CONTOUR_REAL) return plan_taylor(a, plan);
  plan->block_threads = kBlockThreads;
  plan->shared_nodes = (a.contour == GF_CONTOUR_REAL);
  // lanes per point: enough threads for >= 2 CTAs on each of the 148 SMs, at most a warp
  int sl = 0;
  const long long want = 148LL * 2 * kBlockThreads;
  while (sl < 5 && (a.n_points << sl) < want && (2 << sl) <= a.n_rad) ++sl;
  plan->split_log2 = sl;
  const long long threads = a.n_points << sl;
  plan->grid_blocks = (threads + kBlockThreads - 1) / kBlockThreads;
  plan->layout = make_blob_layout(a.n_rad, a.n_pairs, a.n_terms, precision == 32, !plan->shared_nodes, true,
                                 a.routing == 1, a.taylor_order);
  plan->smem_bytes = 16 + (size_t)plan->layout.n_doubles * sizeof(double);
  if (plan->smem_bytes > 200 * 1024) {
    set_error("eval_grid: tables need %zu bytes of shared memory (limit 200 KiB): reduce n_rad/n_ang",
              plan->smem_bytes);
    return GF_ERR_ARG;
  }
  if (plan->grid_blocks > 0x7fffffffLL) {
    set_error("eval_grid: too many points for one launch");
    return GF_ERR_ARG;
  }
  return GF_OK;
}

template <typename T, bool COUNT, int NT, bool BLK, bool SPLIT>
static int launch_real_kern(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* counters,
                            cudaStream_t stream) {
  auto kern = eval_real_kernel<T, COUNT, NT, BLK, SPLIT>;
  if (plan.smem_bytes > 48 * 1024) {
    int rc = check_cuda(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes),
                        "cudaFuncSetAttribute(max dynamic shared memory)");
    if (rc) return rc;
  }
  kern<<<(unsigned)plan.grid_blocks, plan.block_threads, plan.smem_bytes, stream>>>(a, plan.layout, blob, counters);
  return check_cuda(cudaGetLastError(), "eval kernel launch");
}
// the kernel instantiation for this launch: the unsplit one exists for the timed FP64 kernels only, the blocked one
// for FP64 only
template <typename T, bool COUNT, int NT, bool BLK>
static int launch_real_nt(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* counters,
                          cudaStream_t stream) {
  if constexpr (!COUNT && sizeof(T) == 8)
    if (a.split_log2 == 0) return launch_real_kern<T, COUNT, NT, BLK, false>(a, plan, blob, counters, stream);
  return launch_real_kern<T, COUNT, NT, BLK, true>(a, plan, blob, counters, stream);
}
template <typename T, bool COUNT>
static int launch_real(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* counters,
                       cudaStream_t stream) {
  if constexpr (sizeof(T) == 8)
    if (plan.layout.n_blk > 0)
      return a.n_terms == 1 ? launch_real_nt<T, COUNT, 1, true>(a, plan, blob, counters, stream)
                            : launch_real_nt<T, COUNT, 2, true>(a, plan, blob, counters, stream);
  return a.n_terms == 1 ? launch_real_nt<T, COUNT, 1, false>(a, plan, blob, counters, stream)
                        : launch_real_nt<T, COUNT, 2, false>(a, plan, blob, counters, stream);
}

int launch_radial_map(double Llog_hi, double Llog_lo, double s0, const double* d_nodes, int n, double* d_y,
                      cudaStream_t stream) {
  radial_map_kernel<<<(n + 127) / 128, 128, 0, stream>>>(Llog_hi, Llog_lo, s0, d_nodes, n, d_y);
  return check_cuda(cudaGetLastError(), "radial_map launch");
}

static int check_variant(const LaunchPlan& plan, int precision) {
  if (!plan.shared_nodes && precision == 32) {
    set_error("eval_grid: the FP32 comparison variant exists for the REAL contour only");
    return GF_ERR_UNSUPPORTED;
  }
  return GF_OK;
}

// Preparation alone: the x-independent tables of this (params, rules) into `blob` (plan.layout.n_total doubles).
int launch_prepare(const EvalArgs& a, int precision, double* blob, cudaStream_t stream) {
  LaunchPlan plan;
  int rc = plan_eval(a, precision, &plan);
  if (rc) return rc;
  if ((rc = check_variant(plan, precision))) return rc;
  if (a.taylor_order > 0 && plan.shared_nodes) return launch_taylor_prepare(a, plan, blob, stream);
  prep_real_kernel<<<kPrepRoles, kPrepThreads, 0, stream>>>(a, plan.layout, blob);
  if ((rc = check_cuda(cudaGetLastError(), "prep kernel launch"))) return rc;
  return plan.shared_nodes ? GF_OK : launch_prepare_rungs(a, plan, blob, stream);
}

// Evaluation alone, from tables made by launch_prepare with the same params, orders and precision.
int launch_prepared(const EvalArgs& a_in, int precision, const double* blob, unsigned long long* d_counters,
                    cudaStream_t stream) {
  if (a_in.n_points == 0) return GF_OK;
  LaunchPlan plan;
  int rc = plan_eval(a_in, precision, &plan);
  if (rc) return rc;
  if ((rc = check_variant(plan, precision))) return rc;
  EvalArgs a = a_in;
  a.split_log2 = plan.split_log2;
  if (a.taylor_order > 0) {
    if (d_counters) { set_error("eval_grid_counted: the route counters exist for taylor_order 0 only"); return GF_ERR_UNSUPPORTED; }
    return launch_taylor(a, plan, blob, stream);
  }
  if (!plan.shared_nodes) return launch_contour(a, plan, blob, d_counters, stream);
  if (d_counters)
    return precision == 32 ? launch_real<float, true>(a, plan, blob, d_counters, stream)
                           : launch_real<double, true>(a, plan, blob, d_counters, stream);
  return precision == 32 ? launch_real<float, false>(a, plan, blob, nullptr, stream)
                         : launch_real<double, false>(a, plan, blob, nullptr, stream);
}

int launch_eval(const EvalArgs& a, int precision, unsigned long long* d_counters, cudaStream_t stream) {
  if (a.n_points == 0) return GF_OK;
  LaunchPlan plan;
  int rc = plan_eval(a, precision, &plan);
  if (rc) return rc;
  // scratch for the prepared tables: stream-ordered, freed in stream order after the evaluation
  double* blob = nullptr;
  if ((rc = scratch_alloc(reinterpret_cast<void**>(&blob), (size_t)plan.layout.n_total * sizeof(double), stream))) return rc;
  rc = launch_prepare(a, precision, blob, stream);
  if (!rc) rc = launch_prepared(a, precision, blob, d_counters, stream);
  cudaFreeAsync(blob, stream);
  return rc;
}

}  // namespace gf
