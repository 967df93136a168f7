// gf_contour.cu -- Step 3 inside Kernel 2: evaluation on radial contours
// that depend on the grid point.  The paper's Kernel 2 picks one of four hand-made contours per thread
// with an IF-THEN-ELSE on the region of x; here each thread builds its contour from x by one of the
// policies of include/gf.h (gf_contour) and walks its nodes:
//
//   REAL     [0, Lambda^2], shifted-log map (nodes prepared once per launch, as in gf_eval.cu);
//   RAY_ARC  ray y = r x/|x|, r in [0,R] shifted-log (n_rad/2 nodes), arc of |y| = R back to the real axis
//            (n_rad/4), real tail [R, Lambda^2] shifted-log (n_rad/4);  R the smallest rung of the ladder
//            {2^k, 1.5 2^k} above 1.5 (sqrt|x| + sqrt(|x|+sc))^2, sc the size of line 2's singular structure,
//            Lambda^2/2 beyond the ladder (generalises the paper's region-2/5 contour);
//   THREAD   equal real masses, next to the negative axis below -4 m^2: five straight pieces through
//            the waypoints W0..W5 that pass the pole of line 1 and thread the opening of the cut at
//            |x + m^2| x/|x|, an arc from 3 pi/4 to 0 and the real tail (n_rad/8 nodes each, n_rad/4
//            on the tail); mirrored for Im x < 0 (the analogue of the region-3/4 polylines);
//   AUTO     per point: REAL inside the parabola where it is the continuation, THREAD next to the cut, RAY_ARC
//            elsewhere (auto_policy below).
//
// The geometry uses no angle: the direction of the ray is x/|x| by two correctly rounded divisions, arcs are the
// rational parametrisation y = R ((1 + i tau v)/(1 - i tau v))^2, every operation is a +, -, *, /, sqrt written
// with the _rn intrinsics in the order gf.h states, so the nodes are the same doubles as the oracle's on any IEEE
// machine.  Because R comes from a ladder, the radial nodes of the ray and of the real tail do not depend on x
// beyond the choice of the rung: a preparation kernel maps them once per launch (one CTA per rung, in
// double-double, correctly rounded like the REAL contour's, reading G18) together with the tail's node
// prefactors and its Rhat tables, so the large-y part of the real tail costs one tail series per point as on
// the REAL contour (gf_routes.cuh, tail_series).
// Per node the angular sum is the same folded sum S(eta, zeta) as on the REAL contour (gf_routes.cuh):
// with complex y, eta = (x + y + mu)/(4y) and zeta = (x + y + mu)^2/(4xy) are simply complex.
#include "gf_geometry.cuh"
#include "gf_routes.cuh"

namespace gf {
namespace {

// ---------------------------------------------------------------------------------------------
// Rung tables (one CTA per row): the ray's and the real tail's nodes for the contour radius R_k, the tail's node
// prefactors pref_{r,i} = c0 Wr_i y_i D1(y_i) (-R_r/(y_i + mu_r)) and its Rhat tables.  Rows whose radius is not
// below Lambda^2/2 are never read and stay unwritten; the last row is R = Lambda^2/2.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) prep_rungs_kernel(const __grid_constant__ EvalArgs a,
                                                         const __grid_constant__ BlobLayout L,
                                                         double* __restrict__ blob) {
  const int k = blockIdx.x;
  double R = 0.5 * a.cutoff2;
  if (k < kRungs) {
    R = rung_value(a.rung_lo + k);
    if (!(R < 0.5 * a.cutoff2)) return;
  }
  double* row = blob + L.off_rung + (long long)k * L.rung_stride;
  const int n = a.n_rad, n2 = n >> 1, n4 = n >> 2;
  // ray: r(u) = s0 expm1(u L), L = ln((R + s0)/s0), dr = (w/2) L (r + s0)            (level 1 of the pyramid)
  const dd L1 = dd_log(dd_div_d(two_sum(R, a.s0), a.s0));
  for (int i = threadIdx.x; i < n2; i += blockDim.x) {
    const double t = a.rad_nodes[n + i], w = a.rad_weights[n + i];
    const double r = radial_node(t, L1, a.s0);
    const double dr = dd_mul(dd_mul_d(L1, 0.5 * w), two_sum(r, a.s0)).hi;
    row[L.rg_r + i] = r;
    row[L.rg_q4 + i] = 0.25 / r;
    row[L.rg_w + i] = a.c0 * (a.ypow == 1.0 ? r : pow(r, a.ypow)) * dr;   // c0 r^p dr, p = (d-2)/2
  }
  // real tail: y(u) = R + (R + s0) expm1(u L), L = ln((Lambda^2 + s0)/(R + s0))      (level 2)
  const dd as = two_sum(R, a.s0);
  const dd L2 = dd_log(dd_div(two_sum(a.cutoff2, a.s0), as));
  for (int i = threadIdx.x; i < L.n4p; i += blockDim.x) {
    const int ii = min(i, n4 - 1);
    const double t = a.rad_nodes[n + n2 + ii], w = i < n4 ? a.rad_weights[n + n2 + ii] : 0.0;
    const double u = 0.5 * (t + 1.0);
    const double y = dd_add_d(dd_mul(as, dd_expm1(dd_mul_d(L2, u))), R).hi;
    const double dy = dd_mul(dd_mul_d(L2, 0.5 * w), two_sum(y, a.s0)).hi;
    row[L.rg_y + i] = y;
    row[L.rg_yq4 + i] = 0.25 / y;
    const cd d1 = cscale(line_k_real(a.line_k, y), a.c0 * dy * (a.ypow == 1.0 ? y : pow(y, a.ypow)));
    for (int r = 0; r < a.n_terms; ++r) {
      const cd ic = cinv(cd{y + a.term[r].mu_re, a.term[r].mu_im});
      const cd pr = cmul(cmul(d1, cd{-a.term[r].R_re, -a.term[r].R_im}), ic);
      row[L.rg_pref + 2 * (r * L.n4p + i)] = pr.re;
      row[L.rg_pref + 2 * (r * L.n4p + i) + 1] = pr.im;
    }
  }
  __syncthreads();
  const TailJob J = {n4, a.n_terms, L.n4p, row + L.rg_y, row + L.rg_pref, reinterpret_cast<double2*>(row + L.rg_tail),
                     row + L.rg_s2, row + L.rg_s3};
  prep_tail_powers(J);
  __syncthreads();
  prep_tail_sums(J);
}

// ---------------------------------------------------------------------------------------------
// Evaluation on point-dependent contours.  Same staging, lane split, routes, reductions and store as
// eval_real_kernel; counters as there.
// ---------------------------------------------------------------------------------------------
#ifndef GF_CONTOUR_MIN_BLOCKS
#define GF_CONTOUR_MIN_BLOCKS 4
#endif
// POL >= 0: every point of the launch walks this policy (an explicit gf_params.contour), known at compile time: the
// other policies' code and registers are gone; POL = -1: the policy is each point's own (AUTO)
template <bool COUNT, int NT, bool BLK, int POL>
__global__ void __launch_bounds__(kBlockThreads, GF_CONTOUR_MIN_BLOCKS)
    eval_contour_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                        const double* __restrict__ blob, unsigned long long* __restrict__ counters) {
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

  const Tabs<double> tb = make_tabs<double>(sb, L, a.n_pairs);
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
  // G(0) = 0 exactly (invariant I1); 0 < |x| < 2^-200 rescaled as in eval_real_kernel
  const bool is_zero = (x.re == 0.0 && x.im == 0.0);
  double out_scale = 1.0;
  const double xmax = fmax(fabs(x.re), fabs(x.im));
  if (is_zero) x = {1.0, 0.0};
  else if (xmax < 0x1p-200) {
    const int k = -200 - ilogb(xmax);
    x = {scalbn(x.re, k), scalbn(x.im, k)};
    out_scale = scalbn(1.0, -k);
  }
  // Symmetric routing (lines k + p/2, k - p/2; equal massive lines): the folded sum is S(eta', zeta') with
  // zeta' = zeta(x/4, y, mu) and eta' = 1/2 + (2 mu + x/4)/(4y), the node prefactor -c0 wy y/(y + mu)^2 as for equal masses,
  // and the cut is the paper routing's at x/4: from here on x IS x/4 (geometry, policy, zeta); only delta differs.
  const bool sym = a.routing == 1;
  if (sym) x = cscale(x, 0.25);
  const double d0 = sym ? 0.25 : 0.0, dmu = sym ? 2.0 : 1.0;   // delta = d0 + (x + dmu mu)/(4y)
  const cd xinv = cinv(x);

  const Geo geo = build_geo(a, x.re, x.im, POL);
  const int pol = POL >= 0 ? POL : geo.pol;
  const cd dir2 = ray_measure_dir(a, geo);   // dir^2 in d = 4
  // One pole (NT == 1): on a piece y = dir r with real r from a table (the ray; dir = 1 on the real pieces)
  //   zeta = (x + mu + y)^2/(4 x y) = Z1/(4r) + C2 + Z3 r,  Z1 = (x + mu)^2/x conj(dir), C2 = (x + mu)/(2x), Z3 = dir/(4x)
  //   delta = (x + mu)/(4y) = Dc/(4r),  Dc = (x + mu) conj(dir)
  // as on the REAL contour (four DFMA instead of three complex products); zdir: the direction the constants are for.
  cd Z1 = {0.0, 0.0}, C2 = {0.0, 0.0}, Z3 = {0.0, 0.0}, Dc = {0.0, 0.0}, C1x4 = {0.0, 0.0};
  int zdir = -1;   // -1 not set, 0 dir = 1, 1 dir = geo.d
  // The three terms are of the size |C2| = |x + mu|/|2x| each, and on the ray (y along x) they can cancel to a zeta
  // next to [0,1]: the form is used only where |C2| <= 8, which keeps its absolute error below 1e-15 (for |x| << |mu|
  // the product form below, accurate to an ulp of zeta itself, is taken instead).
  bool affine_ok = false;
  if (NT == 1) {
    const cd xm0 = {x.re + a.term[0].mu_re, x.im + a.term[0].mu_im};
    C2 = cmul(xm0, cscale(xinv, 0.5));
    C1x4 = cscale(cmul(xm0, C2), 2.0);
    affine_ok = fma(C2.re, C2.re, C2.im * C2.im) <= 64.0;
  }
  // tables of the real nodes this point walks: the REAL contour's (policy REAL) or its rung's tail piece
  const double* row = blob + L.off_rung + (long long)geo.row * L.rung_stride;
  const bool real_pol = pol == GF_CONTOUR_REAL;
  const double* ty = real_pol ? blob + L.off_y : row + L.rg_y;
  const double* tq4 = real_pol ? blob + L.off_q4 : row + L.rg_yq4;
  const double2* tpref = reinterpret_cast<const double2*>(real_pol ? blob + L.off_pref : row + L.rg_pref);
  const int tstride = real_pol ? L.n_rad_pad : L.n4p;
  const int tn = real_pol ? a.n_rad : a.n_rad >> 2;
  const int t0 = tail_start(pol, a.n_rad);

  // where the tail series takes over: the first real node with y >= Y0 = 4 (sqrt|x| + sqrt(|x| + |x + mu|))^2
  int i_end;
  {
    const double ax = sqrt(fma(x.re, x.re, x.im * x.im));
    double Y0 = 0.0;
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      const cd az = {x.re + a.term[r].mu_re, x.im + a.term[r].mu_im};
      const double q = sqrt(ax) + sqrt(ax + sqrt(fma(az.re, az.re, az.im * az.im)));
      Y0 = fmax(Y0, kTailFactor * q * q);
    }
    int lo = 0, hi = tn;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (ty[mid] < Y0) lo = mid + 1; else hi = mid;
    }
    i_end = sym ? tn : lo;   // (the symmetric routing's tail needs a second table pair: its real nodes take routes)
  }
  const int g_end = t0 + i_end;
  const int g_stop = __reduce_max_sync(0xffffffffu, g_end);

  RouteCount rc;
  double g_re = 0.0, g_im = 0.0;
  int k_line = -1;           // the straight piece whose end points are in la, ld
  cd la = {0.0, 0.0}, ld = {0.0, 0.0};
  // warp-synchronous node loop (node_term is warp-collective): a lane past its last node repeats it with weight 0
#pragma unroll 1
  for (int g0 = 0; g0 < g_stop; g0 += S) {
    const bool valid = g0 + sub < g_end;
    const int g = valid ? g0 + sub : g_end - 1 + (g_end == 0);
    const NodeAt at = locate(pol, a.n_rad, g);
    // ---- the node: y, 1/(4y), and the prefactor c0 (rule weight) dy/dt y D1(y) without the pole factors
    cd y, q4, base = {0.0, 0.0};
    const bool table = at.type == SEG_TABLE || at.type == SEG_TAIL;
    if (table) {
      y = {ty[at.i], 0.0};
      q4 = {tq4[at.i], 0.0};
    } else if (at.type == SEG_RAY) {
      const double r = row[L.rg_r + at.i], q4r = row[L.rg_q4 + at.i], rw = row[L.rg_w + at.i];
      y = {__dmul_rn(geo.dre, r), __dmul_rn(geo.dim, r)};
      q4 = {geo.dre * q4r, -geo.dim * q4r};
      base = {dir2.re * rw, dir2.im * rw};          // c0 wy y = c0 dir^2 r dr
    } else {
      const double t = srt[at.rule + at.i], w = srw[at.rule + at.i];
      cd wy;
      if (at.type == SEG_LINE) {
        if (at.k != k_line) {
          k_line = at.k;
          la = thread_waypoint(geo, at.k);
          const cd lb = thread_waypoint(geo, at.k + 1);
          ld = {__dadd_rn(lb.re, -la.re), __dadd_rn(lb.im, -la.im)};
        }
        line_node(la, ld, t, w, &y, &wy);
      } else {
        arc_node(geo.R, geo.tau, t, w, &y, &wy);
      }
      base = measure_base(a, geo, at.type, at.k, t, y, wy);
      if (geo.mirror) { y.im = -y.im; wy.im = -wy.im; base.im = -base.im; }
      q4 = cscale(cinv_fast(y), 0.25);
    }
    const bool affine = NT == 1 && affine_ok && (table || at.type == SEG_RAY);
    cd xq = {0.0, 0.0};
    if (affine) {
      const int want = at.type == SEG_RAY;
      if (zdir != want) {   // once per piece
        zdir = want;
        const cd d = want ? cd{geo.dre, geo.dim} : cd{1.0, 0.0}, dc = {d.re, -d.im};
        Z1 = cmul(C1x4, dc);
        Z3 = cscale(cmul(xinv, d), 0.25);
        Dc = cmul(cd{fma(dmu, a.term[0].mu_re, x.re), fma(dmu, a.term[0].mu_im, x.im)}, dc);
      }
    } else {
      xq = cmul(xinv, q4);                           // 1/(4 x y)
    }
    cd ic0 = {0.0, 0.0};
    if (!table) {
      if (a.same_mass) ic0 = cinv_fast(y_plus_mu(y, a.term[0]));
      base = cmul(base, a.same_mass ? ic0 : line_k_complex(a, y));
    }
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      const double mur = a.term[r].mu_re, mui = a.term[r].mu_im;
      cd delta, zeta;
      if (affine) {
        const double q4r = table ? q4.re : row[L.rg_q4 + at.i], rr = table ? y.re : row[L.rg_r + at.i];
        delta = {fma(Dc.re, q4r, d0), Dc.im * q4r};
        zeta = {fma(Z1.re, q4r, fma(Z3.re, rr, C2.re)), fma(Z1.im, q4r, fma(Z3.im, rr, C2.im))};
      } else {
        const cd xm = {x.re + mur, x.im + mui};
        const cd A = {xm.re + y.re, xm.im + y.im};
        delta = cmul(cd{fma(dmu, mur, x.re), fma(dmu, mui, x.im)}, q4);   // eta - 1/4
        delta.re += d0;
        zeta = cmul(csqr(A), xq);
      }
      const cd s = node_term<double, COUNT, BLK>(tb, x, y, delta, zeta, mur, mui, rc, a.term[r].mu_re_lo, a.term[r].mu_im_lo);
      cd pr;
      if (table) {
        const double2 p2 = tpref[r * tstride + at.i];
        pr = {p2.x, p2.y};
      } else {
        const cd ic = a.same_mass ? ic0 : cinv_fast(y_plus_mu(y, a.term[r]));
        // a massive line 2 is its one pole with residue 1
        pr = NT == 1 ? cd{-base.re, -base.im} : cmul(base, cd{-a.term[r].R_re, -a.term[r].R_im});
        pr = cmul(pr, ic);
      }
      if (valid) {   // (four predicated DFMA)
        g_re = fma(pr.re, s.re, fma(-pr.im, s.im, g_re));
        g_im = fma(pr.re, s.im, fma(pr.im, s.re, g_im));
      }
    }
  }
  // the large-y part of the real piece, all nodes from i_end on at once
  if (__any_sync(0xffffffffu, i_end < tn)) {
    const double invy0 = 4.0 * tq4[min(i_end, tn - 1)];
    const double2* Rt = reinterpret_cast<const double2*>(real_pol ? blob + L.off_tail : row + L.rg_tail) +
                        (size_t)i_end * kTailN;
#pragma unroll
    for (int r = 0; r < NT; ++r) {
      const cd az = {x.re + a.term[r].mu_re, x.im + a.term[r].mu_im};
      const cd tl = tail_series(sb + L.off_gam, Rt + (size_t)r * (tn + 1) * kTailN, x, az, invy0);
      if (sub == 0) {
        g_re += tl.re;
        g_im += tl.im;
      }
      if (COUNT) ++rc.tails;
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
  if (COUNT) flush_counters(rc, active, counters);
}

// The nodes the evaluation kernel walks for one x, read from the same tables by the same code (diagnostic:
// tests compare them with the oracle's bit for bit).  One thread per node; wy = (rule weight) x dy/dt.
__global__ void contour_nodes_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                                     const double* __restrict__ blob, double xr, double xi, int* __restrict__ policy,
                                     double2* __restrict__ out_y, double2* __restrict__ out_wy) {
  const double f = a.routing == 1 ? 0.25 : 1.0;   // symmetric routing: the contour of x/4 (exact scaling)
  const Geo geo = build_geo(a, f * xr, f * xi);
  if (blockIdx.x == 0 && threadIdx.x == 0) *policy = geo.pol;
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= a.n_rad) return;
  const double* row = blob + L.off_rung + (long long)geo.row * L.rung_stride;
  const NodeAt at = locate(geo.pol, a.n_rad, g);
  cd y, wy;
  if (at.type == SEG_TABLE) {
    y = {blob[L.off_y + at.i], 0.0};
    wy = {0.5 * a.rad_weights[at.i] * a.Llog_hi * (y.re + a.s0), 0.0};
  } else if (at.type == SEG_TAIL) {
    y = {row[L.rg_y + at.i], 0.0};
    // the row keeps pref, not the weight: recover (rule weight) dy/dt from the map itself
    const dd L2 = dd_log(dd_div(two_sum(a.cutoff2, a.s0), two_sum(geo.R, a.s0)));
    wy = {0.5 * a.rad_weights[a.n_rad + a.n_rad / 2 + at.i] * L2.hi * (y.re + a.s0), 0.0};
  } else if (at.type == SEG_RAY) {
    const double r = row[L.rg_r + at.i];
    y = {__dmul_rn(geo.dre, r), __dmul_rn(geo.dim, r)};
    const double dr = row[L.rg_w + at.i] / (a.c0 * r);
    wy = {geo.dre * dr, geo.dim * dr};
  } else {
    const int lvl2 = a.n_rad + a.n_rad / 2;
    const double t = a.rad_nodes[lvl2 + at.rule + at.i], w = a.rad_weights[lvl2 + at.rule + at.i];
    if (at.type == SEG_LINE) {
      const cd la = thread_waypoint(geo, at.k), lb = thread_waypoint(geo, at.k + 1);
      line_node(la, cd{__dadd_rn(lb.re, -la.re), __dadd_rn(lb.im, -la.im)}, t, w, &y, &wy);
    } else {
      arc_node(geo.R, geo.tau, t, w, &y, &wy);
    }
  }
  if (geo.mirror) { y.im = -y.im; wy.im = -wy.im; }
  out_y[g] = make_double2(y.re, y.im);
  out_wy[g] = make_double2(wy.re, wy.im);
}

template <bool COUNT, int NT, bool BLK, int POL>
int launch_contour_kern(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* counters,
                        cudaStream_t stream) {
  auto kern = eval_contour_kernel<COUNT, NT, BLK, POL>;
  if (plan.smem_bytes > 48 * 1024) {
    int rc = check_cuda(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes),
                        "cudaFuncSetAttribute(max dynamic shared memory)");
    if (rc) return rc;
  }
  kern<<<(unsigned)plan.grid_blocks, plan.block_threads, plan.smem_bytes, stream>>>(a, plan.layout, blob, counters);
  return check_cuda(cudaGetLastError(), "contour kernel launch");
}

// the instantiations for one policy exist for the timed kernels only
template <bool COUNT, int NT, bool BLK>
int launch_contour_t(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* counters,
                     cudaStream_t stream) {
  if constexpr (!COUNT) {
    if (a.contour == GF_CONTOUR_RAY_ARC) return launch_contour_kern<COUNT, NT, BLK, GF_CONTOUR_RAY_ARC>(a, plan, blob, counters, stream);
    if (a.contour == GF_CONTOUR_THREAD) return launch_contour_kern<COUNT, NT, BLK, GF_CONTOUR_THREAD>(a, plan, blob, counters, stream);
  }
  return launch_contour_kern<COUNT, NT, BLK, -1>(a, plan, blob, counters, stream);
}

}  // namespace

int launch_contour(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* d_counters,
                   cudaStream_t stream) {
  const bool blk = plan.layout.n_blk > 0;
  if (a.n_terms == 1) {
    if (d_counters) return blk ? launch_contour_t<true, 1, true>(a, plan, blob, d_counters, stream)
                               : launch_contour_t<true, 1, false>(a, plan, blob, d_counters, stream);
    return blk ? launch_contour_t<false, 1, true>(a, plan, blob, nullptr, stream)
               : launch_contour_t<false, 1, false>(a, plan, blob, nullptr, stream);
  }
  if (d_counters) return blk ? launch_contour_t<true, 2, true>(a, plan, blob, d_counters, stream)
                             : launch_contour_t<true, 2, false>(a, plan, blob, d_counters, stream);
  return blk ? launch_contour_t<false, 2, true>(a, plan, blob, nullptr, stream)
             : launch_contour_t<false, 2, false>(a, plan, blob, nullptr, stream);
}

int launch_prepare_rungs(const EvalArgs& a, const LaunchPlan& plan, double* blob, cudaStream_t stream) {
  prep_rungs_kernel<<<plan.layout.n_rungs, 256, 0, stream>>>(a, plan.layout, blob);
  return check_cuda(cudaGetLastError(), "rung preparation kernel launch");
}

int launch_contour_nodes(const EvalArgs& a, const LaunchPlan& plan, const double* blob, double x_re, double x_im,
                         int* d_policy, double2* d_y, double2* d_wy, cudaStream_t stream) {
  contour_nodes_kernel<<<(a.n_rad + 127) / 128, 128, 0, stream>>>(a, plan.layout, blob, x_re, x_im, d_policy, d_y,
                                                                 d_wy);
  return check_cuda(cudaGetLastError(), "contour_nodes launch");
}

}  // namespace gf
