// gf_contour.cu -- Step 3 inside Kernel 2: evaluation on radial contours
// that depend on the grid point.  The paper's Kernel 2 picks one of four hand-made contours per thread
// with an IF-THEN-ELSE on the region of x; here each thread builds its contour from x by one of the
// policies of DESIGN.md "Contour policies" and walks its n_rad nodes:
//
//   REAL     [0, Lambda^2], shifted-log map (nodes prepared once per launch, as in gf_eval.cu);
//   RAY_ARC  ray y = r e^{i arg x}, r in [0,R] shifted-log (n_rad/2 nodes), arc R e^{i theta} back to the real
//            axis (n_rad/4), real tail [R, Lambda^2] shifted-log (n_rad/4);  R = 1.5 (sqrt|x| + sqrt(|x|+sc))^2
//            with sc the size of line 2's singular structure, capped at Lambda^2/2
//            (generalises the paper's region-2/5 contour);
//   THREAD   equal real masses, next to the negative axis below -4 m^2: five straight pieces through
//            the waypoints W0..W5 that pass the pole of line 1 and thread the opening of the cut at
//            |x + m^2| e^{i arg x}, an arc from 3 pi/4 to 0 and the real tail (n_rad/8 nodes each, n_rad/4
//            on the tail); mirrored for Im x < 0 (the analogue of the region-3/4 polylines);
//   AUTO     per point: RAY_ARC outside the wedge {Re x < -sc, |Im x| n_ang sc < 5 |x|^2}, inside it THREAD
//            where it applies and Re x <= -4.1 sc, else REAL.
//
// The geometry is written with the _rn intrinsics in the order DESIGN.md states it, so that region tests
// and waypoints do not depend on contraction; sqrt is correctly rounded; atan2, sincos, hypot, log, expm1
// are the device's (within 1-2 ulp; the sums are insensitive to that).
// Per node the angular sum is the same folded sum S(eta, zeta) as on the REAL contour (gf_routes.cuh):
// with complex y, eta = (x + y + mu)/(4y) and zeta = (x + y + mu)^2/(4xy) are simply complex.
#include "gf_routes.cuh"

namespace gf {
namespace {

enum { SEG_TABLE = 0, SEG_LOG = 1, SEG_LINE = 2, SEG_ARC = 3 };
constexpr int kMaxSeg = 7;

// One piece of a contour.  off/n: its Gauss-Legendre rule inside the pyramid; start: index of its first
// node among the point's n_rad nodes.  p[]: LOG  a, L_hi, L_lo, dir.re, dir.im, a + s0;
// LINE a.re, a.im, (b-a).re, (b-a).im;  ARC  R, theta0, theta1 - theta0.
struct Seg {
  int type, off, n, start;
  double p[6];
};

// ln(v) for a double-double v >= 1: libm seed, one Newton step on exp in double-double
__device__ dd dd_log(dd v) {
  const double l0 = log(v.hi);
  const dd e = dd_add_d(dd_expm1(dd{l0, 0.0}), 1.0);
  const dd c = dd_div(dd_add(v, dd_neg(e)), e);
  return quick_two_sum(l0, c.hi);
}

__device__ void seg_log(Seg& s, double a, double b, double s0, double dre, double dim, int off, int n) {
  // L = ln((b + s0)/(a + s0)) (readings G3/G4)
  const dd L = dd_log(dd_div(two_sum(b, s0), two_sum(a, s0)));
  s.type = SEG_LOG; s.off = off; s.n = n;
  s.p[0] = a; s.p[1] = L.hi; s.p[2] = L.lo; s.p[3] = dre; s.p[4] = dim; s.p[5] = __dadd_rn(a, s0);
}
__device__ void seg_line(Seg& s, cd a, cd b, int off, int n) {
  s.type = SEG_LINE; s.off = off; s.n = n;
  s.p[0] = a.re; s.p[1] = a.im; s.p[2] = __dadd_rn(b.re, -a.re); s.p[3] = __dadd_rn(b.im, -a.im);
  s.p[4] = s.p[5] = 0.0;
}
__device__ void seg_arc(Seg& s, double R, double th0, double th1, int off, int n) {
  s.type = SEG_ARC; s.off = off; s.n = n;
  s.p[0] = R; s.p[1] = th0; s.p[2] = __dadd_rn(th1, -th0);
  s.p[3] = s.p[4] = s.p[5] = 0.0;
}

// AUTO's per-point choice; half-open tests exactly as DESIGN.md writes them
__device__ int auto_policy(const EvalArgs& a, double xr, double xi) {
  const double sc = a.line2_scale;
  const double ax2 = __fma_rn(xr, xr, __dmul_rn(xi, xi));
  const bool wedge = (xr < -sc) && (__dmul_rn(fabs(xi), __dmul_rn((double)a.n_ang, sc)) < __dmul_rn(5.0, ax2));
  if (!wedge) return GF_CONTOUR_RAY_ARC;
  if (a.thread_ok && xr <= __dmul_rn(-4.1, sc)) return GF_CONTOUR_THREAD;
  return GF_CONTOUR_REAL;
}

// Build the segments of the point's contour; returns their number.  *mirror: conjugate every node.
__device__ int build_contour(const EvalArgs& a, int pol, double xr, double xi, Seg* seg, bool* mirror) {
  const int n = a.n_rad, o1 = n, o2 = n + n / 2, o3 = n + n / 2 + n / 4;
  *mirror = false;
  int ns = 0;
  if (pol == GF_CONTOUR_REAL) {
    seg[0].type = SEG_TABLE; seg[0].off = 0; seg[0].n = n;
    ns = 1;
  } else if (pol == GF_CONTOUR_RAY_ARC) {
    const double ax = __dsqrt_rn(__fma_rn(xr, xr, __dmul_rn(xi, xi)));
    const double phi = atan2(xi, xr);
    const double q = __dadd_rn(__dsqrt_rn(ax), __dsqrt_rn(__dadd_rn(ax, a.line2_scale)));
    const double R = fmin(__dmul_rn(__dmul_rn(1.5, q), q), 0.5 * a.cutoff2);
    double sn, cs;
    sincos(phi, &sn, &cs);
    seg_log(seg[0], 0.0, R, a.s0, cs, sn, o1, n / 2);
    seg_arc(seg[1], R, phi, 0.0, o2, n / 4);
    seg_log(seg[2], R, a.cutoff2, a.s0, 1.0, 0.0, o2, n / 4);
    ns = 3;
  } else {
    *mirror = xi < 0.0;
    const double yi = fabs(xi);
    const double m2 = a.term[0].mu_re, m = __dsqrt_rn(m2);
    const double s = __dsqrt_rn(__fma_rn(xr, xr, __dmul_rn(yi, yi)));
    const double phi = atan2(yi, xr);
    const double rs = __dsqrt_rn(s);
    const double dm = __dadd_rn(rs, -m), dp = __dadd_rn(rs, m);
    const double Aa = __dmul_rn(dm, dm), Bb = __dmul_rn(dp, dp);
    const double r0 = hypot(__dadd_rn(xr, m2), yi);
    double sn, cs;
    sincos(phi, &sn, &cs);
    cd W[6];
    W[0] = {0.0, 0.0};
    W[1] = {-m2, __dmul_rn(0.5, __dadd_rn(Aa, -m2))};
    const double h2 = __dmul_rn(0.5, __dadd_rn(Aa, m2));
    W[2] = {__dmul_rn(h2, cs), __dmul_rn(h2, sn)};
    W[3] = {__dmul_rn(-0.5, __dadd_rn(Aa, r0)), __dmul_rn(-0.5, __dadd_rn(r0, -Aa))};
    W[4] = {__dmul_rn(r0, cs), __dmul_rn(r0, sn)};
    const double R = fmin(__dmul_rn(1.5, Bb), 0.5 * a.cutoff2);
    W[5] = {__dmul_rn(R, a.cos_th5), __dmul_rn(R, a.sin_th5)};
    for (int k = 0; k < 5; ++k) seg_line(seg[k], W[k], W[k + 1], o3, n / 8);
    seg_arc(seg[5], R, a.th5, 0.0, o3, n / 8);
    seg_log(seg[6], R, a.cutoff2, a.s0, 1.0, 0.0, o2, n / 4);
    ns = 7;
  }
  int start = 0;
  for (int k = 0; k < ns; ++k) {
    seg[k].start = start;
    start += seg[k].n;
  }
  return ns;
}

// D1(y) for complex y
__device__ __forceinline__ cd line_k_complex(const gf_propagator& p, cd y) {
  if (p.kind == GF_PROP_MASSIVE) return cinv_fast(cd{y.re + p.m2_re, y.im + p.m2_im});
  const cd ya = {y.re + p.a, y.im};
  cd den = cmul(y, ya);
  den.re += p.b;
  return cmul(cd{y.re + p.M2, y.im}, cinv_fast(den));
}

// ---------------------------------------------------------------------------------------------
// Evaluation on point-dependent contours.  Same staging, lane split, routes, reductions and store as
// eval_real_kernel; counters as there.
// ---------------------------------------------------------------------------------------------
template <bool COUNT>
__global__ void __launch_bounds__(kBlockThreads, 2)
    eval_contour_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                        const double* __restrict__ blob, unsigned long long* __restrict__ counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
  double* sb = reinterpret_cast<double*>(smem_raw + 16);
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) bulk_load(sb, blob, (uint32_t)(L.n_doubles * sizeof(double)), bar);
  mbar_wait(bar, 0);

  const Tabs<double> tb = make_tabs<double>(sb, L, a.n_pairs);
  const double* sy = sb + L.off_y;
  const double* sq4 = sb + L.off_q4;
  const double2* spref = reinterpret_cast<const double2*>(sb + L.off_pref);
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
  const cd xinv = cinv(x);

  Seg seg[kMaxSeg];
  bool mirror;
  const int pol = a.contour == GF_CONTOUR_AUTO ? auto_policy(a, x.re, x.im) : a.contour;
  const int n_seg = build_contour(a, pol, x.re, x.im, seg, &mirror);

  RouteCount rc;
  double g_re = 0.0, g_im = 0.0;
  int ks = 0;
  // warp-synchronous node loop (node_term is warp-collective): a lane past the last node repeats it with weight 0
#pragma unroll 1
  for (int g0 = 0; g0 < a.n_rad; g0 += S) {
    const bool valid = g0 + sub < a.n_rad;
    const int g = valid ? g0 + sub : a.n_rad - 1;
    while (ks + 1 < n_seg && g >= seg[ks].start + seg[ks].n) ++ks;
    const Seg& sg = seg[ks];
    const int i = g - sg.start;
    // ---- the node: y and (rule weight) x dy/dt
    cd y, wy = {0.0, 0.0}, q4;
    const bool table = sg.type == SEG_TABLE;
    if (table) {
      y = {sy[i], 0.0};
      q4 = {sq4[i], 0.0};
    } else {
      const double t = srt[sg.off + i], w = srw[sg.off + i];
      const double u = __dmul_rn(0.5, __dadd_rn(t, 1.0));
      if (sg.type == SEG_LOG) {
        // r = a + (a + s0) expm1(u L), dr = (w/2) L (r + s0); L = L_hi + L_lo
        const dd uL = dd_mul_d(dd{sg.p[1], sg.p[2]}, u);
        const double e1 = expm1(uL.hi);
        const double E = fma(uL.lo, e1 + 1.0, e1);
        const double r = fma(sg.p[5], E, sg.p[0]);
        const double dr = 0.5 * w * sg.p[1] * (r + a.s0);
        y = {sg.p[3] * r, sg.p[4] * r};
        wy = {sg.p[3] * dr, sg.p[4] * dr};
      } else if (sg.type == SEG_LINE) {
        const double hw = __dmul_rn(0.5, w);
        y = {__dadd_rn(sg.p[0], __dmul_rn(sg.p[2], u)), __dadd_rn(sg.p[1], __dmul_rn(sg.p[3], u))};
        wy = {__dmul_rn(sg.p[2], hw), __dmul_rn(sg.p[3], hw)};
      } else {
        const double th = __dadd_rn(sg.p[1], __dmul_rn(sg.p[2], u));
        double sn, cs;
        sincos(th, &sn, &cs);
        y = {__dmul_rn(sg.p[0], cs), __dmul_rn(sg.p[0], sn)};
        const double f = __dmul_rn(__dmul_rn(sg.p[2], 0.5), w);
        wy = {__dmul_rn(-y.im, f), __dmul_rn(y.re, f)};  // i y dtheta
      }
      if (mirror) { y.im = -y.im; wy.im = -wy.im; }
      q4 = cscale(cinv_fast(y), 0.25);
    }
    cd base = {0.0, 0.0};
    if (!table) base = cscale(cmul(cmul(wy, y), line_k_complex(a.line_k, y)), a.c0);
    const cd xq = cmul(xinv, q4);                    // 1/(4 x y)
#pragma unroll 1
    for (int r = 0; r < a.n_terms; ++r) {
      const double mur = a.term[r].mu_re, mui = a.term[r].mu_im;
      const cd xm = {x.re + mur, x.im + mui};
      const cd A = {xm.re + y.re, xm.im + y.im};
      const cd delta = cmul(xm, q4);                 // eta - 1/4
      const cd zeta = cmul(csqr(A), xq);
      const cd s = node_term<double, COUNT>(tb, x, y, delta, zeta, mur, mui, rc);
      cd pr;
      if (table) {
        const double2 p2 = spref[r * L.n_rad_pad + i];
        pr = {p2.x, p2.y};
      } else {
        const cd ic = cinv_fast(cd{y.re + mur, y.im + mui});
        pr = cmul(cmul(base, cd{-a.term[r].R_re, -a.term[r].R_im}), ic);
      }
      if (!valid) pr = {0.0, 0.0};
      g_re = fma(pr.re, s.re, fma(-pr.im, s.im, g_re));
      g_im = fma(pr.re, s.im, fma(pr.im, s.re, g_im));
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

template <bool COUNT>
int launch_contour_t(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* counters,
                     cudaStream_t stream) {
  auto kern = eval_contour_kernel<COUNT>;
  if (plan.smem_bytes > 48 * 1024) {
    int rc = check_cuda(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes),
                        "cudaFuncSetAttribute(max dynamic shared memory)");
    if (rc) return rc;
  }
  kern<<<(unsigned)plan.grid_blocks, plan.block_threads, plan.smem_bytes, stream>>>(a, plan.layout, blob, counters);
  return check_cuda(cudaGetLastError(), "contour kernel launch");
}

}  // namespace

int launch_contour(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* d_counters,
                   cudaStream_t stream) {
  return d_counters ? launch_contour_t<true>(a, plan, blob, d_counters, stream)
                    : launch_contour_t<false>(a, plan, blob, nullptr, stream);
}

}  // namespace gf
