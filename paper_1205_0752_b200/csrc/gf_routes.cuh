// gf_routes.cuh -- device code shared by the two evaluation kernels (gf_eval.cu: REAL contour, nodes
// prepared once per launch; gf_contour.cu: contours that depend on the grid point): the routes that
// evaluate the folded angular sum S = sum_j w_j (eta - t_j)/(zeta - t_j) of one (point, radial node, pole),
// the 1-D TMA staging of the prepared tables, and the folding of the angular rule.  See gf_eval.cu's
// header for the algebra.  Everything here is internal to the translation unit that includes it.
#pragma once
#include <cfloat>
#include <cmath>
#include <cstdint>

#include "gf_dd.cuh"
#include "gf_internal.h"

namespace gf {
namespace {

constexpr int kKmc = 256;             // series coefficients staged per table (even)
// fixed places of the series tables in the staged block, in doubles (make_blob_layout)
constexpr int kOffMom = 2, kOffCheb = kOffMom + 2 * kKmc, kOffKreq = kOffCheb + 2 * kKmc,
              kOffSf = kOffKreq + kKreqBins / 2 + 4;
constexpr int kMomTerms = 32;         // genuine coefficients of the centred-moment series (zero beyond)
#ifndef GF_SERIES_BITS
#define GF_SERIES_BITS 46
#endif
constexpr float kSeriesBits = GF_SERIES_BITS;    // series are cut where the dropped terms are below 2^-50 of the leading one
// extra bits of error the FP32 phase of a series may cost over the truncation budget 2^-kSeriesBits (0: none)
#ifndef GF_FP32_SLACK_BITS
#define GF_FP32_SLACK_BITS 0
#endif
constexpr float kFp32Slack = GF_FP32_SLACK_BITS;
// the centred-moment series (far nodes, at most 20 terms) is cut four bits later than the Chebyshev series: where
// |x| >> the masses on a deformed contour its leading terms cancel in S and the truncation shows (measured: 1.2e-11
// at 46 bits on a ray next to the negative axis, 3e-12 at 50)
#ifndef GF_MOMENT_BITS
#define GF_MOMENT_BITS (GF_SERIES_BITS + 4)
#endif
constexpr float kMomentBits = GF_MOMENT_BITS;
#ifndef GF_GOERTZEL_UNROLL
#define GF_GOERTZEL_UNROLL 2
#endif
constexpr int kGoertzelUnroll = GF_GOERTZEL_UNROLL;   // trips of the series loop (2 terms each) unrolled
#ifndef GF_NEAR_UNROLL
#define GF_NEAR_UNROLL 1
#endif
constexpr int kNearUnroll = GF_NEAR_UNROLL;           // trips of the plain direct loop (4 pairs each) unrolled
// MOMENT route when max(|Re zeta|, |Im zeta|) >= 4.5 (then |zeta - 1/2| >= 4), compared on the high words
// (measured again with the cheaper CHEB set-up: from 6 or 8 the cfg3 kernel is 0.5 / 0.75 % faster, but CHEB's s = w - 2 root
// loses 2 |w|^2 of its digits and the worst case of the random deformed-contour problems goes 3.2e-12 -> 5.8e-12: not taken)
#ifndef GF_MOMENT_HIWORD
#define GF_MOMENT_HIWORD 0x40120000
#endif
constexpr double kTau64 = 0x1p-8;     // EXACT route inside this distance of [0,1] (FP64)
constexpr double kTau32 = 0x1p-4;     // the FP32 variant's NEAR loop is only good further away
// Kreq table: bins of log2(rho) from kEllLo in steps of kEllStep (the lower edge of a bin decides, so K is safe)
constexpr float kEllLo = 0.235f, kEllStep = 0.02f;

// Blocks of the folded rule for the direct routes (angular_blocked): kBlkPairs consecutive pairs each; a block that is
// far from zeta (ellipse parameter of ITS interval rho_b^2 >= kBlkRho2Min) is summed by its own Chebyshev series of at
// most kBlkTerms terms instead of pair by pair.  K_b = 112/log2(rho_b^2) + 1: dropped terms below 2^-56 rho-scaled.
#ifndef GF_BLK_TERMS
#define GF_BLK_TERMS 64
#endif
constexpr int kBlkPairs = 32, kBlkTerms = GF_BLK_TERMS;
#ifndef GF_BLK_MIN_PAIRS
#define GF_BLK_MIN_PAIRS 128           // REAL contour
#endif
#ifndef GF_BLK_MIN_PAIRS_CONTOUR
#define GF_BLK_MIN_PAIRS_CONTOUR 192   // deformed contours (measured: 128 pairs lose 4 % there, 256 gain 15 %)
#endif
#ifndef GF_BLK_CHEB_CAP
#define GF_BLK_CHEB_CAP 256
#endif
constexpr int kBlkChebCap = GF_BLK_CHEB_CAP;   // with a split rule, Chebyshev series longer than this go to the direct route
constexpr int kBlkMinPairs = GF_BLK_MIN_PAIRS, kBlkMinPairsContour = GF_BLK_MIN_PAIRS_CONTOUR;   // smaller rules are not split
constexpr float kBlkRho2Min = GF_BLK_TERMS == 32 ? 12.3f : GF_BLK_TERMS == 48 ? 5.3f : 3.5f;   // 2^(112/(kBlkTerms - 1))
static_assert(GF_BLK_TERMS == 32 || GF_BLK_TERMS == 48 || GF_BLK_TERMS == 64, "block series of 32, 48 or 64 terms");
// |w'|^2 beyond which a block is far: the squared semi-major axis of the ellipse rho^2 = kBlkRho2Min, (R + 2 + 1/R)/4
constexpr double kBlkFarW2 = (kBlkRho2Min + 2.0 + 1.0 / kBlkRho2Min) / 4.0;

enum { ROUTE_MOMENT = 0, ROUTE_CHEB = 1, ROUTE_NEAR = 2, ROUTE_EXACT = 3 };

struct cd {
  double re, im;
};
__device__ __forceinline__ cd cmul(cd a, cd b) {
  return {fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re)};
}
__device__ __forceinline__ cd csqr(cd a) { return {fma(a.re, a.re, -(a.im * a.im)), (a.re + a.re) * a.im}; }
__device__ __forceinline__ cd cscale(cd a, double s) { return {a.re * s, a.im * s}; }
__device__ __forceinline__ cd cadd(cd a, cd b) { return {a.re + b.re, a.im + b.im}; }
__device__ __forceinline__ cd cinv(cd a) {
  // set-up code only (once per point / node): plain division, scaled against overflow
  const double m = fmax(fabs(a.re), fabs(a.im));
  const double ar = a.re / m, ai = a.im / m;
  const double d = 1.0 / (m * fma(ar, ar, ai * ai));
  return {ar * d, -ai * d};
}

__device__ __forceinline__ double rcp_seed(double s) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(s));  // MUFU.RCP64H
  return r;
}
__device__ __forceinline__ float rcp_seed(float s) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s));  // MUFU.RCP
  return r;
}
__device__ __forceinline__ double rsqrt_seed(double s) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(s));  // MUFU.RSQ64H
  return r;
}
// FP32 helpers for the term counts (flush-to-zero, approximate: one MUFU each)
__device__ __forceinline__ float lg2_ftz(float s) {
  float r;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s));
  return r;
}
__device__ __forceinline__ float rcp_ftz(float s) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s));
  return r;
}
// 1/s and 1/sqrt(s) for normal s well inside the exponent range: seed + one cubic correction, no slow path
__device__ __forceinline__ double rcp_fast(double s) {
  const double r0 = rcp_seed(s);
  const double e = fma(-s, r0, 1.0);
  return fma(r0, fma(e, e, e), r0);
}
__device__ __forceinline__ double rsqrt_fast(double s) {
  const double r0 = rsqrt_seed(s);
  const double e = fma(-s * r0, r0, 1.0);                // 1 - s r0^2
  return fma(r0, e * fma(0.375, e, 0.5), r0);            // r0 (1 + e/2 + 3 e^2/8)
}

// 1/a per radial node on the deformed contours: |a|^2 stays far inside the exponent range there
// (|y| <= Lambda^2 <= 1e60, and a node or y + mu exactly 0 gives inf/NaN as the header says)
__device__ __forceinline__ cd cinv_fast(cd a) {
  const double in = rcp_fast(fma(a.re, a.re, a.im * a.im));
  return {a.re * in, -a.im * in};
}

// ---- 1-D TMA: one bulk copy global -> shared, completion on an mbarrier ------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase) {
  uint32_t done = 0;
  for (long long spin = 0; !done; ++spin) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(phase)
        : "memory");
    if (spin > (1LL << 26)) __trap();  // a copy of a few KB that has not landed after seconds: fail, do not hang
  }
}

// bad input found by a kernel: leave a code in the mapped host word (gf_internal.h), read by the next API call
__device__ __forceinline__ void report_status(int* status, int code) {
  if (status) {
    atomicOr_system(status, code);
    __threadfence_system();
  }
}
// the header of a prepared workspace: [0] != 0: bad tables (every output NaN), [1] = EvalArgs::ws_tag
__device__ __forceinline__ bool workspace_matches(const EvalArgs& a, const double* __restrict__ blob) {
  return __ldg(blob + 1) == a.ws_tag;
}
// radial tables (every level of the pyramid a deformed contour uses): strictly inside (-1,1) and ascending
__device__ void check_radial_tables(const EvalArgs& a, int* bad) {
  const int levels = a.contour == GF_CONTOUR_REAL ? 1 : 4;
  int off = 0, n = a.n_rad;
  for (int l = 0; l < levels; ++l) {
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const double t = a.rad_nodes[off + i];
      if (!(t > -1.0 && t < 1.0) || (i > 0 && !(t > a.rad_nodes[off + i - 1]))) atomicOr(bad, kStatusRadialNodes);
    }
    off += n;
    n >>= 1;
  }
}

template <typename T>
struct Vec2;
template <>
struct Vec2<double> { typedef double2 type; };
template <>
struct Vec2<float> { typedef float2 type; };

// Shared-memory views of the staged tables
template <typename T>
struct Tabs {
  const double *st, *stlo, *sw;                   // folded angular rule
  const T *stT, *swT;                             // the same in the loop's type
  const typename Vec2<T>::type *mom, *cheb;       // series coefficients (P_k, N_k), kmc entries each
  uint32_t a_kreq;                                // shared-window address of kreq
  uint32_t a_mom, a_momf;                         // shared-window addresses of the double2 / float2 series tables
                                                  // (moment table first, the Chebyshev table kmc entries further)
  const int* kreq;                                // Chebyshev terms needed per bin of log2(rho): K | K1 << 16
  double mu0;                                     // sum of the folded weights
  int n_pairs, kmc;
  int kcap;                                       // longest Chebyshev series taken (kmc, or less where the split rule's
                                                  // direct route is cheaper than a long series)
  int n_blk;                                      // leaf blocks of the folded rule (0: not split)
  int n_lev;                                      // levels of the tree of blocks
  unsigned long long lev_pack;                    // level l's blocks start at table index (lev_pack >> 16 l) & 0xffff
  const double2* blk;                             // per block: centre c_b and 1/h_b of its interval [c - h, c + h]
  const double* blkM;                             // per block: M_k = sum'_{j in b} w_j T_k((t_j - c)/h), kBlkTerms each
};
template <typename T>
__device__ __forceinline__ Tabs<T> make_tabs(const double* sb, const BlobLayout& L, int n_pairs) {
  Tabs<T> tb;
  tb.st = sb + L.off_t;
  tb.stlo = sb + L.off_tlo;
  tb.sw = sb + L.off_w;
  typedef typename Vec2<T>::type V2;
  if (sizeof(T) == 8) {
    tb.stT = reinterpret_cast<const T*>(tb.st);
    tb.swT = reinterpret_cast<const T*>(tb.sw);
    tb.mom = reinterpret_cast<const V2*>(sb + L.off_mom);
    tb.cheb = reinterpret_cast<const V2*>(sb + L.off_cheb);
  } else {
    tb.stT = reinterpret_cast<const T*>(sb + L.off_f32);
    tb.swT = tb.stT + L.npad;
    tb.mom = reinterpret_cast<const V2*>(sb + L.off_sf);
    tb.cheb = tb.mom + L.kmc;
  }
  const uint32_t base = smem_u32(sb);   // one base, immediates from the fixed layout
  tb.a_kreq = base + 8u * kOffKreq;
  tb.a_mom = base + 8u * kOffMom;
  tb.a_momf = base + 8u * kOffSf;
  tb.kreq = reinterpret_cast<const int*>(sb + kOffKreq);
  tb.mu0 = sb[kOffMom];  // a_0 of the moment series = sum of the folded weights
  tb.n_pairs = n_pairs;
  tb.kmc = L.kmc;
  tb.n_blk = L.n_blk;
  tb.n_lev = L.n_lev;
  tb.lev_pack = 0;
#pragma unroll
  for (int l = 0; l < kBlkMaxLev; ++l) tb.lev_pack |= (unsigned long long)(L.lev_off[l] & 0xffff) << (16 * l);
  tb.kcap = (sizeof(T) == 8 && L.n_blk > 0) ? min(L.kmc, kBlkChebCap) : L.kmc;
  tb.blk = reinterpret_cast<const double2*>(sb + (L.n_blk ? L.off_blk : 0));
  tb.blkM = sb + (L.n_blk ? L.off_blkM : 0);
  return tb;
}

// Work counters of one thread (COUNT launches only)
struct RouteCount {
  unsigned long long near_pairs = 0, series_exec = 0, exact_pairs = 0, n_near = 0, n_moment = 0, n_exact = 0,
                     n_cheb = 0, series_used = 0, tails = 0, series_exec32 = 0, blk_series = 0, blk_terms = 0,
                     blk_leaves = 0;
};
constexpr int kNumCounters = 13;

// ---- NEAR: one folded angular pair: q = w/|zeta - t|^2 and the two sums ---------------------------
__device__ __forceinline__ void pair_step(double zr, double zi2, double t, double w, double& u0, double& u1) {
  const double a = zr - t;              // DADD
  const double s = fma(a, a, zi2);      // DFMA  |zeta - t|^2
  const double r0 = rcp_seed(s);        // MUFU.RCP64H
  const double e = fma(-s, r0, 1.0);    // DFMA
  const double p = fma(e, e, e);        // DFMA  e + e^2
  const double v = r0 * w;              // DMUL
  const double q = fma(v, p, v);        // DFMA  w/s (1 - e^3)
  u0 += q;                              // DADD
  u1 = fma(q, t, u1);                   // DFMA
}
__device__ __forceinline__ void pair_step(float zr, float zi2, float t, float w, float& u0, float& u1) {
  const float a = zr - t;
  const float s = fmaf(a, a, zi2);
  const float q = w * rcp_seed(s);
  u0 += q;
  u1 = fmaf(q, t, u1);
}

// S = mu0 - (zeta - eta)(conj(zeta) U0 - U1).  Two independent accumulator sets (even / odd pairs).
template <typename T>
__device__ __forceinline__ cd angular_near(cd eta, cd zeta, double mu0, const T* __restrict__ st,
                                           const T* __restrict__ sw, int n_pairs) {
  typedef typename Vec2<T>::type V2;
  const T zr = (T)zeta.re;
  const T zi2 = (T)(zeta.im * zeta.im);
  T a0 = 0, a1 = 0, b0 = 0, b1 = 0;
  int j = 0;
#pragma unroll(kNearUnroll)
  for (; j + 4 <= n_pairs; j += 4) {
    const V2 t01 = *reinterpret_cast<const V2*>(st + j), t23 = *reinterpret_cast<const V2*>(st + j + 2);
    const V2 w01 = *reinterpret_cast<const V2*>(sw + j), w23 = *reinterpret_cast<const V2*>(sw + j + 2);
    pair_step(zr, zi2, t01.x, w01.x, a0, a1);
    pair_step(zr, zi2, t01.y, w01.y, b0, b1);
    pair_step(zr, zi2, t23.x, w23.x, a0, a1);
    pair_step(zr, zi2, t23.y, w23.y, b0, b1);
  }
  for (; j < n_pairs; ++j) pair_step(zr, zi2, st[j], sw[j], a0, a1);
  const double u0 = (double)a0 + (double)b0, u1 = (double)a1 + (double)b1;
  const double cr = fma(zeta.re, u0, -u1), ci = -zeta.im * u0;  // conj(zeta) U0 - U1
  const double dr = zeta.re - eta.re, di = zeta.im - eta.im;
  cd s;
  s.re = mu0 - fma(dr, cr, -(di * ci));
  s.im = -fma(dr, ci, di * cr);
  return s;
}

// ---- series routes: P(s) = sum_k a_k s^k and N(s) = sum_k b_k s^k, real coefficients (a_k, b_k) =
// tab[k], complex s, by the second-order (Goertzel) recurrence c_k = coef_k + r c_{k+1} - |s|^2 c_{k+2},
// r = 2 Re s, run from k = Kw-1 down to 0 (Kw even): P(s) = c_0 - c_1 conj(s).  On return p1 = c_0,
// p2 = c_1 (and n1, n2 for N).  Two real DFMA per coefficient instead of a complex multiply-add.
// Coefficients k_hi-1 down to k_lo (both multiples of 4, k_hi >= k_lo) on top of the incoming state: on entry
// p1 = c_{k_hi}, p2 = c_{k_hi+1} (zero to start a series), on return p1 = c_{k_lo}, p2 = c_{k_lo+1}.  Four terms per
// trip, no remainder.  The tables are addressed by their 32-bit shared-window addresses (one register, no
// generic-to-shared conversion per node).  With GF_PREFETCH64 the coefficients of the next trip are loaded while the
// current four terms are used (the last trip then reads the four entries below its range, which exist in the staged
// block and are not used): 16 more live registers for one load latency less per trip.
#ifndef GF_PREFETCH64
#define GF_PREFETCH64 0
#endif
__device__ __forceinline__ double2 lds_d2(uint32_t a) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ double lds_d(uint32_t a) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ float4 lds_f4(uint32_t a) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
#ifndef GF_GOERTZEL_ORDER
#define GF_GOERTZEL_ORDER 1
#endif
__device__ __forceinline__ void goertzel4(double r, double ns, double2 c3, double2 c2, double2 c1, double2 c0, double& p1,
                                          double& p2, double& n1, double& n2) {
#if GF_GOERTZEL_ORDER
  // the four products with -|s|^2 of two terms first, then the four with r: runs of one loop-invariant multiplier
  // (served by the operand-reuse cache) leave two register-file operands per DFMA, which issues every 2 cycles
  // instead of 3.  Same operations, same values.
  double t1 = fma(ns, p2, c3.x), u1 = fma(ns, n2, c3.y), t2 = fma(ns, p1, c2.x), u2 = fma(ns, n1, c2.y);
  p2 = fma(r, p1, t1); n2 = fma(r, n1, u1); p1 = fma(r, p2, t2); n1 = fma(r, n2, u2);
  t1 = fma(ns, p2, c1.x); u1 = fma(ns, n2, c1.y); t2 = fma(ns, p1, c0.x); u2 = fma(ns, n1, c0.y);
  p2 = fma(r, p1, t1); n2 = fma(r, n1, u1); p1 = fma(r, p2, t2); n1 = fma(r, n2, u2);
#else
  p2 = fma(r, p1, fma(ns, p2, c3.x));
  n2 = fma(r, n1, fma(ns, n2, c3.y));
  p1 = fma(r, p2, fma(ns, p1, c2.x));
  n1 = fma(r, n2, fma(ns, n1, c2.y));
  p2 = fma(r, p1, fma(ns, p2, c1.x));
  n2 = fma(r, n1, fma(ns, n2, c1.y));
  p1 = fma(r, p2, fma(ns, p1, c0.x));
  n1 = fma(r, n2, fma(ns, n1, c0.y));
#endif
}
// tab: shared address of the double2 table's entry 0
__device__ __forceinline__ void goertzel_range(uint32_t tab, int k_hi, int k_lo, double r, double ns, double& p1,
                                               double& p2, double& n1, double& n2) {
  uint32_t c = tab + 16u * (uint32_t)k_hi;
#if GF_PREFETCH64
  double2 c3 = lds_d2(c - 16), c2 = lds_d2(c - 32), c1 = lds_d2(c - 48), c0 = lds_d2(c - 64);
#pragma unroll(kGoertzelUnroll)
  for (int k = k_hi; k > k_lo; k -= 4) {
    c -= 64;
    const double2 m3 = lds_d2(c - 16), m2 = lds_d2(c - 32), m1 = lds_d2(c - 48), m0 = lds_d2(c - 64);
    goertzel4(r, ns, c3, c2, c1, c0, p1, p2, n1, n2);
    c3 = m3; c2 = m2; c1 = m1; c0 = m0;
  }
#else
#pragma unroll 1
  for (int k = k_hi; k > k_lo; k -= 4) {
    const double2 c3 = lds_d2(c - 16), c2 = lds_d2(c - 32), c1 = lds_d2(c - 48), c0 = lds_d2(c - 64);
    c -= 64;
    goertzel4(r, ns, c3, c2, c1, c0, p1, p2, n1, n2);
  }
#endif
}

// The same recurrence in FP32 for both polynomials at once with the packed fused multiply-add of sm_100
// (fma.rn.f32x2, SASS FFMA2): s1 = (p1, n1), s2 = (p2, n2); a coefficient pair (P_k, N_k) is one 64-bit operand.
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
  unsigned long long ua, ub, uc, ud;
  asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
  asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
  asm("mov.b64 %0, {%1, %2};" : "=l"(uc) : "f"(c.x), "f"(c.y));
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
  float2 d;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(ud));
  return d;
}
// tab: shared address of the float2 table's entry 0; the coefficients of the next trip are loaded one trip ahead
__device__ __forceinline__ void goertzel_range_f32x2(uint32_t tab, int k_hi, int k_lo, float r, float ns, float2& s1,
                                                     float2& s2) {
  const float2 rr = {r, r}, nn = {ns, ns};
  uint32_t c = tab + 8u * (uint32_t)k_hi;
  float4 hi = lds_f4(c - 16), lo = lds_f4(c - 32);    // (tab[k-2], tab[k-1]), (tab[k-4], tab[k-3])
#pragma unroll(kGoertzelUnroll)
  for (int k = k_hi; k > k_lo; k -= 4) {
    c -= 32;
    const float4 mh = lds_f4(c - 16), ml = lds_f4(c - 32);
    s2 = ffma2(rr, s1, ffma2(nn, s2, make_float2(hi.z, hi.w)));
    s1 = ffma2(rr, s2, ffma2(nn, s1, make_float2(hi.x, hi.y)));
    s2 = ffma2(rr, s1, ffma2(nn, s2, make_float2(lo.z, lo.w)));
    s1 = ffma2(rr, s2, ffma2(nn, s1, make_float2(lo.x, lo.y)));
    hi = mh; lo = ml;
  }
}

// EXACT: zeta = A^2/(4 x y) in double-double, A = x + y + mu (y complex on a deformed contour).
struct ZetaDD {
  double re_hi, re_lo, im, im2;   // Re zeta = hi + lo, Im zeta, (Im zeta)^2
};
__device__ __noinline__ ZetaDD zeta_dd(double xr, double xi, double yr, double yi, double mur, double mui,
                                       double mur_lo = 0.0, double mui_lo = 0.0) {
  const dd Ar = dd_add_d(dd_add_d(two_sum(xr, mur), yr), mur_lo), Ai = dd_add_d(dd_add_d(two_sum(xi, mui), yi), mui_lo);
  const dd A2r = dd_add(dd_mul(Ar, Ar), dd_neg(dd_mul(Ai, Ai)));
  const dd A2i = dd_scale2(dd_mul(Ar, Ai), 2.0);
  // den = 4 x y;  zeta = A^2 conj(den) / |den|^2
  const dd dr = dd_scale2(dd_add(two_prod(xr, yr), dd_neg(two_prod(xi, yi))), 4.0);
  const dd di = dd_scale2(dd_add(two_prod(xr, yi), two_prod(xi, yr)), 4.0);
  const dd nr = dd_add(dd_mul(A2r, dr), dd_mul(A2i, di));
  const dd ni = dd_add(dd_mul(A2i, dr), dd_neg(dd_mul(A2r, di)));
  const dd den = dd_add(dd_mul(dr, dr), dd_mul(di, di));
  const dd zr = dd_div(nr, den), zi = dd_div(ni, den);
  return {zr.hi, zr.lo, zi.hi, fma(zi.hi, zi.hi, 2.0 * zi.hi * zi.lo)};
}

// The direct sum with Re(zeta - t_j) formed from double-double zeta and t_j = z_j^2 = hi + lo exactly, so that it
// is accurate to an ulp of ITSELF next to a zero of a denominator:  a_j = (zeta_hi - t_hi) + (zeta_lo - t_lo),
// q_j = w_j/(a_j^2 + Im^2), U0 = sum q_j, Ua = sum q_j a_j, sum_j w_j/(zeta - t_j) = Ua - i Im U0, and
// S = mu0 + (eta - zeta) (Ua - i Im U0).  10 FP64 instructions per pair (the reciprocal as in pair_step).
// The FP64 kernel runs its NEAR lanes (zeta_lo = 0) and its EXACT lanes through this one loop.
__device__ __forceinline__ void direct_step(double zh, double zl, double zi2, double t, double tlo, double w,
                                            double& u0, double& ua) {
  const double a = (zh - t) + (zl - tlo);
  const double s = fma(a, a, zi2);
  const double r0 = rcp_seed(s);
  const double e = fma(-s, r0, 1.0);
  const double p = fma(e, e, e);
  const double v = r0 * w;
  const double q = fma(v, p, v);
  u0 += q;
  ua = fma(q, a, ua);
}
__device__ __forceinline__ cd angular_direct(cd eta, ZetaDD z, double mu0, const double* __restrict__ st,
                                             const double* __restrict__ stlo, const double* __restrict__ sw,
                                             int n_pairs) {
  double a0 = 0, a1 = 0, b0 = 0, b1 = 0;
  int j = 0;
#pragma unroll 1
  for (; j + 4 <= n_pairs; j += 4) {
    const double2 t01 = *reinterpret_cast<const double2*>(st + j), t23 = *reinterpret_cast<const double2*>(st + j + 2);
    const double2 l01 = *reinterpret_cast<const double2*>(stlo + j), l23 = *reinterpret_cast<const double2*>(stlo + j + 2);
    const double2 w01 = *reinterpret_cast<const double2*>(sw + j), w23 = *reinterpret_cast<const double2*>(sw + j + 2);
    direct_step(z.re_hi, z.re_lo, z.im2, t01.x, l01.x, w01.x, a0, a1);
    direct_step(z.re_hi, z.re_lo, z.im2, t01.y, l01.y, w01.y, b0, b1);
    direct_step(z.re_hi, z.re_lo, z.im2, t23.x, l23.x, w23.x, a0, a1);
    direct_step(z.re_hi, z.re_lo, z.im2, t23.y, l23.y, w23.y, b0, b1);
  }
  for (; j < n_pairs; ++j) direct_step(z.re_hi, z.re_lo, z.im2, st[j], stlo[j], sw[j], a0, a1);
  const double u0 = a0 + b0, ua = a1 + b1;
  const double cr = ua, ci = -z.im * u0;                       // sum_j w_j/(zeta - t_j)
  const double dr = (eta.re - z.re_hi) - z.re_lo, di = eta.im - z.im;
  return {mu0 + fma(dr, cr, -(di * ci)), fma(dr, ci, di * cr)};
}

// The direct routes on a rule split into blocks (FP64 kernel, n_pairs >= kBlkMinPairs): C(zeta) = sum_j w_j/(zeta - t_j)
// block by block.  For block b with interval [c - h, c + h]: w' = (zeta - c)/h, root = sqrt(w'^2 - 1) on the branch
// |w' + root| >= 1, s = 1/(w' + root) (|s| = 1/rho_b), and
//     sum_{j in b} w_j/(zeta - t_j) = (1/h) (2/root) sum'_k M_k s^k          (M_k: the block's Chebyshev moments)
// wherever rho_b^2 >= kBlkRho2Min (K_b <= kBlkTerms terms, one real-coefficient polynomial: 2 DFMA per term); the
// blocks next to zeta are summed pair by pair as before (DD: with zeta and t_j in double-double, the EXACT form).
// S = mu0 + (eta - zeta) C(zeta).  Near [0,1] a node-term costs its own block (and at times a neighbour) instead of
// every pair of the rule.
#ifndef GF_BLK_INLINE
#define GF_BLK_INLINE 1   // measured: as a called function 3 to 10 % slower on every config
#endif
template <bool DD, bool COUNT>
#if GF_BLK_INLINE
__device__ __forceinline__
#else
__device__ __noinline__
#endif
cd angular_blocked(cd eta, ZetaDD z, const Tabs<double>& tb, RouteCount& rc) {
  double u0 = 0.0, u1 = 0.0, v0 = 0.0, v1 = 0.0;   // direct sums: U0 = sum q_j; U1 = sum q_j a_j (DD) or sum q_j t_j
  cd far = {0.0, 0.0};
  // The blocks form a binary tree (level l joins 2^l leaves).  Walk the leaves from the left; at leaf b try the
  // largest block that starts there, then its left descendants: a block is taken by its series if |w'|^2 >= kBlkFarW2
  // (w' outside the disk that contains the ellipse rho_b^2 = kBlkRho2Min, so its series needs <= kBlkTerms terms);
  // a leaf that is not far is summed pair by pair.  A NaN fails the test: direct.
  int b = 0;
#pragma unroll 1
  while (b < tb.n_blk) {
    int l = min(tb.n_lev - 1, b ? __ffs(b) - 1 : kBlkMaxLev - 1), idx = 0;
    double wr = 0.0, wi = 0.0, ih = 0.0;
    bool is_far = false;
#pragma unroll 1
    for (; l >= 0; --l) {
      idx = (int)((tb.lev_pack >> (16 * l)) & 0xffffu) + (b >> l);
      const double2 ch = tb.blk[idx];
      ih = ch.y;
      wr = (z.re_hi - ch.x) * ih;
      wi = z.im * ih;
      if (fma(wr, wr, wi * wi) >= kBlkFarW2) { is_far = true; break; }
    }
    if (is_far) {
      const double qr = fma(wr, wr, -fma(wi, wi, 1.0)), qi = 2.0 * wr * wi;   // w'^2 - 1
      const double n2 = fma(qr, qr, qi * qi);
      const double rm = rsqrt_fast(n2);                                      // 1/|q| = 1/|root|^2
      const double h2 = 0.5 * fma(n2, rm, fabs(qr));
      const double rh = rsqrt_fast(h2);
      const double h = h2 * rh, kk = 0.5 * qi * rh;
      double ar = qr >= 0.0 ? h : fabs(kk), ai = qr >= 0.0 ? kk : copysign(h, qi);
      if (fma(wr, ar, wi * ai) < 0.0) { ar = -ar; ai = -ai; }
      const double Dr = wr + ar, Di = wi + ai;
      const double rho2 = fma(Dr, Dr, Di * Di);
      const double in = rcp_fast(rho2);
      const double sr = Dr * in, si = -Di * in, rr = sr + sr, ns = -in;
      // whole trips of four terms (the table holds kBlkTerms, a multiple of 4; extra terms are below the cut)
      const int K = min(((int)(112.f * rcp_ftz(lg2_ftz((float)rho2))) + 4) & ~3, kBlkTerms);
      const double2* M2 = reinterpret_cast<const double2*>(tb.blkM + idx * kBlkTerms) + (K >> 1);
      double p1 = 0.0, p2 = 0.0;
#pragma unroll 1
      for (int k = K; k > 0; k -= 4) {
        M2 -= 2;
        const double2 c23 = M2[1], c01 = M2[0];
        p2 = fma(rr, p1, fma(ns, p2, c23.y));
        p1 = fma(rr, p2, fma(ns, p1, c23.x));
        p2 = fma(rr, p1, fma(ns, p2, c01.y));
        p1 = fma(rr, p2, fma(ns, p1, c01.x));
      }
      const cd P = {fma(-p2, sr, p1), p2 * si};          // c_0 - c_1 conj(s)
      const double g2 = 2.0 * ih * rm;                   // (1/h) 2/root = (2/h) conj(root)/|root|^2
      far = cadd(far, cmul(cd{ar * g2, -ai * g2}, P));
      if (COUNT) { ++rc.blk_series; rc.blk_terms += K; rc.blk_leaves += 1 << l; }
      b += 1 << l;
    } else {
      const int j0 = b * kBlkPairs, j1 = min(j0 + kBlkPairs, tb.n_pairs);
      int j = j0;
#pragma unroll 1
      for (; j + 2 <= j1; j += 2) {
        if (DD) {
          direct_step(z.re_hi, z.re_lo, z.im2, tb.st[j], tb.stlo[j], tb.sw[j], u0, u1);
          direct_step(z.re_hi, z.re_lo, z.im2, tb.st[j + 1], tb.stlo[j + 1], tb.sw[j + 1], v0, v1);
        } else {
          pair_step(z.re_hi, z.im2, tb.st[j], tb.sw[j], u0, u1);
          pair_step(z.re_hi, z.im2, tb.st[j + 1], tb.sw[j + 1], v0, v1);
        }
      }
      if (j < j1) {
        if (DD) direct_step(z.re_hi, z.re_lo, z.im2, tb.st[j], tb.stlo[j], tb.sw[j], u0, u1);
        else pair_step(z.re_hi, z.im2, tb.st[j], tb.sw[j], u0, u1);
      }
      if (COUNT) { if (DD) rc.exact_pairs += j1 - j0; else rc.near_pairs += j1 - j0; }
      ++b;
    }
  }
  u0 += v0;
  u1 += v1;
  // sum over the direct blocks of w_j/(zeta - t_j): U1 - i Im U0 (DD: U1 = sum q a), conj(zeta) U0 - U1 otherwise
  const cd Cd = DD ? cd{u1, -z.im * u0} : cd{fma(z.re_hi, u0, -u1), -z.im * u0};
  const cd C = cadd(Cd, far);
  const double dr = (eta.re - z.re_hi) - z.re_lo, di = eta.im - z.im;
  return {tb.mu0 + fma(dr, C.re, -(di * C.im)), fma(dr, C.im, di * C.re)};
}

// ---------------------------------------------------------------------------------------------
// One (point, radial node, pole): S(delta, zeta) by the route zeta selects.  delta = eta - 1/4.
// WARP-COLLECTIVE: all 32 lanes must call it together (the series loop runs to the warp's longest
// series, lanes on other routes idle through it; extra terms are below the cut and harmless).
//   MOMENT  max(|Re zeta|, |Im zeta|) >= 4.5: s = 1/(zeta - 1/2), S = s [delta P(s) - N(s)] with the moments
//           a_k = sum_j w_j (t_j - 1/2)^k, b_k = sum_j w_j (t_j - 1/4)(t_j - 1/2)^k; |t - 1/2| <= 1/2 and
//           |s| <= 1/4, so K = kSeriesBits/(1 - log2|s|) + 2 <= 20 terms.
//   CHEB    else, with w = 2 zeta - 1 and s = 1/(w + sqrt(w^2 - 1)) the smaller root of s + 1/s = 2w
//           (|s| = 1/rho, rho the parameter of the ellipse with foci 0, 1 through zeta):
//           1/(zeta - t) = 4/sqrt(w^2-1) sum'_k s^k T_k(2t-1), so S = 4/sqrt(w^2-1) [delta P(s) - N(s)] with the
//           Chebyshev moments a_k = sum_j w_j T_k(2t_j-1), b_k = sum_j w_j (t_j - 1/4) T_k(2t_j-1) (k = 0 halved);
//           K terms from the Kreq table (prep_series_kreq), taken when K <= kmc and cheaper than the NEAR loop.
//   EXACT   zeta within tau of [0,1];   NEAR  the rest (zeta close to [0,1], or few angular nodes).
// ---------------------------------------------------------------------------------------------
// The series argument of one (point, radial node, pole), as route_setup leaves it
struct SeriesArg {
  cd sg, g;     // series argument s and prefactor
  double ns;    // -|s|^2
  int K, K1;    // terms needed; terms from K1 on may run in FP32 (their sum is below 2^-24 of the budget)
  int route;
};

template <typename T>
__device__ __forceinline__ SeriesArg route_setup(const Tabs<T>& tb, cd zeta) {
  SeriesArg o;
  // |Re zeta| or |Im zeta| >= 4.5, compared on the high words (4.5 = 0x40120000'00000000) to keep the test off the
  // FP64 pipe; a NaN lands here too and stays a NaN
  if (max(__double2hiint(zeta.re) & 0x7fffffff, __double2hiint(zeta.im) & 0x7fffffff) >= GF_MOMENT_HIWORD) {
    o.route = ROUTE_MOMENT;
    const double zc = zeta.re - 0.5;
    const double in = rcp_fast(fma(zc, zc, zeta.im * zeta.im));   // |zeta| < 2^500 (gf.h: domain)
    o.sg = {zc * in, -zeta.im * in};
    o.ns = -in;
    o.g = o.sg;
    // (|s|/2)^K <= 2^-kSeriesBits;  log2 |s|^2 <= -4 (-inf when it underflows in FP32: K = 2)
    const float l2 = lg2_ftz((float)in), il = rcp_ftz(2.f - l2);
    o.K = ((int)(2.f * kMomentBits * il) + 5) & ~3;         // + 2, rounded up to whole trips of four terms
    // FP32 from term K1 on: its rounding error 2^-24 A (|s|/2)^K1 (A <= 2.4 the recurrence's amplification) must stay
    // below 2^-kSeriesBits of the first-order term b_1 s of N, the smallest S can be: (|s|/2)^K1 <= 2^-(kSeriesBits-14) |s|
    o.K1 = min(((int)((2.f * (kMomentBits - 14.f - kFp32Slack) - l2) * il) + 5) & ~3, o.K);
  } else {
    // root = sqrt(zeta (zeta - 1)) = sqrt(w^2 - 1)/2, sign such that |w + 2 root| >= 1
    const double zm = zeta.re - 1.0, wr = fma(2.0, zeta.re, -1.0), wi = zeta.im + zeta.im;
    const double qr = fma(zeta.re, zm, -(zeta.im * zeta.im)), qi = zeta.im * wr;
    const double n2 = fma(qr, qr, qi * qi);
    const double rm = rsqrt_fast(n2);            // 1/|q|
    const double h2 = 0.5 * fma(n2, rm, fabs(qr));
    const double rh = rsqrt_fast(h2);
    const double h = h2 * rh, kk = 0.5 * qi * rh;
    // signs by integer operations on the high words (sign tests and negations would take FP64-pipe slots)
    const bool qpos = __double2hiint(qr) >= 0;
    double ar = qpos ? h : __hiloint2double(__double2hiint(kk) & 0x7fffffff, __double2loint(kk));   // |kk|
    double ai = qpos ? kk : copysign(h, qi);
    const int flip = __double2hiint(fma(wr, ar, wi * ai)) & 0x80000000;   // Re(conj(w) root) < 0: the other root
    ar = __hiloint2double(__double2hiint(ar) ^ flip, __double2loint(ar));
    ai = __hiloint2double(__double2hiint(ai) ^ flip, __double2loint(ai));
    // s = 1/(w + 2 root) = w - 2 root exactly ((w + 2 root)(w - 2 root) = w^2 - (w^2 - 1)): no reciprocal.  The
    // difference cancels |w|/|s| <= 2 |w|^2 of its operands' digits; |w| < 14 on this route (MOMENT beyond)
    const double sr = fma(-2.0, ar, wr), si = fma(-2.0, ai, wi);
    const double ns = fma(-sr, sr, -(si * si));        // -|s|^2 = -1/rho^2
    // terms needed at this rho (table made from the coefficients themselves, prep_series_kreq): entry 0 says "no usable
    // series" (log2 rho below kEllLo; zeta on [0,1] itself gives rho = 1 or NaN: entry 0 too), entry 1 + b is bin b.
    // index = floor((log2 rho - kEllLo)/kEllStep) + 1 by one FFMA from log2 |s|^2 and a conversion rounding down
    // (a NaN converts to 0), clamped: no comparison, no branch
    const float fidx = fmaf(lg2_ftz(fabsf((float)ns)), -0.5f / kEllStep, 1.f - kEllLo / kEllStep);
    int kq;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(kq)
                 : "r"(tb.a_kreq + 4u * (uint32_t)min(max(__float2int_rd(fidx), 0), kKreqBins - 1)));
    o.K = kq & 0xffff;     // 0xffff: no usable series in this bin
    o.K1 = kq >> 16;
    o.sg = {sr, si};
    o.ns = ns;
    const double g2 = rm + rm;                   // 4/sqrt(w^2-1) = 2 conj(root)/|q|
    o.g = {ar * g2, -ai * g2};
    o.route = ROUTE_CHEB;
    // CHEB whenever its series is short enough, whatever the direct loop would cost: next to [0,1] S is O(1), but
    // further out S can be 1e-7 of mu0 (the rule nearly integrates eta - t to zero) and the direct form
    // mu0 + (eta - zeta) C(zeta) would lose those digits; the series carry that cancellation in their tables
    if (!(o.K <= tb.kcap)) {
      o.K = o.K1 = 0;   // sg, ns stay as they are: this lane idles through the series loop and its result is dropped
      // |Im zeta| < tau and -tau < Re zeta < 1 + tau on the high words: tau and 1 + tau have a zero low word (tau a
      // power of two >= 2^-20), so a < c is hi(a) < hi(c) exactly; a NaN compares as a large number (NEAR, as before)
      constexpr double tau = sizeof(T) == 8 ? kTau64 : kTau32;
      const int th = __double2hiint(tau), oh = __double2hiint(1.0 + tau);
      const int zih = __double2hiint(zeta.im) & 0x7fffffff, zrh = __double2hiint(zeta.re);
      o.route = (zih < th && (zrh >= 0 ? zrh < oh : (zrh & 0x7fffffff) < th)) ? ROUTE_EXACT : ROUTE_NEAR;
    }
  }
  return o;
}

// S = g [delta P(s) - N(s)] from the recurrence's last two values of each polynomial
template <bool COUNT>
__device__ __forceinline__ cd series_finish(const SeriesArg& o, cd delta, double b0, double b1, double d0, double d1,
                                            RouteCount& rc) {
  const double Pr = fma(-b1, o.sg.re, b0), Pi = b1 * o.sg.im;     // c_0 - c_1 conj(s)
  const double Nr = fma(-d1, o.sg.re, d0), Ni = d1 * o.sg.im;
  const cd acc = {fma(delta.re, Pr, fma(-delta.im, Pi, -Nr)), fma(delta.re, Pi, fma(delta.im, Pr, -Ni))};
  if (COUNT) {
    rc.series_used += o.K;
    if (o.route == ROUTE_CHEB) ++rc.n_cheb; else ++rc.n_moment;
  }
  return cmul(o.g, acc);
}

// The direct loop for a lane on the NEAR or EXACT route
template <typename T, bool COUNT, bool BLK>
__device__ __forceinline__ cd direct_route(const Tabs<T>& tb, int route, bool warp_has_exact, cd x, cd y, cd delta,
                                           cd zeta, double mur, double mui, RouteCount& rc, double mur_lo = 0.0,
                                           double mui_lo = 0.0) {
  cd s;
  const cd eta = {__dadd_rn(0.25, delta.re), delta.im};
  bool dd_loop = true;
  if (BLK && sizeof(T) == 8 && tb.n_blk > 0) {
    // the rule is split into blocks: far blocks by their own short series, the blocks next to zeta pair by pair
    ZetaDD z = {zeta.re, 0.0, zeta.im, zeta.im * zeta.im};
    if (route == ROUTE_EXACT) z = zeta_dd(x.re, x.im, y.re, y.im, mur, mui, mur_lo, mui_lo);
    const Tabs<double>& tbd = reinterpret_cast<const Tabs<double>&>(tb);
    s = warp_has_exact ? angular_blocked<true, COUNT>(eta, z, tbd, rc) : angular_blocked<false, COUNT>(eta, z, tbd, rc);
    if (COUNT) { if (route == ROUTE_EXACT) ++rc.n_exact; else ++rc.n_near; }
    return s;
  }
  if (sizeof(T) == 8 && !warp_has_exact) {
    // no EXACT lane in this warp (voted by all 32 lanes before the routes diverge, so the choice of loop does
    // not depend on how the hardware groups the lanes): the 8-instruction pair
    s = angular_near<T>(eta, zeta, tb.mu0, tb.stT, tb.swT, tb.n_pairs);
    dd_loop = false;
  } else if (sizeof(T) == 8 || route == ROUTE_EXACT) {
    ZetaDD z = {zeta.re, 0.0, zeta.im, zeta.im * zeta.im};
    if (route == ROUTE_EXACT) z = zeta_dd(x.re, x.im, y.re, y.im, mur, mui, mur_lo, mui_lo);
    s = angular_direct(eta, z, tb.mu0, tb.st, tb.stlo, tb.sw, tb.n_pairs);
  } else {
    s = angular_near<T>(eta, zeta, tb.mu0, tb.stT, tb.swT, tb.n_pairs);
    dd_loop = false;
  }
  if (COUNT) {
    if (dd_loop) rc.exact_pairs += tb.n_pairs; else rc.near_pairs += tb.n_pairs;   // by loop, not by route
    if (route == ROUTE_EXACT) ++rc.n_exact; else ++rc.n_near;
  }
  return s;
}

// BLK: the kernel instantiation that carries the blocked direct routes (launched for rules of kBlkMinPairs and more
// folded pairs; the other instantiation does not pay their registers)
template <typename T, bool COUNT, bool BLK = false>
__device__ __forceinline__ cd node_term(const Tabs<T>& tb, cd x, cd y, cd delta, cd zeta, double mur, double mui,
                                        RouteCount& rc, double mur_lo = 0.0, double mui_lo = 0.0) {
  const SeriesArg o = route_setup<T>(tb, zeta);
  // every lane's K and K1 are multiples of 4 and at most kmc (route_setup): so are the warp's
  const int Kw = __reduce_max_sync(0xffffffffu, o.K);
  const bool warp_has_exact = __any_sync(0xffffffffu, o.route == ROUTE_EXACT);
  cd s = {0.0, 0.0};
  if (Kw > 0) {  // warp-uniform
    // terms Kw-1 .. K1w run in FP32 on the FMA pipe (the warp's largest K1: every lane's own need is met), the
    // recurrence's state is widened, and terms K1w-1 .. 0 run in FP64 (the FP32 variant: everything in FP32)
    const int K1w = sizeof(T) == 8 ? __reduce_max_sync(0xffffffffu, o.K1) : 0;
    const uint32_t tsel = o.route == ROUTE_CHEB ? (uint32_t)tb.kmc : 0u;   // the Chebyshev tables follow the moment tables
    float2 s1 = {0.f, 0.f}, s2 = {0.f, 0.f};
    goertzel_range_f32x2(tb.a_momf + 8u * tsel, Kw, K1w, (float)(o.sg.re + o.sg.re), (float)o.ns, s1, s2);
    double p1 = (double)s1.x, n1 = (double)s1.y, p2 = (double)s2.x, n2 = (double)s2.y;
    if (sizeof(T) == 8) goertzel_range(tb.a_mom + 16u * tsel, K1w, 0, o.sg.re + o.sg.re, o.ns, p1, p2, n1, n2);
    if (COUNT) { rc.series_exec += sizeof(T) == 8 ? K1w : Kw; rc.series_exec32 += sizeof(T) == 8 ? Kw - K1w : 0; }
    if (o.route <= ROUTE_CHEB) s = series_finish<COUNT>(o, delta, p1, p2, n1, n2, rc);
  }
  if (o.route >= ROUTE_NEAR)
    s = direct_route<T, COUNT, BLK>(tb, o.route, warp_has_exact, x, y, delta, zeta, mur, mui, rc, mur_lo, mui_lo);
  return s;
}

// Add this thread's counters to the launch's (one atomic per warp and counter)
__device__ __forceinline__ void flush_counters(const RouteCount& rc, bool active, unsigned long long* counters) {
  unsigned long long v[kNumCounters] = {rc.near_pairs, rc.series_exec, rc.exact_pairs,   rc.n_near,
                                        rc.n_moment,   rc.n_exact,     rc.n_cheb,        rc.series_used,
                                        rc.tails,      rc.series_exec32, rc.blk_series,  rc.blk_terms,
                                        rc.blk_leaves};
  for (int k = 0; k < kNumCounters; ++k) {
    if (!active) v[k] = 0;
    for (int o = 16; o; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    if ((threadIdx.x & 31) == 0 && v[k]) atomicAdd(counters + k, v[k]);
  }
}

// Stage the folded angular rule: pair j = nodes (j, n_ang-1-j); t = z^2 (hi + lo exactly), weight =
// w_j + w_mirror (the middle node of an odd rule enters once).  *bad is set if the rule is not symmetric.
__device__ void prep_angular(const EvalArgs& a, const BlobLayout& L, double* blob, int* bad) {
  float* tf = reinterpret_cast<float*>(blob + L.off_f32);
  float* wf = tf + L.npad;
  for (int j = threadIdx.x; j < L.npad; j += blockDim.x) {
    double t = 0, tlo = 0, w = 0;
    if (j < a.n_pairs) {
      const int jm = a.n_ang - 1 - j;
      const double zp = a.ang_nodes[jm], zm = a.ang_nodes[j];
      const double wp = a.ang_weights[jm], wm = a.ang_weights[j];
      const double tol = 16.0 * DBL_EPSILON;
      const bool ok = (jm == j) ? (fabs(zp) <= 1e-15)
                                : (fabs(zp + zm) <= tol * fabs(zp) && fabs(wp - wm) <= tol * fabs(wp));
      if (!ok) atomicOr(bad, kStatusAsymmetricRule);
      const dd tt = two_prod(zp, zp);
      t = tt.hi;
      tlo = tt.lo;
      w = (jm == j) ? wp : wp + wm;
    }
    blob[L.off_t + j] = t;
    blob[L.off_tlo + j] = tlo;
    blob[L.off_w + j] = w;
    if (L.off_f32 >= 0) {
      tf[j] = (float)t;
      wf[j] = (float)w;
    }
  }
}

// The series coefficients of the folded rule (call after prep_angular and a __syncthreads()):
//   phase 1 (prep_series_T): T_k(2 t_j - 1), k < kmc, by the three-term recurrence in double-double, one
//            thread per node j, into the scratch matrix [j][k];
//   phase 2 (prep_series_sums, after a __syncthreads()): one thread per k sums over the nodes with
//            double-double accumulators.
__device__ void prep_series_T(const EvalArgs& a, const BlobLayout& L, double* blob) {
  double* scratch = blob + L.off_scratch;
  for (int j = threadIdx.x; j < a.n_pairs; j += blockDim.x) {
    // s = 2 t - 1 with t = hi + lo exactly
    const dd s2 = dd_add_d(dd{2.0 * blob[L.off_t + j], 2.0 * blob[L.off_tlo + j]}, -1.0);
    const dd twos = dd_scale2(s2, 2.0);
    dd Tm = {1.0, 0.0}, Tk = s2;
    double* row = scratch + (size_t)j * L.kmc;
    row[0] = 1.0;
    row[1] = Tk.hi;
    for (int k = 2; k < L.kmc; ++k) {
      const dd Tn = dd_add(dd_mul(twos, Tk), dd_neg(Tm));
      Tm = Tk;
      Tk = Tn;
      row[k] = Tn.hi;
    }
  }
}

// Block tables of the folded rule, in two phases (both after prep_angular and a __syncthreads(), with another one
// between them): per block its interval [c - h, c + h] (the extreme t of its pairs) as (c, 1/h), and
// M_k = sum'_{j in b} w_j T_k(tau_j), tau_j = (t_j - c)/h, k < kBlkTerms (k = 0 halved).
//   phase 1 (prep_blocks_T): one thread per pair j runs the three-term recurrence once, in double-double, and leaves
//            w_j T_k(tau_j) (hi, lo) in the scratch [j][k];
//   phase 2 (prep_blocks_sums): one thread per (b, k) adds its block's 32 entries in double-double.
// block i of level l covers the pairs [i 2^l kBlkPairs, (i + 1) 2^l kBlkPairs) of the rule
__device__ __forceinline__ void block_interval(const BlobLayout& L, const double* blob, int l, int i, int n_pairs,
                                               double* c, double* ih) {
  const int span = kBlkPairs << l;
  const int j0 = i * span, j1 = min(j0 + span, n_pairs);
  double tmin = blob[L.off_t + j0], tmax = tmin;
  for (int j = j0 + 1; j < j1; ++j) {
    tmin = fmin(tmin, blob[L.off_t + j]);
    tmax = fmax(tmax, blob[L.off_t + j]);
  }
  *c = 0.5 * (tmin + tmax);
  *ih = 1.0 / fmax(0.5 * (tmax - tmin), 1e-12);
}
__device__ void prep_blocks_T(const EvalArgs& a, const BlobLayout& L, double* blob) {
  if (L.n_blk == 0) return;
  double2* S = reinterpret_cast<double2*>(blob + L.off_blkS);
  for (int e = threadIdx.x; e < a.n_pairs * L.n_lev; e += blockDim.x) {
    const int l = e / a.n_pairs, j = e % a.n_pairs;
    double c, ih;
    block_interval(L, blob, l, j / (kBlkPairs << l), a.n_pairs, &c, &ih);
    const double w = blob[L.off_w + j];
    const dd tau = dd_mul_d(dd_add_d(dd{blob[L.off_t + j], blob[L.off_tlo + j]}, -c), ih);
    const dd twot = dd_scale2(tau, 2.0);
    dd Tm = {1.0, 0.0}, Tk = tau;       // T_0, T_1
    double2* row = S + ((size_t)l * a.n_pairs + j) * kBlkTerms;
    row[0] = make_double2(w, 0.0);
    const dd w1 = dd_mul_d(Tk, w);
    row[1] = make_double2(w1.hi, w1.lo);
    for (int q = 2; q < kBlkTerms; ++q) {
      const dd Tn = dd_add(dd_mul(twot, Tk), dd_neg(Tm));
      Tm = Tk;
      Tk = Tn;
      const dd wq = dd_mul_d(Tk, w);
      row[q] = make_double2(wq.hi, wq.lo);
    }
  }
}
__device__ void prep_blocks_sums(const EvalArgs& a, const BlobLayout& L, double* blob) {
  const double2* S = reinterpret_cast<const double2*>(blob + L.off_blkS);
  for (int e = threadIdx.x; e < L.n_blk_all * kBlkTerms; e += blockDim.x) {
    const int idx = e / kBlkTerms, k = e % kBlkTerms;
    int l = 0;
    while (l + 1 < L.n_lev && idx >= L.lev_off[l + 1]) ++l;
    const int i = idx - L.lev_off[l], span = kBlkPairs << l;
    const int j0 = i * span, j1 = min(j0 + span, a.n_pairs);
    dd acc = {0.0, 0.0};
    for (int j = j0; j < j1; ++j) {
      const double2 v = S[((size_t)l * a.n_pairs + j) * kBlkTerms + k];
      acc = dd_add(acc, dd{v.x, v.y});
    }
    blob[L.off_blkM + idx * kBlkTerms + k] = (k == 0 ? 0.5 : 1.0) * acc.hi;
    if (k == 0) {
      double c, ih;
      block_interval(L, blob, l, i, a.n_pairs, &c, &ih);
      blob[L.off_blk + 2 * idx] = c;
      blob[L.off_blk + 2 * idx + 1] = ih;
    }
  }
}

__device__ __forceinline__ double powi(double t, int k) {
  double r = 1.0;
  while (k) {
    if (k & 1) r *= t;
    t *= t;
    k >>= 1;
  }
  return r;
}

__device__ void prep_series_sums(const EvalArgs& a, const BlobLayout& L, double* blob, dd (*s_cpart)[2][kMomTerms]) {
  const double* scratch = blob + L.off_scratch;
  float2* momf = reinterpret_cast<float2*>(blob + L.off_sf);
  float2* chebf = momf + L.kmc;
  for (int k = threadIdx.x; k < L.kmc; k += blockDim.x) {
    dd tau = {0.0, 0.0}, nu = {0.0, 0.0}, tau1 = {0.0, 0.0}, nu1 = {0.0, 0.0}, mo = {0.0, 0.0}, no = {0.0, 0.0};
    for (int j = 0; j < a.n_pairs; j += 2) {   // two independent accumulator chains (npad is even, padding has w = 0)
      const double t0 = blob[L.off_t + j], w0 = blob[L.off_w + j], t1 = blob[L.off_t + j + 1], w1 = blob[L.off_w + j + 1];
      const double wT0 = w0 * scratch[(size_t)j * L.kmc + k];
      const double wT1 = j + 1 < a.n_pairs ? w1 * scratch[(size_t)(j + 1) * L.kmc + k] : 0.0;
      tau = dd_add_d(tau, wT0);
      tau1 = dd_add_d(tau1, wT1);
      nu = dd_add(nu, dd_mul_d(dd_add_d(two_sum(t0, -0.25), blob[L.off_tlo + j]), wT0));
      nu1 = dd_add(nu1, dd_mul_d(dd_add_d(two_sum(t1, -0.25), blob[L.off_tlo + j + 1]), wT1));
    }
    tau = dd_add(tau, tau1);
    nu = dd_add(nu, nu1);
    {
      // centred moments: thread k sums chunk k/32 of 8 of the nodes for the moment k%32; combined below
      const int km = k % kMomTerms, c = (k / kMomTerms) % 8;
      if (k < 8 * kMomTerms) {
        for (int j = c; j < a.n_pairs; j += 8) {
          const double t = blob[L.off_t + j];
          const double wp = blob[L.off_w + j] * powi(t - 0.5, km);
          mo = dd_add_d(mo, wp);
          // t - 1/4 with t = hi + lo: b_0 = sum_j w_j (t_j - 1/4) is ~1e-8 of its terms (0 in the continuum)
          no = dd_add(no, dd_mul_d(dd_add_d(two_sum(t, -0.25), blob[L.off_tlo + j]), wp));
        }
        s_cpart[c][0][km] = mo;
        s_cpart[c][1][km] = no;
      }
    }
    const double half = k == 0 ? 0.5 : 1.0;   // sum' : the k = 0 term of a Chebyshev series is halved
    const double c0 = half * tau.hi, c1 = half * nu.hi;
    blob[L.off_cheb + 2 * k] = c0;
    blob[L.off_cheb + 2 * k + 1] = c1;
    chebf[k] = make_float2((float)c0, (float)c1);
  }
  __syncthreads();
  for (int k = threadIdx.x; k < L.kmc; k += blockDim.x) {
    dd mo = {0.0, 0.0}, no = {0.0, 0.0};
    if (k < kMomTerms)
      for (int c = 0; c < 8; ++c) {
        mo = dd_add(mo, s_cpart[c][0][k]);
        no = dd_add(no, s_cpart[c][1][k]);
      }
    const double m0 = mo.hi, m1 = no.hi;     // zero beyond kMomTerms
    blob[L.off_mom + 2 * k] = m0;
    blob[L.off_mom + 2 * k + 1] = m1;
    momf[k] = make_float2((float)m0, (float)m1);
  }
}

// Taylor orders n > 0 (gf_taylor.cu): the n + 2 series tables per family, the moments of the measures w_j t_j^q,
//   momA[k][q] = sum_j w_j t_j^q (t_j - 1/2)^k (k < kMomTerms),  chebA[k][q] = sum'_j w_j t_j^q T_k(2 t_j - 1) (k < kmc),
// in double-double (call after prep_series_T and a __syncthreads(): the T_k matrix is in the scratch).
__device__ void prep_series_A(const EvalArgs& a, const BlobLayout& L, double* blob) {
  const int NA = L.n_poly;
  const double* scratch = blob + L.off_scratch;
  for (int k = threadIdx.x; k < L.kmc; k += blockDim.x) {
    dd ch[kMaxTaylor + 2], mo[kMaxTaylor + 2];
    for (int q = 0; q < NA; ++q) ch[q] = mo[q] = dd{0.0, 0.0};
    for (int j = 0; j < a.n_pairs; ++j) {
      const dd t = {blob[L.off_t + j], blob[L.off_tlo + j]};
      const double w = blob[L.off_w + j];
      const double wT = w * scratch[(size_t)j * L.kmc + k];
      dd cp = {0.0, 0.0};                   // w (t - 1/2)^k, k < kMomTerms
      if (k < kMomTerms) {
        const dd c = dd_add_d(t, -0.5);
        dd p = {1.0, 0.0}, b = c;
        for (int ex = k; ex; ex >>= 1) {
          if (ex & 1) p = dd_mul(p, b);
          b = dd_mul(b, b);
        }
        cp = dd_mul_d(p, w);
      }
      dd ta = {1.0, 0.0};                   // t^q
      for (int q = 0; q < NA; ++q) {
        ch[q] = dd_add(ch[q], dd_mul_d(ta, wT));
        if (k < kMomTerms) mo[q] = dd_add(mo[q], dd_mul(ta, cp));
        ta = dd_mul(ta, t);
      }
    }
    const double half = k == 0 ? 0.5 : 1.0;   // sum': the k = 0 term of a Chebyshev series is halved
    for (int q = 0; q < NA; ++q) {
      blob[L.off_chebA + k * NA + q] = half * ch[q].hi;
      if (k < kMomTerms) blob[L.off_momA + k * NA + q] = mo[q].hi;
    }
  }
}

// Kreq[b]: the number of Chebyshev terms after which every dropped term is below 2^-(kSeriesBits+2) of the leading
// coefficient when log2(rho) >= kEllLo + b kEllStep: the smallest K with |c_j| rho^-j <= 2^-(kSeriesBits+2) |c_0| for all
// j >= K, c_j the larger of the two coefficients.  For a rule that integrates the measure well the c_j beyond
// the first few are the rule's defect (~1e-7), so far fewer terms are needed than rho^-K <= 2^-60 asks for.
// Coefficients beyond kmc are not known: a bin is usable only if rho^-kmc <= 2^-60.
// coef: the Chebyshev tables, n_poly coefficients per k ([k][n_poly]); c_j is the largest of them in modulus.
__device__ void prep_series_kreq(const BlobLayout& L, double* blob, float* s_lc /* [kKmc] shared */, const double* coef,
                                 int n_poly) {
  int* kreq = reinterpret_cast<int*>(blob + L.off_kreq);
  auto cmax = [&](int j) {
    double m = 0.0;
    for (int q = 0; q < n_poly; ++q) m = fmax(m, fabs(coef[j * n_poly + q]));
    return m;
  };
  const double c00 = cmax(0);
  for (int j = threadIdx.x; j < L.kmc; j += blockDim.x)   // log2 |c_j / c_0|, rounded up a little (c = 0: -inf)
    s_lc[j] = (float)log2(cmax(j) / c00) + 1e-3f;
  __syncthreads();
  if (threadIdx.x == 0) kreq[0] = 0xffff;   // entry 0: log2(rho) below kEllLo, no usable series (route_setup)
  for (int b = threadIdx.x; b < kKreqBins - 1; b += blockDim.x) {
    const float ell = kEllLo + (float)b * kEllStep;
    int K = 0xffff, K1 = 0;
    if (ell * L.kmc >= 60.f) {
      K = 4;
      // the dropped terms sum like a geometric series: the bound is on |c_j| rho^-j / (1 - 1/rho), so that a slowly
      // converging series next to [0,1] (rho -> 1.18: a factor 6.5) is cut as safely as a fast one
      const float geo = log2f(1.f / (1.f - exp2f(-ell)));
      for (int j = L.kmc - 1; j >= 4; --j)
        if (s_lc[j] - (float)j * ell + geo > -kSeriesBits - 2.f) {
          K = j + 1;
          break;
        }
      K = (K + 4) & ~3;   // one spare term, whole trips of four terms (kmc is a multiple of 4)
      // K1: from here on the terms may run in FP32.  A rounding error of the recurrence at step k acts like a
      // perturbation of c_k by <= 4 2^-24 max_{j>=k}|c_j| / (1 - 1/rho)^2, and the perturbations sum like a geometric
      // series: the FP32 phase costs <= 2^-22 max_{j>=K1} |c_j| rho^-j / (1 - 1/rho)^3, held below the truncation
      // budget: |c_j| rho^-j <= 2^-(kSeriesBits - 20) (1 - 1/rho)^3 |c_0| for all j >= K1
      const float thr = kSeriesBits - 20.f - kFp32Slack + 3.f * geo;
      for (int j = L.kmc - 1; j >= 0; --j)
        if (s_lc[j] - (float)j * ell > -thr) {
          K1 = j + 1;
          break;
        }
      K1 = min((K1 + 3) & ~3, K);
    }
    kreq[b + 1] = K | (K1 << 16);
  }
}

// ---------------------------------------------------------------------------------------------
// Large-y tail (REAL contour; gf_eval.cu header "Tail"): tables that do not depend on x.
//   gamma_{n,k} = -nu_k C(n+k, n-1-k) - (mu_k/4) C(n+k-1, n-2-k),  0 <= k < n <= kTailN, with the monomial
//   moments mu_k = sum_j w_j t_j^k and nu_k = sum_j w_j (t_j - 1/4) t_j^k of the folded rule (double-double);
//   Rhat_n(i0) = sum_{i >= i0} pref_i (y_i0 / y_i)^n by the downward recurrence
//   Rhat_n(i) = pref_i + (y_i/y_{i+1})^n Rhat_n(i+1), the powers of q_i = y_i/y_{i+1} in double-double.
// ---------------------------------------------------------------------------------------------
__device__ dd dd_binom(int n, int k) {   // C(n, k) as a double-double (exact while it fits 106 bits)
  if (k < 0 || k > n) return {0.0, 0.0};
  if (k > n - k) k = n - k;
  dd c = {1.0, 0.0};
  for (int i = 1; i <= k; ++i) c = dd_div_d(dd_mul_d(c, (double)(n - k + i)), (double)i);   // stays an integer
  return c;
}

// phase A (after prep_angular + __syncthreads): thread (k, c) sums chunk c of 8 of the nodes into s_part[c][k]
// (mu in [0], nu in [1]); phase B adds the 8 parts
__device__ void prep_tail_moments(const EvalArgs& a, const BlobLayout& L, const double* blob, dd (*s_part)[2][kTailN]) {
  for (int e = threadIdx.x; e < 8 * kTailN; e += blockDim.x) {
    const int k = e % kTailN, c = e / kTailN;
    dd mu = {0.0, 0.0}, nu = {0.0, 0.0};
    for (int j = c; j < a.n_pairs; j += 8) {
      const dd t = {blob[L.off_t + j], blob[L.off_tlo + j]};
      dd p = {1.0, 0.0}, b = t;   // t^k
      for (int ex = k; ex; ex >>= 1) {
        if (ex & 1) p = dd_mul(p, b);
        b = dd_mul(b, b);
      }
      const dd wp = dd_mul_d(p, blob[L.off_w + j]);
      mu = dd_add(mu, wp);
      nu = dd_add(nu, dd_mul(wp, dd_add_d(t, -0.25)));
    }
    s_part[c][0][k] = mu;
    s_part[c][1][k] = nu;
  }
}
// phase B (after a __syncthreads): gamma table
__device__ void prep_tail_gamma(const BlobLayout& L, double* blob, dd (*s_part)[2][kTailN], dd* s_mu, dd* s_nu) {
  for (int k = threadIdx.x; k < 2 * kTailN; k += blockDim.x) {
    dd acc = {0.0, 0.0};
    for (int c = 0; c < 8; ++c) acc = dd_add(acc, s_part[c][k / kTailN][k % kTailN]);
    (k < kTailN ? s_mu : s_nu)[k % kTailN] = acc;
  }
  __syncthreads();
  for (int e = threadIdx.x; e < kTailN * (kTailN + 1) / 2; e += blockDim.x) {
    int n = 1;
    while (n * (n + 1) / 2 <= e) ++n;      // row n holds k = 0 .. n-1 at n(n-1)/2
    const int k = e - n * (n - 1) / 2;
    const dd t1 = dd_mul(s_nu[k], dd_binom(n + k, n - 1 - k));
    const dd t2 = dd_scale2(dd_mul(s_mu[k], dd_binom(n + k - 1, n - 2 - k)), 0.25);
    blob[L.off_gam + e] = dd_neg(dd_add(t1, t2)).hi;
    if (L.off_gam2 >= 0) blob[L.off_gam2 + e] = dd_mul(s_mu[k], dd_binom(n + k, n - 1 - k)).hi;   // kappa_{n,k}
  }
}
// One set of Rhat tables: the n real nodes y[0..n) (ascending) with prefactors pref[r][i] = (re, im) at
// pref[2 (r stride + i)], r < n_pref; out: double2 R[n_pref][n + 1][kTailN]; s2, s3: scratch of 2 kTailN n and
// kTailN n + 2 kTailChunks (2 n_pref kTailN + kTailN) doubles.
struct TailJob {
  int n, n_pref, stride;
  const double* y;
  const double* pref;
  double2* R;
  double *s2, *s3;
};
// phase C: thread per node i: q_i^n, n = 1..kTailN, in double-double into the scratch as (hi, lo) [i][n] (n fastest:
// phase D's warps hold 32 consecutive n of one node)
__device__ void prep_tail_powers(const TailJob& J) {
  double2* q2 = reinterpret_cast<double2*>(J.s2);
  for (int i = threadIdx.x; i < J.n; i += blockDim.x) {
    dd q = {1.0, 0.0};
    if (i + 1 < J.n) q = dd_div(dd{J.y[i], 0.0}, dd{J.y[i + 1], 0.0});
    dd p = q;
    for (int n = 0; n < kTailN; ++n) {
      q2[(size_t)i * kTailN + n] = make_double2(p.hi, p.lo);
      p = dd_mul(p, q);
    }
  }
}
// phase D (after a __syncthreads): the downward recurrence, split into kTailChunks runs of nodes so that the CTA's
// threads share it: item = (pole r, power n + 1, real / imaginary part), run c.  Pass 1 runs the recurrence inside
// each run from 0 (L_c(i)) with the run's product of q (Q_c(i)); pass 2 folds the runs above c into the carry
// Rhat(end of run c) in double-double and completes Rhat(i) = L_c(i) + Q_c(i) carry.
constexpr int kTailChunks = 16;
__device__ void prep_tail_sums(const TailJob& J) {
  const double2* q2 = reinterpret_cast<const double2*>(J.s2);
  double2* R = J.R;
  const int n_items = 2 * J.n_pref * kTailN, CL = (J.n + kTailChunks - 1) / kTailChunks;
  double* Qs = J.s3;                                                   // Q_c(i), [n][kTailN]
  dd* Lstart = reinterpret_cast<dd*>(Qs + (size_t)kTailN * J.n);       // [kTailChunks][n_items]
  dd* Qstart = Lstart + (size_t)n_items * kTailChunks;                 // [kTailChunks][kTailN]
  for (int w = threadIdx.x; w < n_items * kTailChunks; w += blockDim.x) {
    const int e = w % n_items, c = w / n_items;
    const int part = e / (J.n_pref * kTailN), r = (e / kTailN) % J.n_pref, n = e % kTailN;
    double* Rr = reinterpret_cast<double*>(R + (size_t)r * (J.n + 1) * kTailN) + part;
    const bool owner = r == 0 && part == 0;
    if (c == 0) Rr[2 * ((size_t)J.n * kTailN + n)] = 0.0;
    dd acc = {0.0, 0.0}, Q = {1.0, 0.0};
    // the next node's operands are fetched before this node's result is stored (the stores could alias the loads
    // as far as the compiler knows: without this every step would wait a whole L2 round trip)
    const int i_hi = min((c + 1) * CL, J.n) - 1, i_lo = c * CL;
    double2 nq = make_double2(0.0, 0.0);
    double np = 0.0;
    if (i_hi >= i_lo) {
      nq = q2[(size_t)i_hi * kTailN + n];
      np = J.pref[2 * (r * J.stride + i_hi) + part];
    }
    for (int i = i_hi; i >= i_lo; --i) {
      const dd q = {nq.x, nq.y};
      const double pf = np;
      if (i > i_lo) {
        nq = q2[(size_t)(i - 1) * kTailN + n];
        np = J.pref[2 * (r * J.stride + i - 1) + part];
      }
      acc = dd_add_d(dd_mul(acc, q), pf);
      Rr[2 * ((size_t)i * kTailN + n)] = acc.hi;
      if (owner) {
        Q = dd_mul(Q, q);
        Qs[(size_t)i * kTailN + n] = Q.hi;
      }
    }
    Lstart[(size_t)c * n_items + e] = acc;
    if (owner) Qstart[(size_t)c * kTailN + n] = Q;
  }
  __syncthreads();
  for (int w = threadIdx.x; w < n_items * kTailChunks; w += blockDim.x) {
    const int e = w % n_items, c = w / n_items;
    const int part = e / (J.n_pref * kTailN), r = (e / kTailN) % J.n_pref, n = e % kTailN;
    double* Rr = reinterpret_cast<double*>(R + (size_t)r * (J.n + 1) * kTailN) + part;
    dd carry = {0.0, 0.0};
    for (int cc = kTailChunks - 1; cc > c; --cc)
      carry = dd_add(Lstart[(size_t)cc * n_items + e], dd_mul(Qstart[(size_t)cc * kTailN + n], carry));
    if (carry.hi != 0.0 || carry.lo != 0.0) {
      const int i_hi = min((c + 1) * CL, J.n) - 1, i_lo = c * CL;
      for (int ib = i_hi; ib >= i_lo; ib -= 4) {   // four independent nodes: loads first, then the stores
        double qv[4], rv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (ib - u >= i_lo) {
            qv[u] = Qs[(size_t)(ib - u) * kTailN + n];
            rv[u] = Rr[2 * ((size_t)(ib - u) * kTailN + n)];
          }
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (ib - u >= i_lo) Rr[2 * ((size_t)(ib - u) * kTailN + n)] = dd_add_d(dd_mul_d(carry, qv[u]), rv[u]).hi;
      }
    }
  }
}
// the REAL contour's job: all n_rad nodes of the prepared block
__device__ __forceinline__ TailJob real_tail_job(const EvalArgs& a, const BlobLayout& L, double* blob) {
  return TailJob{a.n_rad, L.n_pref, L.n_rad_pad, blob + L.off_y, blob + L.off_pref,
                 reinterpret_cast<double2*>(blob + L.off_tail), blob + L.off_scratch2, blob + L.off_scratch3};
}

// D1(y) for real y (REAL contour): massive 1/(y + m2) or rational (y + M2)/(y^2 + a y + b).
__device__ __forceinline__ cd line_k_real(const gf_propagator& p, double y) {
  if (p.kind == GF_PROP_MASSIVE) return cinv(cd{y + p.m2_re, p.m2_im});
  return cd{(y + p.M2) / fma(y, y + p.a, p.b), 0.0};
}

// y = s0 expm1(u L) in double-double, rounded once (readings G3/G4, G18)
__device__ __forceinline__ double radial_node(double t, dd Llog, double s0) {
  const double u = 0.5 * (t + 1.0);
  return dd_mul_d(dd_expm1(dd_mul_d(Llog, u)), s0).hi;
}


// ---------------------------------------------------------------------------------------------
// Tail: all radial nodes with y_i >= Y0(x) at once.  With a = x + mu, eps = 1/y:
//   S(x, y) = sum_k omega^(k+1) [delta mu_k - nu_k],  omega = 4 x eps/(1 + a eps)^2,  delta = a eps/4
//           = sum_n eps^n X h_n(X, Z),   X = 4x, Z = -a,   h_n = sum_{k<n} gamma_{n,k} X^k Z^(n-1-k)
// (binomial series of (1 + a eps)^(-2k-2); gamma_{n,k} in gf_routes.cuh).  The series converges absolutely,
// term n below 4^-n, for y >= Y0 = 4 (sqrt|x| + sqrt(|x| + |a|))^2, so
//   sum_{i >= i0} pref_i S(x, y_i) = X sum_n h_n sum_{i >= i0} pref_i y_i^-n = (X/y_i0) sum_n h_n(X/y_i0, Z/y_i0) Rhat_n(i0)
// with the x-independent tables Rhat_n(i0) made once per launch.  h_n is a real-coefficient polynomial in the
// ratio of X and Z (the smaller over the larger) and is evaluated by the same second-order recurrence as the
// angular series.  A log-mapped radial rule has most of its nodes in this tail (about 60 % on the production
// scan), and they cost kTailN (kTailN + 1) DFMA per point instead of a series each.
// ---------------------------------------------------------------------------------------------
#ifndef GF_TAIL_ILP
#define GF_TAIL_ILP 1
#endif
__device__ __forceinline__ cd tail_series(const double* __restrict__ gam, const double2* __restrict__ Rrow, cd x,
                                          cd a, double invy0) {
  const cd X = {4.0 * x.re * invy0, 4.0 * x.im * invy0}, Z = {-a.re * invy0, -a.im * invy0};
  const double nX = fma(X.re, X.re, X.im * X.im), nZ = fma(Z.re, Z.re, Z.im * Z.im);
  const bool fwd = nX <= nZ;                        // powers of X/Z, else of Z/X
  const cd base = fwd ? Z : X, oth = fwd ? X : Z;
  const double inb = 1.0 / (fwd ? nZ : nX);
  const cd rho = {fma(oth.re, base.re, oth.im * base.im) * inb, fma(oth.im, base.re, -(oth.re * base.im)) * inb};
  const double rr = rho.re + rho.re, ns = -fma(rho.re, rho.re, rho.im * rho.im);
  cd pw = {1.0, 0.0}, acc = {0.0, 0.0};
  const double* row = gam;
#if GF_TAIL_ILP
  // rows n and n + 1 together (kTailN is even): two independent recurrences, so that the one dependent chain per point
  // that the series is does not wait on its own latency.  Row n holds the n coefficients of h_n, highest power of the
  // ratio first when read from its end (fwd) or from its start.
  static_assert(kTailN % 2 == 0, "the tail series takes its rows in pairs");
  const int step = fwd ? -1 : 1;
  const cd base2 = csqr(base);
#pragma unroll 1
  for (int n = 1; n <= kTailN; n += 2) {
    const double* rowB = row + n;                       // row n + 1
    const double* cA = fwd ? row + n - 1 : row;
    const double* cB = fwd ? rowB + n : rowB;
    double a0 = 0.0, a1 = 0.0, b1 = 0.0;
    double b0 = *cB;                                    // row n + 1 is one coefficient longer
    cB += step;
#pragma unroll 2
    for (int j = 0; j < n; ++j, cA += step, cB += step) {
      const double ta = fma(rr, a0, fma(ns, a1, *cA));
      const double tb = fma(rr, b0, fma(ns, b1, *cB));
      a1 = a0; a0 = ta;
      b1 = b0; b0 = tb;
    }
    const cd PA = {fma(-a1, rho.re, a0), a1 * rho.im};   // c_0 - c_1 conj(rho)
    const cd PB = {fma(-b1, rho.re, b0), b1 * rho.im};
    const double2 RA = Rrow[n - 1], RB = Rrow[n];
    // acc += pw [PA RA + base PB RB]
    const cd tB = cmul(cmul(PB, base), cd{RB.x, RB.y});
    const cd tA = cmul(PA, cd{RA.x, RA.y});
    acc = cadd(acc, cmul(pw, cadd(tA, tB)));
    pw = cmul(pw, base2);
    row += 2 * n + 1;
  }
#else
#pragma unroll 1
  for (int n = 1; n <= kTailN; ++n) {
    double b0 = 0.0, b1 = 0.0;
    const double* c = fwd ? row + n - 1 : row;      // highest power of the ratio first
    const int step = fwd ? -1 : 1;
    if (n & 1) {
      b0 = *c;
      c += step;
    }
#pragma unroll 2
    for (int j = n >> 1; j > 0; --j, c += 2 * step) {   // two coefficients per trip, roles of b0, b1 alternate
      b1 = fma(rr, b0, fma(ns, b1, c[0]));
      b0 = fma(rr, b1, fma(ns, b0, c[step]));
    }
    const cd P = {fma(-b1, rho.re, b0), b1 * rho.im};   // c_0 - c_1 conj(rho)
    const double2 R = Rrow[n - 1];
    acc = cadd(acc, cmul(cmul(P, pw), cd{R.x, R.y}));
    pw = cmul(pw, base);
    row += n;
  }
#endif
  return cmul(X, acc);
}


}  // namespace
}  // namespace gf
