// gf_routes.cuh -- device code shared by the two evaluation kernels (gf_eval.cu: REAL contour, nodes
// prepared once per launch; gf_contour.cu: contours that depend on the grid point): the three routes that
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

constexpr int kKmCap = 60;           // most far-field terms ever used (|zeta| >= 2 -> K <= 59)
constexpr int kFarBits = 116;        // 2 * 58: K = kFarBits / (2 ilogb|zeta|) + 1
constexpr double kTau64 = 0x1p-8;    // EXACT route inside this distance of [0,1] (FP64)
constexpr double kTau32 = 0x1p-4;    // the FP32 variant's NEAR loop is only good further away

struct cd {
  double re, im;
};
__device__ __forceinline__ cd cmul(cd a, cd b) {
  return {fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re)};
}
__device__ __forceinline__ cd cscale(cd a, double s) { return {a.re * s, a.im * s}; }
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
    if (spin > (1LL << 26)) __trap();  // a 20 KB copy that has not landed after seconds: fail, do not hang
  }
}

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

template <typename T>
struct Vec2;
template <>
struct Vec2<double> { typedef double2 type; };
template <>
struct Vec2<float> { typedef float2 type; };

// S = mu0 - (zeta - eta)(conj(zeta) U0 - U1).  Two independent accumulator sets (even / odd pairs).
template <typename T>
__device__ __forceinline__ cd angular_near(cd eta, cd zeta, double mu0, const T* __restrict__ st,
                                           const T* __restrict__ sw, int n_pairs) {
  typedef typename Vec2<T>::type V2;
  const T zr = (T)zeta.re;
  const T zi2 = (T)(zeta.im * zeta.im);
  T a0 = 0, a1 = 0, b0 = 0, b1 = 0;
  int j = 0;
#pragma unroll 1
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

// FAR: S = omega [ delta P(omega) + N(omega) ], K terms (Horner from the top).
__device__ __forceinline__ cd angular_far(cd delta, cd zeta, int K, const double* __restrict__ smu,
                                          const double* __restrict__ snu) {
  const cd om = cinv(zeta);
  double pr = smu[K - 1], pi = 0.0, nr = snu[K - 1], ni = 0.0;
#pragma unroll 1
  for (int k = K - 2; k >= 0; --k) {
    const double m = smu[k], n = snu[k];
    const double tpr = fma(pr, om.re, fma(-pi, om.im, m));
    pi = fma(pr, om.im, pi * om.re);
    pr = tpr;
    const double tnr = fma(nr, om.re, fma(-ni, om.im, n));
    ni = fma(nr, om.im, ni * om.re);
    nr = tnr;
  }
  const cd acc = {fma(delta.re, pr, fma(-delta.im, pi, nr)), fma(delta.re, pi, fma(delta.im, pr, ni))};
  return cmul(om, acc);
}

// EXACT: zeta = A^2/(4 x y) in double-double, A = x + y + mu (y complex on a deformed contour); every
// term formed directly.
__device__ __noinline__ cd angular_exact(double xr, double xi, double yr, double yi, double mur, double mui, cd eta,
                                         const double* __restrict__ st, const double* __restrict__ stlo,
                                         const double* __restrict__ sw, int n_pairs) {
  const dd Ar = dd_add_d(two_sum(xr, mur), yr), Ai = dd_add_d(two_sum(xi, mui), yi);
  const dd A2r = dd_add(dd_mul(Ar, Ar), dd_neg(dd_mul(Ai, Ai)));
  const dd A2i = dd_scale2(dd_mul(Ar, Ai), 2.0);
  // den = 4 x y;  zeta = A^2 conj(den) / |den|^2
  const dd dr = dd_scale2(dd_add(two_prod(xr, yr), dd_neg(two_prod(xi, yi))), 4.0);
  const dd di = dd_scale2(dd_add(two_prod(xr, yi), two_prod(xi, yr)), 4.0);
  const dd nr = dd_add(dd_mul(A2r, dr), dd_mul(A2i, di));
  const dd ni = dd_add(dd_mul(A2i, dr), dd_neg(dd_mul(A2r, di)));
  const dd den = dd_add(dd_mul(dr, dr), dd_mul(di, di));
  const dd zr = dd_div(nr, den), zi = dd_div(ni, den);
  const double zi2 = fma(zi.hi, zi.hi, 2.0 * zi.hi * zi.lo);
  double sr = 0.0, si = 0.0;
#pragma unroll 1
  for (int j = 0; j < n_pairs; ++j) {
    const double t = st[j];
    const double a = (zr.hi - t) + (zr.lo - stlo[j]);  // Re(zeta - t), accurate to an ulp of ITSELF
    const double s = fma(a, a, zi2);
    const double wq = sw[j] / s;
    const double d = eta.re - t;
    // (eta - t) conj(zeta - t)
    sr = fma(wq, fma(d, a, eta.im * zi.hi), sr);
    si = fma(wq, fma(eta.im, a, -(d * zi.hi)), si);
  }
  return {sr, si};
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
      if (!ok) atomicExch(bad, 1);
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

__device__ __forceinline__ double powi(double t, int k) {
  double r = 1.0;
  while (k) {
    if (k & 1) r *= t;
    t *= t;
    k >>= 1;
  }
  return r;
}

}  // namespace
}  // namespace gf
