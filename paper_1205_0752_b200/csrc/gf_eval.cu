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
//    which needs no square root.  Per (point, radial node, pole) the angular sum
//        S = sum_j w_j (eta - t_j)/(zeta - t_j)          (w_j: folded weights)
//    is evaluated by one of three routes, chosen from zeta alone:
//      FAR    |zeta| >= 2 and few enough terms: the finite geometric series in omega = 1/zeta,
//             S = omega [ delta P(omega) + N(omega) ],  P = sum_k mu_k omega^k,  N = sum_k nu_k omega^k,
//             mu_k = sum_j w_j t_j^k,  nu_k = sum_j w_j t_j^k (1/4 - t_j)  (moments of the rule, made once
//             per launch).  K = ceil(58 / log2|zeta|) terms make the truncation < 2^-58.  Cancellation
//             free, O(K) instead of O(N_a).  Most radial nodes of a log-mapped rule are FAR.
//      NEAR   otherwise: q_j = w_j/|zeta - t_j|^2 by one real reciprocal per PAIR (MUFU.RCP64H seed + one
//             cubic correction, 3 DFMA, no slow path), two real sums U0 = sum q_j, U1 = sum q_j t_j, and
//             S = mu_0 - (zeta - eta)(conj(zeta) U0 - U1).  8 FP64 instructions per pair.  Its
//             cancellation grows like |zeta|^2, which FAR bounds.
//      EXACT  zeta within 2^-8 of the segment [0,1] (the radial contour passes next to a zero of a
//             denominator): zeta is recomputed in double-double and each term is formed directly with
//             a = (zeta_hi - t_hi) + (zeta_lo - t_lo), t_hi + t_lo = z^2 exactly.  Rare (a few nodes per
//             point outside the parabola where REAL is the continuation), so its cost does not matter;
//             without it such terms carry an error eps/dist (reading G18).
//  * x = 0 gives exactly 0 (invariant I1); 0 < |x| < 2^-200 is rescaled (the sum is analytic at 0).
//  * A one-CTA preparation kernel makes every x-independent table once per launch (folded angular rule,
//    moments, the radial map y_i in double-double so that it is correctly rounded, per-node prefactors);
//    each CTA of the evaluation kernel pulls that block into shared memory with ONE bulk copy
//    (cp.async.bulk + mbarrier, the 1-D TMA path) and reads it as warp-wide broadcasts.
//  * One thread owns one grid point (or 1/S of its radial nodes when the grid is too small to fill 148
//    SMs; the S lanes are merged with warp shuffles); results leave as coalesced 16-byte stores.
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

// EXACT: zeta = A^2/(4 x y) in double-double, A = x + y + mu; every term formed directly.
__device__ __noinline__ cd angular_exact(double xr, double xi, double y, double mur, double mui, cd eta,
                                         const double* __restrict__ st, const double* __restrict__ stlo,
                                         const double* __restrict__ sw, int n_pairs) {
  const dd Ar = dd_add_d(two_sum(xr, mur), y), Ai = two_sum(xi, mui);
  const dd A2r = dd_add(dd_mul(Ar, Ar), dd_neg(dd_mul(Ai, Ai)));
  const dd A2i = dd_scale2(dd_mul(Ar, Ai), 2.0);
  // zeta = A^2 conj(x) / (4 y |x|^2)
  const dd nr = dd_add(dd_mul_d(A2r, xr), dd_mul_d(A2i, xi));
  const dd ni = dd_add(dd_mul_d(A2i, xr), dd_neg(dd_mul_d(A2r, xi)));
  const dd den = dd_scale2(dd_mul_d(dd_add(two_prod(xr, xr), two_prod(xi, xi)), y), 4.0);
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

__global__ void radial_map_kernel(double Lhi, double Llo, double s0, const double* __restrict__ nodes, int n,
                                  double* __restrict__ y) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) y[i] = radial_node(nodes[i], dd{Lhi, Llo}, s0);
}

// ---------------------------------------------------------------------------------------------
// Preparation (one CTA): everything that does not depend on x, for the REAL contour.
//   header [0] = 1.0 if the angular rule is not symmetric;  t, t_lo, w (folded rule);
//   mu_k, nu_k (moments);  y_i, 1/(4 y_i);  pref_{r,i} = c0 Wr_i y_i D1(y_i) (-R_r/(y_i + mu_r)).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) prep_real_kernel(const __grid_constant__ EvalArgs a,
                                                        const __grid_constant__ BlobLayout L,
                                                        double* __restrict__ blob) {
  __shared__ int bad;
  if (threadIdx.x == 0) bad = 0;
  __syncthreads();
  prep_angular(a, L, blob, &bad);
  {
    // shifted-log map of [0, Lambda^2] (readings G3/G4): y(u) = s0 expm1(u L), dy/du = L (y + s0),
    // L = ln((Lambda^2 + s0)/s0) as a double-double from the host; y_i correctly rounded.
    const dd Llog = {a.Llog_hi, a.Llog_lo};
    for (int i = threadIdx.x; i < a.n_rad; i += blockDim.x) {
      const double y = radial_node(a.rad_nodes[i], Llog, a.s0);
      const double Wr = 0.5 * a.rad_weights[i] * a.Llog_hi * (y + a.s0);
      blob[L.off_y + i] = y;
      blob[L.off_q4 + i] = 0.25 / y;
      const cd d1 = cscale(line_k_real(a.line_k, y), a.c0 * Wr * y);
      for (int r = 0; r < a.n_terms; ++r) {
        const cd ic = cinv(cd{y + a.term[r].mu_re, a.term[r].mu_im});
        const cd pr = cmul(cmul(d1, cd{-a.term[r].R_re, -a.term[r].R_im}), ic);
        blob[L.off_pref + 2 * (r * a.n_rad + i)] = pr.re;
        blob[L.off_pref + 2 * (r * a.n_rad + i) + 1] = pr.im;
      }
    }
  }
  __syncthreads();  // t, w written by this CTA are visible to it
  for (int k = threadIdx.x; k < L.km; k += blockDim.x) {
    dd mu = {0.0, 0.0}, nu = {0.0, 0.0};
    for (int j = 0; j < a.n_pairs; ++j) {
      const double t = blob[L.off_t + j], wp = blob[L.off_w + j] * powi(t, k);
      mu = dd_add_d(mu, wp);
      nu = dd_add(nu, two_prod(wp, 0.25 - t));
    }
    blob[L.off_mu + k] = mu.hi;
    blob[L.off_nu + k] = nu.hi;
  }
  if (threadIdx.x == 0) {
    blob[0] = bad ? 1.0 : 0.0;
    blob[1] = 0.0;
  }
}

// ---------------------------------------------------------------------------------------------
// Evaluation, REAL contour.  counters (COUNT only): [0] NEAR pairs, [1] FAR terms, [2] EXACT pairs,
// [3] NEAR node-terms, [4] FAR node-terms, [5] EXACT node-terms.
// ---------------------------------------------------------------------------------------------
template <typename T, bool COUNT>
__global__ void __launch_bounds__(kBlockThreads, 2)
    eval_real_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                     const double* __restrict__ blob, unsigned long long* __restrict__ counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
  double* sb = reinterpret_cast<double*>(smem_raw + 16);
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) bulk_load(sb, blob, (uint32_t)(L.n_doubles * sizeof(double)), bar);
  mbar_wait(bar, 0);

  const double* st = sb + L.off_t;
  const double* stlo = sb + L.off_tlo;
  const double* sw = sb + L.off_w;
  const double* smu = sb + L.off_mu;
  const double* snu = sb + L.off_nu;
  const double* sy = sb + L.off_y;
  const double* sq4 = sb + L.off_q4;
  const double2* spref = reinterpret_cast<const double2*>(sb + L.off_pref);
  const T* stT = sizeof(T) == 8 ? reinterpret_cast<const T*>(st) : reinterpret_cast<const T*>(sb + L.off_f32);
  const T* swT = sizeof(T) == 8 ? reinterpret_cast<const T*>(sw) : stT + L.npad;
  const bool bad_rule = sb[0] != 0.0;
  const double mu0 = smu[0];
  const double tau = sizeof(T) == 8 ? kTau64 : kTau32;

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

  unsigned long long c_near = 0, c_far = 0, c_exact = 0, n_near = 0, n_far = 0, n_exact = 0;
  double g_re = 0.0, g_im = 0.0;
#pragma unroll 1
  for (int i = sub; i < a.n_rad; i += S) {
    const double y = sy[i], q4 = sq4[i];
#pragma unroll 1
    for (int r = 0; r < a.n_terms; ++r) {
      const double mur = a.term[r].mu_re, mui = a.term[r].mu_im;
      const cd xm = {x.re + mur, x.im + mui};
      const cd A = {xm.re + y, xm.im};
      const cd delta = cscale(xm, q4);               // eta - 1/4
      const cd eta = {0.25 + delta.re, delta.im};
      const cd zeta = cmul(cmul(eta, A), xinv);
      // 2 ilogb(max component) <= log2 |zeta|^2
      const int e2 = 2 * ilogb(fmax(fabs(zeta.re), fabs(zeta.im)));
      const int K = e2 >= 2 ? (e2 >= kFarBits ? 2 : kFarBits / e2 + 1) : 0x7fffffff;
      cd s;
      if (K <= L.km && (K <= a.n_pairs || e2 > 6)) {
        s = angular_far(delta, zeta, K, smu, snu);
        if (COUNT) { c_far += K; ++n_far; }
      } else if (zeta.im * zeta.im < tau * tau && zeta.re > -tau && zeta.re < 1.0 + tau) {
        s = angular_exact(x.re, x.im, y, mur, mui, eta, st, stlo, sw, a.n_pairs);
        if (COUNT) { c_exact += a.n_pairs; ++n_exact; }
      } else {
        s = angular_near<T>(eta, zeta, mu0, stT, swT, a.n_pairs);
        if (COUNT) { c_near += a.n_pairs; ++n_near; }
      }
      const double2 pr = spref[r * a.n_rad + i];
      g_re = fma(pr.x, s.re, fma(-pr.y, s.im, g_re));
      g_im = fma(pr.x, s.im, fma(pr.y, s.re, g_im));
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
  if (COUNT) {
    if (!active) c_near = c_far = c_exact = n_near = n_far = n_exact = 0;
    unsigned long long v[6] = {c_near, c_far, c_exact, n_near, n_far, n_exact};
    for (int k = 0; k < 6; ++k) {
      for (int o = 16; o; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
      if ((threadIdx.x & 31) == 0 && v[k]) atomicAdd(counters + k, v[k]);
    }
  }
}

BlobLayout make_layout(int n_rad, int n_pairs, int n_terms, bool f32) {
  BlobLayout L;
  L.npad = (n_pairs + 3) & ~3;
  L.km = kKmCap;
  int o = 2;  // header
  auto take = [&](int n) { int at = o; o += (n + 1) & ~1; return at; };
  L.off_t = take(L.npad);
  L.off_tlo = take(L.npad);
  L.off_w = take(L.npad);
  L.off_mu = take(L.km);
  L.off_nu = take(L.km);
  L.off_y = take(n_rad);
  L.off_q4 = take(n_rad);
  L.off_pref = take(2 * n_terms * n_rad);
  L.off_f32 = f32 ? take(L.npad) : -1;  // 2 float tables of npad entries = npad doubles
  L.n_doubles = o;
  return L;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
int plan_eval(const EvalArgs& a, int precision, LaunchPlan* plan) {
  plan->block_threads = kBlockThreads;
  plan->shared_nodes = (a.contour == GF_CONTOUR_REAL);
  // lanes per point: enough threads for >= 2 CTAs on each of the 148 SMs, at most a warp
  int sl = 0;
  const long long want = 148LL * 2 * kBlockThreads;
  while (sl < 5 && (a.n_points << sl) < want && (2 << sl) <= a.n_rad) ++sl;
  plan->split_log2 = sl;
  const long long threads = a.n_points << sl;
  plan->grid_blocks = (threads + kBlockThreads - 1) / kBlockThreads;
  plan->layout = make_layout(a.n_rad, a.n_pairs, a.n_terms, precision == 32);
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

template <typename T, bool COUNT>
static int launch_real(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* counters,
                       cudaStream_t stream) {
  auto kern = eval_real_kernel<T, COUNT>;
  if (plan.smem_bytes > 48 * 1024) {
    int rc = check_cuda(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes),
                        "cudaFuncSetAttribute(max dynamic shared memory)");
    if (rc) return rc;
  }
  kern<<<(unsigned)plan.grid_blocks, plan.block_threads, plan.smem_bytes, stream>>>(a, plan.layout, blob, counters);
  return check_cuda(cudaGetLastError(), "eval kernel launch");
}

int launch_radial_map(double Llog_hi, double Llog_lo, double s0, const double* d_nodes, int n, double* d_y,
                      cudaStream_t stream) {
  radial_map_kernel<<<(n + 127) / 128, 128, 0, stream>>>(Llog_hi, Llog_lo, s0, d_nodes, n, d_y);
  return check_cuda(cudaGetLastError(), "radial_map launch");
}

int launch_eval(const EvalArgs& a_in, int precision, unsigned long long* d_counters, cudaStream_t stream) {
  if (a_in.n_points == 0) return GF_OK;
  LaunchPlan plan;
  int rc = plan_eval(a_in, precision, &plan);
  if (rc) return rc;
  if (!plan.shared_nodes) {
    set_error("eval_grid: contour %d is not implemented yet", a_in.contour);
    return GF_ERR_UNSUPPORTED;
  }
  EvalArgs a = a_in;
  a.split_log2 = plan.split_log2;
  // scratch for the prepared tables: stream-ordered, freed in stream order after the evaluation
  double* blob = nullptr;
  rc = check_cuda(cudaMallocAsync(reinterpret_cast<void**>(&blob), (size_t)plan.layout.n_doubles * sizeof(double), stream),
                  "cudaMallocAsync(tables)");
  if (rc) return rc;
  prep_real_kernel<<<1, 256, 0, stream>>>(a, plan.layout, blob);
  rc = check_cuda(cudaGetLastError(), "prep kernel launch");
  if (!rc) {
    if (d_counters)
      rc = precision == 32 ? launch_real<float, true>(a, plan, blob, d_counters, stream)
                           : launch_real<double, true>(a, plan, blob, d_counters, stream);
    else
      rc = precision == 32 ? launch_real<float, false>(a, plan, blob, nullptr, stream)
                           : launch_real<double, false>(a, plan, blob, nullptr, stream);
  }
  cudaFreeAsync(blob, stream);
  return rc;
}

}  // namespace gf
