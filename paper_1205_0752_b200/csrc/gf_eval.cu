// gf_eval.cu -- Step 5 / Kernel 2 of the paper: the double integral of
// eq. (14)/(15) for every grid point, as hand-written sm_100a CUDA.
//
// The sum that is computed:
//
//   G(x) = c0 sum_i Wr_i y_i D1(y_i) sum_j w'_j [ D2(u_ij) - D2(y_i) ],   u_ij = A_i - B_i z_j,
//   A_i = x + y_i,  B_i = 2 sqrt(x) sqrt(y_i)                                  eq. (10),(12),(20)
//
// How it is restructured for the FP64 pipe (none of this is in the paper):
//
//  * Line 2 is a sum of simple poles, D2(u) = sum_r R_r/(u + mu_r) (one term for 1/(u+m^2), two for the
//    rational propagator).  For one pole, with c = y + mu and A = x + c, a +-z pair of a symmetric
//    angular rule folds into
//        1/(A - Bz) + 1/(A + Bz) - 2/c = -(2/c) (eta - t)/(zeta - t),
//        t = z^2,  eta = A/(4y),  zeta = A^2/(4xy),
//    which needs no square root and has one real reciprocal per PAIR of angular nodes.
//  * (eta - t)/(zeta - t) = (eta - t)(conj(zeta) - t)/|zeta - t|^2, and the numerator is a quadratic
//    in t, so with q_j = w_j/|zeta - t_j|^2 only three REAL sums are accumulated in the inner loop,
//        U0 = sum q_j,  U1 = sum q_j t_j,  U2 = sum q_j t_j^2,
//    and  sum_j w_j (eta - t_j)/(zeta - t_j) = eta conj(zeta) U0 - (eta + conj(zeta)) U1 + U2.
//    Inner loop per pair: 9 FP64-pipe instructions (6 DFMA, 1 DMUL, 2 DADD) + 1 MUFU.RCP64H.
//    No difference of nearly equal numbers is formed: G(x) keeps full relative accuracy as x -> 0
//    (the paper's reason for the combined form of eq. (20)), and G(0) = 0 exactly.
//  * The reciprocal is MUFU.RCP64H (a ~2^-20.. seed) with one cubically convergent correction
//    r = r0 (1 + e + e^2), e = 1 - s r0 -- three DFMA, no slow-path branch.
//  * One thread owns one grid point (or 1/S of its radial nodes when the grid is too small to fill 148
//    SMs; the S lanes are merged with warp shuffles).  Tables are staged once per CTA in shared memory
//    and read as warp-wide broadcasts (LDS.128); results leave as coalesced 16-byte stores.
#include <cfloat>
#include <cmath>

#include "gf_internal.h"

namespace gf {
namespace {

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

// One folded angular pair: q = w/|zeta - t|^2 and the three moment sums.
__device__ __forceinline__ void pair_step(double zr, double zi2, double t, double t2, double w, double& u0,
                                          double& u1, double& u2) {
  const double a = zr - t;              // DADD
  const double s = fma(a, a, zi2);      // DFMA  |zeta - t|^2
  const double r0 = rcp_seed(s);        // MUFU.RCP64H
  const double e = fma(-s, r0, 1.0);    // DFMA
  const double p = fma(e, e, e);        // DFMA  e + e^2
  const double v = r0 * w;              // DMUL
  const double q = fma(v, p, v);        // DFMA  w/s (1 - e^3)
  u0 += q;                              // DADD
  u1 = fma(q, t, u1);                   // DFMA
  u2 = fma(q, t2, u2);                  // DFMA
}
__device__ __forceinline__ void pair_step(float zr, float zi2, float t, float t2, float w, float& u0, float& u1,
                                          float& u2) {
  const float a = zr - t;
  const float s = fmaf(a, a, zi2);
  const float q = w * rcp_seed(s);
  u0 += q;
  u1 = fmaf(q, t, u1);
  u2 = fmaf(q, t2, u2);
}

template <typename T>
struct Vec2;
template <>
struct Vec2<double> { typedef double2 type; };
template <>
struct Vec2<float> { typedef float2 type; };

// sum_j w_j (eta - t_j)/(zeta - t_j) over the folded angular rule, tables in shared memory.
// Two independent sets of accumulators (even / odd pairs): ILP for the FP64 pipe, and a shallower
// summation tree for the FP32 variant.
template <typename T>
__device__ __forceinline__ cd angular_sum(cd eta, cd zeta, const T* __restrict__ st, const T* __restrict__ st2,
                                          const T* __restrict__ sw, int n_pairs) {
  typedef typename Vec2<T>::type V2;
  const T zr = (T)zeta.re;
  const T zi2 = (T)(zeta.im * zeta.im);
  T a0 = 0, a1 = 0, a2 = 0, b0 = 0, b1 = 0, b2 = 0;
  int j = 0;
#pragma unroll 1
  for (; j + 4 <= n_pairs; j += 4) {
    const V2 t01 = *reinterpret_cast<const V2*>(st + j), t23 = *reinterpret_cast<const V2*>(st + j + 2);
    const V2 q01 = *reinterpret_cast<const V2*>(st2 + j), q23 = *reinterpret_cast<const V2*>(st2 + j + 2);
    const V2 w01 = *reinterpret_cast<const V2*>(sw + j), w23 = *reinterpret_cast<const V2*>(sw + j + 2);
    pair_step(zr, zi2, t01.x, q01.x, w01.x, a0, a1, a2);
    pair_step(zr, zi2, t01.y, q01.y, w01.y, b0, b1, b2);
    pair_step(zr, zi2, t23.x, q23.x, w23.x, a0, a1, a2);
    pair_step(zr, zi2, t23.y, q23.y, w23.y, b0, b1, b2);
  }
  for (; j < n_pairs; ++j) pair_step(zr, zi2, st[j], st2[j], sw[j], a0, a1, a2);
  const double u0 = (double)a0 + (double)b0, u1 = (double)a1 + (double)b1, u2 = (double)a2 + (double)b2;
  // eta conj(zeta) U0 - (eta + conj(zeta)) U1 + U2
  const double k6 = fma(eta.re, zeta.re, eta.im * zeta.im);
  const double k5 = fma(eta.im, zeta.re, -(eta.re * zeta.im));
  cd s;
  s.re = fma(k6, u0, fma(-(eta.re + zeta.re), u1, u2));
  s.im = fma(k5, u0, -(eta.im - zeta.im) * u1);
  return s;
}

// Shared-memory layout (doubles unless T = float for the angular tables).
struct SmemLayout {
  int off_t, off_t2, off_w;   // angular, in units of T, each n_pairs_pad long
  int off_y, off_q4;          // radial (REAL contour): y_i, 1/(4 y_i)
  int off_pref;               // double2 pref[n_terms][n_rad]
  int off_flag;               // int
  size_t bytes;
};

__host__ __device__ inline SmemLayout make_layout(int n_rad, int n_pairs, int n_terms, bool f32) {
  SmemLayout L;
  const int npad = (n_pairs + 3) & ~3;
  size_t b = 0;
  const size_t ts = f32 ? 4 : 8;
  L.off_t = 0;
  L.off_t2 = npad;
  L.off_w = 2 * npad;
  b = 3 * (size_t)npad * ts;
  b = (b + 15) & ~(size_t)15;
  L.off_y = (int)(b / 8);
  L.off_q4 = L.off_y + n_rad;
  b += 2 * (size_t)n_rad * 8;
  b = (b + 15) & ~(size_t)15;
  L.off_pref = (int)(b / 16);
  b += (size_t)n_terms * n_rad * 16;
  L.off_flag = (int)(b / 4);
  b += 16;
  L.bytes = b;
  return L;
}

// Stage the folded angular rule: pair j = nodes (j, n_ang-1-j); t = z^2, weight = w_j + w_mirror
// (the middle node of an odd rule enters once).  Returns through *flag whether the rule is symmetric.
template <typename T>
__device__ void stage_angular(const EvalArgs& a, T* st, T* st2, T* sw, int* flag) {
  const int npad = (a.n_pairs + 3) & ~3;
  for (int j = threadIdx.x; j < npad; j += blockDim.x) {
    double t = 0, w = 0;
    if (j < a.n_pairs) {
      const int jm = a.n_ang - 1 - j;
      const double zp = a.ang_nodes[jm], zm = a.ang_nodes[j];
      const double wp = a.ang_weights[jm], wm = a.ang_weights[j];
      const double tol = 16.0 * DBL_EPSILON;
      const bool ok = (jm == j) ? (fabs(zp) <= 1e-15)
                                : (fabs(zp + zm) <= tol * fabs(zp) && fabs(wp - wm) <= tol * fabs(wp));
      if (!ok) atomicExch(flag, 1);
      t = zp * zp;
      w = (jm == j) ? wp : wp + wm;
    }
    st[j] = (T)t;
    st2[j] = (T)(t * t);
    sw[j] = (T)w;
  }
}

// D1(y) for real y (REAL contour): massive 1/(y + m2) or rational (y + M2)/(y^2 + a y + b).
__device__ __forceinline__ cd line_k_real(const gf_propagator& p, double y) {
  if (p.kind == GF_PROP_MASSIVE) return cinv(cd{y + p.m2_re, p.m2_im});
  return cd{(y + p.M2) / fma(y, y + p.a, p.b), 0.0};
}

// ---------------------------------------------------------------------------------------------
// REAL contour for every point: the radial nodes do not depend on x, so y_i, 1/(4 y_i) and the
// per-node factor  pref_{r,i} = c0 Wr_i y_i D1(y_i) (-R_r/(y_i + mu_r))  are staged once per CTA.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(kBlockThreads, 2) eval_real_kernel(const __grid_constant__ EvalArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const SmemLayout L = make_layout(a.n_rad, a.n_pairs, a.n_terms, sizeof(T) == 4);
  T* st = reinterpret_cast<T*>(smem_raw) + L.off_t;
  T* st2 = reinterpret_cast<T*>(smem_raw) + L.off_t2;
  T* sw = reinterpret_cast<T*>(smem_raw) + L.off_w;
  double* sy = reinterpret_cast<double*>(smem_raw) + L.off_y;
  double* sq4 = reinterpret_cast<double*>(smem_raw) + L.off_q4;
  double2* spref = reinterpret_cast<double2*>(smem_raw) + L.off_pref;
  int* flag = reinterpret_cast<int*>(smem_raw) + L.off_flag;

  if (threadIdx.x == 0) *flag = 0;
  __syncthreads();
  stage_angular<T>(a, st, st2, sw, flag);
  {
    // shifted-log map of [0, Lambda^2]: y(u) = s0 expm1(u L), dy/du = L (y + s0)   (readings G3/G4)
    const double Llog = log1p(a.cutoff2 / a.s0);
    for (int i = threadIdx.x; i < a.n_rad; i += blockDim.x) {
      const double u = 0.5 * (a.rad_nodes[i] + 1.0);
      const double y = a.s0 * expm1(u * Llog);
      const double Wr = 0.5 * a.rad_weights[i] * Llog * (y + a.s0);
      sy[i] = y;
      sq4[i] = 0.25 / y;
      const cd d1 = cscale(line_k_real(a.line_k, y), a.c0 * Wr * y);
      for (int r = 0; r < a.n_terms; ++r) {
        const cd ic = cinv(cd{y + a.term[r].mu_re, a.term[r].mu_im});
        const cd pr = cmul(cmul(d1, cd{-a.term[r].R_re, -a.term[r].R_im}), ic);
        spref[r * a.n_rad + i] = make_double2(pr.re, pr.im);
      }
    }
  }
  __syncthreads();
  const bool bad_rule = *flag != 0;

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
  // exact to O(|x|) because the sum is analytic at 0 and vanishes there (keeps zeta = A^2/(4xy) and its
  // square inside the FP64 range).
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

  double g_re = 0.0, g_im = 0.0;
#pragma unroll 1
  for (int i = sub; i < a.n_rad; i += S) {
    const double y = sy[i], q4 = sq4[i];
#pragma unroll 1
    for (int r = 0; r < a.n_terms; ++r) {
      const cd A = {x.re + (y + a.term[r].mu_re), x.im + a.term[r].mu_im};
      const cd eta = cscale(A, q4);
      const cd zeta = cmul(cmul(eta, A), xinv);
      const cd s = angular_sum<T>(eta, zeta, st, st2, sw, a.n_pairs);
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
  plan->smem_bytes = make_layout(a.n_rad, a.n_pairs, a.n_terms, precision == 32).bytes;
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

template <typename T>
static int launch_real(const EvalArgs& a, const LaunchPlan& plan, cudaStream_t stream) {
  auto kern = eval_real_kernel<T>;
  if (plan.smem_bytes > 48 * 1024) {
    int rc = check_cuda(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes),
                        "cudaFuncSetAttribute(max dynamic shared memory)");
    if (rc) return rc;
  }
  kern<<<(unsigned)plan.grid_blocks, plan.block_threads, plan.smem_bytes, stream>>>(a);
  return check_cuda(cudaGetLastError(), "eval kernel launch");
}

int launch_eval(const EvalArgs& a_in, int precision, cudaStream_t stream) {
  if (a_in.n_points == 0) return GF_OK;
  LaunchPlan plan;
  int rc = plan_eval(a_in, precision, &plan);
  if (rc) return rc;
  EvalArgs a = a_in;
  a.split_log2 = plan.split_log2;
  if (plan.shared_nodes) return precision == 32 ? launch_real<float>(a, plan, stream) : launch_real<double>(a, plan, stream);
  set_error("eval_grid: contour %d is not implemented yet", a.contour);
  return GF_ERR_UNSUPPORTED;
}

// Executed floating-point instructions per launch, from the SASS of the loops above (DESIGN.md
// "Instruction counts"): per (point, radial node, pole term) the inner loop runs n_pairs times
// 6 DFMA + 1 DMUL + 2 DADD (FP64) or 3 FFMA + 1 FMUL + 2 FADD (FP32 variant), plus the set-up and
// finish of one angular sum.
void eval_inst_counts(const EvalArgs& a, int precision, const LaunchPlan& plan, double* fp64_inst,
                      double* fp32_inst, double* flops) {
  const double node_terms = (double)a.n_points * a.n_rad * a.n_terms;
  // per node-term outside the inner loop: A (2 DADD), eta (2 DMUL), zeta (2 cmul = 4 DMUL + 4 DFMA),
  // zi2 (1 DMUL), k5/k6 (2 DMUL + 2 DFMA), u sums (3 DADD), s (2 DADD + 1 DMUL + 3 DFMA), G (4 DFMA)
  const double setup_fma = 13, setup_other = 17;
  double i64 = node_terms * (setup_fma + setup_other), fl = node_terms * (2 * setup_fma + setup_other), i32 = 0;
  if (precision == 32) {
    i32 = node_terms * a.n_pairs * 6.0;
    fl += node_terms * a.n_pairs * (2 * 3.0 + 3.0);
  } else {
    i64 += node_terms * a.n_pairs * 9.0;
    fl += node_terms * a.n_pairs * (2 * 6.0 + 3.0);
  }
  (void)plan;
  *fp64_inst = i64;
  *fp32_inst = i32;
  *flops = fl;
}

}  // namespace gf
