// gf_cut.cu -- the two auxiliary kernels of the paper's Step 3:
//
//   Kernel 3  the angular integral B of eq. (22) for ONE x over an array of complex y (the density plots of
//             Fig. 1):  B(x, y) = sum_j w'_j [ D2(u_j) - D2(y) ] / D2(y),  u_j = x + y - 2 sqrt(x) sqrt(y) z_j.
//             One thread per y; the sum over j is the same folded sum S(delta, zeta) as in the scan and goes
//             through the same routes (gf_routes.cuh, node_term), with complex y:
//             sum_j w'_j [1/(u_j + mu) - 1/(y + mu)] = -S/(y + mu) per pole.
//   Kernel 4  how often the branch cut of the angular integral, eq. (25), crosses the original contour
//             (0, Lambda^2] of the real y-axis, per grid point x (Fig. 2: where it is 0 the contour "remains
//             unharmed").  The paper does not say how its kernel decides; reading G19 fixes the
//             procedure, every step a correctly rounded +, -, *, / or sqrt in a stated order (the _rn
//             intrinsics below), so that the integer result is the same as the oracle's bit for bit.
#include "gf_routes.cuh"

namespace gf {
namespace {

// ---------------------------------------------------------------------------------------------
// Kernel 3
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) prep_angular_only_kernel(const __grid_constant__ EvalArgs a,
                                                                const __grid_constant__ BlobLayout L,
                                                                double* __restrict__ blob) {
  __shared__ int bad;
  __shared__ float s_lc[kKmc];
  __shared__ dd s_cpart[8][2][kMomTerms];
  if (threadIdx.x == 0) bad = 0;
  __syncthreads();
  prep_angular(a, L, blob, &bad);
  __syncthreads();
  prep_blocks_T(a, L, blob);
  prep_series_T(a, L, blob);
  __syncthreads();
  prep_blocks_sums(a, L, blob);
  prep_series_sums(a, L, blob, s_cpart);
  __syncthreads();
  prep_series_kreq(L, blob, s_lc, blob + L.off_cheb, 2);
  if (threadIdx.x == 0) {
    blob[0] = (double)bad;
    blob[1] = a.ws_tag;
    if (bad) report_status(a.status, bad);
  }
}

__global__ void __launch_bounds__(kBlockThreads, 2)
    angular_kernel(const __grid_constant__ EvalArgs a, const __grid_constant__ BlobLayout L,
                   const double* __restrict__ blob, cd x) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);
  double* sb = reinterpret_cast<double*>(smem_raw + 16);
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) bulk_load(sb, blob, (uint32_t)(L.n_doubles * sizeof(double)), bar);
  mbar_wait(bar, 0);
  const Tabs<double> tb = make_tabs<double>(sb, L, a.n_pairs);
  const bool bad_rule = sb[0] != 0.0;

  const long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  const bool active = idx < a.n_points;
  cd y = {1.0, 0.0};
  if (active) {
    const double2 yv = a.x[idx];   // the array of y
    y = {yv.x, yv.y};
  }
  const bool y_zero = y.re == 0.0 && y.im == 0.0;
  if (y_zero) y = {1.0, 0.0};
  const cd xinv = cinv(x);
  const cd q4 = cscale(cinv(y), 0.25);
  const cd xq = cmul(xinv, q4);                       // 1/(4 x y)
  RouteCount rc;
  cd num = {0.0, 0.0}, d2y = {0.0, 0.0}, d2x = {0.0, 0.0};
#pragma unroll 1
  for (int r = 0; r < a.n_terms; ++r) {               // node_term is warp-collective: every lane takes every trip
    const double mur = a.term[r].mu_re, mui = a.term[r].mu_im;
    const cd R = {a.term[r].R_re, a.term[r].R_im};
    const cd xm = {x.re + mur, x.im + mui};
    const cd A = {xm.re + y.re, xm.im + y.im};
    const cd delta = cmul(xm, q4);
    const cd zeta = cmul(csqr(A), xq);
    const cd s = node_term<double, false>(tb, x, y, delta, zeta, mur, mui, rc);
    const cd ic = cinv(cd{y.re + mur, y.im + mui});   // R_r/(y + mu_r)
    const cd Ric = cmul(R, ic);
    num = cadd(num, cmul(Ric, cd{-s.re, -s.im}));     // sum_j w'_j [D2(u_j) - D2(y)], this pole
    d2y = cadd(d2y, Ric);
    d2x = cadd(d2x, cmul(R, cinv(xm)));               // D2(x), used at y = 0
  }
  cd B = cmul(num, cinv(d2y));
  if (y_zero) {
    // u_j = x for every j: B = (sum_j w'_j) (D2(x)/D2(0) - 1)
    cd d20 = {0.0, 0.0};
    for (int r = 0; r < a.n_terms; ++r)
      d20 = cadd(d20, cmul(cd{a.term[r].R_re, a.term[r].R_im}, cinv(cd{a.term[r].mu_re, a.term[r].mu_im})));
    const cd q = cmul(d2x, cinv(d20));
    B = {tb.mu0 * (q.re - 1.0), tb.mu0 * q.im};
  }
  if (bad_rule) B = {nan(""), nan("")};
  if (active) reinterpret_cast<double2*>(a.out)[idx] = make_double2(B.re, B.im);
}

// ---------------------------------------------------------------------------------------------
// Kernel 4
// ---------------------------------------------------------------------------------------------
struct C2 { double re, im; };
// principal square root from real operations only (the same sequence as the oracle's csqrt_rn)
__device__ __forceinline__ C2 csqrt_rn(C2 v) {
  const double m = __dsqrt_rn(__dadd_rn(__dmul_rn(v.re, v.re), __dmul_rn(v.im, v.im)));
  const double h = __dsqrt_rn(__dmul_rn(0.5, __dadd_rn(m, fabs(v.re))));
  if (h == 0.0) return C2{0.0, 0.0};
  const double k = __ddiv_rn(v.im, __dmul_rn(2.0, h));
  if (v.re >= 0.0) return C2{h, k};
  return C2{fabs(k), copysign(h, v.im)};
}
__device__ int cut_crossings_one(C2 x, C2 mu, double cutoff2, int n_z) {
  const C2 sx = csqrt_rn(x);
  int count = 0;
  C2 sprev = {0.0, 0.0};
  double yre_prev = 0.0, yim_prev = 0.0;
  const double nm1 = (double)(n_z - 1);
  for (int k = 0; k < n_z; ++k) {
    const double z = __dadd_rn(-1.0, __ddiv_rn(__dmul_rn(2.0, (double)k), nm1));
    const double omz2 = __dmul_rn(__dadd_rn(1.0, -z), __dadd_rn(1.0, z));
    C2 s = csqrt_rn(C2{__dadd_rn(__dmul_rn(x.re, omz2), mu.re), __dadd_rn(__dmul_rn(x.im, omz2), mu.im)});
    if (k > 0 && __dadd_rn(__dmul_rn(s.re, sprev.re), __dmul_rn(s.im, sprev.im)) < 0.0) { s.re = -s.re; s.im = -s.im; }
    const double kre = __dadd_rn(__dmul_rn(sx.re, z), -s.im), kim = __dadd_rn(__dmul_rn(sx.im, z), s.re);
    const double yre = __dadd_rn(__dmul_rn(kre, kre), -__dmul_rn(kim, kim)), yim = __dmul_rn(2.0, __dmul_rn(kre, kim));
    if (k > 0) {
      const bool cross = (yim_prev < 0.0 && yim >= 0.0) || (yim_prev > 0.0 && yim <= 0.0);
      if (cross) {
        const double t = __ddiv_rn(yim_prev, __dadd_rn(yim_prev, -yim));
        const double re0 = __dadd_rn(yre_prev, __dmul_rn(t, __dadd_rn(yre, -yre_prev)));
        if (re0 > 0.0 && re0 <= cutoff2) ++count;
      }
    }
    sprev = s;
    yre_prev = yre;
    yim_prev = yim;
  }
  return count;
}
__global__ void __launch_bounds__(256) cut_crossings_kernel(const __grid_constant__ EvalArgs a, int n_z,
                                                            int* __restrict__ out) {
  const long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= a.n_points) return;
  const double2 xv = a.x[idx];
  int count = 0;
  for (int r = 0; r < a.n_terms; ++r)
    count += cut_crossings_one(C2{xv.x, xv.y}, C2{a.term[r].mu_re, a.term[r].mu_im}, a.cutoff2, n_z);
  out[idx] = count;
}

}  // namespace

int launch_angular(const EvalArgs& a_in, double x_re, double x_im, cudaStream_t stream) {
  if (a_in.n_points == 0) return GF_OK;
  if (x_re == 0.0 && x_im == 0.0)   // the factor d of eq. (20) vanishes identically: B = 0 exactly
    return check_cuda(cudaMemsetAsync(a_in.out, 0, (size_t)a_in.n_points * 16, stream), "cudaMemsetAsync");
  EvalArgs a = a_in;
  a.n_rad = 0;
  const BlobLayout L = make_blob_layout(0, a.n_pairs, a.n_terms, false, false, false);
  const size_t smem = 16 + (size_t)L.n_doubles * sizeof(double);
  if (smem > 200 * 1024) { set_error("eval_angular: n_ang too large for shared memory"); return GF_ERR_ARG; }
  double* blob = nullptr;
  int rc = scratch_alloc(reinterpret_cast<void**>(&blob), (size_t)L.n_total * sizeof(double), stream);
  if (rc) return rc;
  prep_angular_only_kernel<<<1, 256, 0, stream>>>(a, L, blob);
  rc = check_cuda(cudaGetLastError(), "prep kernel launch");
  if (!rc && smem > 48 * 1024)
    rc = check_cuda(cudaFuncSetAttribute(angular_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                    "cudaFuncSetAttribute(max dynamic shared memory)");
  if (!rc) {
    const long long blocks = (a.n_points + kBlockThreads - 1) / kBlockThreads;
    angular_kernel<<<(unsigned)blocks, kBlockThreads, smem, stream>>>(a, L, blob, cd{x_re, x_im});
    rc = check_cuda(cudaGetLastError(), "angular kernel launch");
  }
  cudaFreeAsync(blob, stream);
  return rc;
}

int launch_cut_crossings(const EvalArgs& a, int n_z, int* d_out, cudaStream_t stream) {
  if (a.n_points == 0) return GF_OK;
  const long long blocks = (a.n_points + 255) / 256;
  cut_crossings_kernel<<<(unsigned)blocks, 256, 0, stream>>>(a, n_z, d_out);
  return check_cuda(cudaGetLastError(), "cut_crossings kernel launch");
}

}  // namespace gf
