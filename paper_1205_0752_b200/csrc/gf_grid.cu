// gf_grid.cu -- Step 4 / Kernel 1 of the paper: discretise the region of
// evaluation.  One thread per grid point writes one complex<double> (a 16-byte store, coalesced
// along the real index).  HBM-bound and tiny: 16 B per point.
#include <cmath>
#include <vector>

#include "gf_internal.h"

namespace gf {
namespace {

// endpoint-inclusive, two-sided: exact mirror for ranges symmetric about 0 (reading G9)
__device__ __forceinline__ double axis_value(double lo, double hi, double d, int n, int i) {
  if (n == 1) return lo;
  if (2 * i <= n - 1) return fma((double)i, d, lo);
  return fma(-(double)(n - 1 - i), d, hi);
}

// im_half: for GF_SPACING_LOG_ABS_IM the n_im/2 ascending values of |Im x| (host-generated, so that
// the grid does not depend on the device's exp()); nullptr for uniform spacing.
__global__ void __launch_bounds__(256) make_grid_kernel(double re_min, double re_max, double d_re, int n_re,
                                                        double im_min, double im_max, double d_im, int n_im,
                                                        const double* __restrict__ im_half, int row_first,
                                                        int n_rows, double2* __restrict__ x) {
  const long long total = (long long)n_re * n_rows;
  for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < total;
       p += (long long)gridDim.x * blockDim.x) {
    const int jl = (int)(p / n_re), i = (int)(p - (long long)jl * n_re);
    const int j = row_first + jl;  // row of the global grid
    double im;
    if (im_half == nullptr) {
      im = axis_value(im_min, im_max, d_im, n_im, j);
    } else {
      // |Im x| log-spaced on each side of the real axis, ascending Im x (reading G10)
      const int half = n_im / 2;
      im = j >= half ? im_half[j - half] : -im_half[half - 1 - j];
    }
    x[p] = make_double2(axis_value(re_min, re_max, d_re, n_re, i), im);
  }
}

}  // namespace

int launch_make_grid(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
                     int spacing, double im_abs_min, int row_first, int n_rows, double2* d_x,
                     cudaStream_t stream) {
  const long long total = (long long)n_re * n_rows;
  if (total == 0) return GF_OK;
  const double d_re = n_re > 1 ? (re_max - re_min) / (double)(n_re - 1) : 0.0;
  const double d_im = n_im > 1 ? (im_max - im_min) / (double)(n_im - 1) : 0.0;
  double* d_half = nullptr;
  if (spacing == GF_SPACING_LOG_ABS_IM) {
    const int half = n_im / 2;
    std::vector<double> v(half);
    const double l0 = std::log(im_abs_min), l1 = std::log(im_max);
    for (int k = 0; k < half; ++k)
      v[k] = k == 0 ? im_abs_min : k == half - 1 ? im_max : std::exp(std::fma((double)k / (double)(half - 1), l1 - l0, l0));
    int rc = check_cuda(cudaMallocAsync(reinterpret_cast<void**>(&d_half), sizeof(double) * half, stream),
                        "cudaMallocAsync(im table)");
    if (rc) return rc;
    // pageable source: staged before the call returns, so v may go out of scope
    rc = check_cuda(cudaMemcpyAsync(d_half, v.data(), sizeof(double) * half, cudaMemcpyHostToDevice, stream),
                    "copy im table");
    if (rc) { cudaFreeAsync(d_half, stream); return rc; }
  }
  long long blocks = (total + 255) / 256;
  if (blocks > 148LL * 16) blocks = 148LL * 16;  // grid-stride: 16 CTAs per SM
  make_grid_kernel<<<(unsigned)blocks, 256, 0, stream>>>(re_min, re_max, d_re, n_re, im_min, im_max, d_im, n_im,
                                                         d_half, row_first, n_rows, d_x);
  int rc = check_cuda(cudaGetLastError(), "make_grid launch");
  if (d_half) cudaFreeAsync(d_half, stream);
  return rc;
}

}  // namespace gf
