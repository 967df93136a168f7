// gf_grid.cu -- Step 4 / Kernel 1 of the paper: discretise the region of
// evaluation.  One thread per grid point writes one complex<double> (a 16-byte store, coalesced
// along the real index).  HBM-bound and tiny: 16 B per point.
#include "gf_internal.h"

namespace gf {
namespace {

// endpoint-inclusive, two-sided: exact mirror for ranges symmetric about 0 (reading G9)
__device__ __forceinline__ double axis_value(double lo, double hi, double d, int n, int i) {
  if (n == 1) return lo;
  if (2 * i <= n - 1) return fma((double)i, d, lo);
  return fma(-(double)(n - 1 - i), d, hi);
}

__global__ void __launch_bounds__(256) make_grid_kernel(double re_min, double re_max, double d_re, int n_re,
                                                        double im_min, double im_max, double d_im, int n_im,
                                                        int spacing, double log_lo, double log_hi,
                                                        double im_abs_min, int row_first, int n_rows,
                                                        double2* __restrict__ x) {
  const long long total = (long long)n_re * n_rows;
  for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < total;
       p += (long long)gridDim.x * blockDim.x) {
    const int jl = (int)(p / n_re), i = (int)(p - (long long)jl * n_re);
    const int j = row_first + jl;  // row of the global grid
    double im;
    if (spacing == GF_SPACING_UNIFORM) {
      im = axis_value(im_min, im_max, d_im, n_im, j);
    } else {
      // |Im x| log-spaced on each side of the real axis, ascending Im x (reading G10)
      const int half = n_im / 2;
      const int k = j >= half ? j - half : half - 1 - j;
      double v;
      if (k == 0) v = im_abs_min;
      else if (k == half - 1) v = im_max;
      else v = exp(fma((double)k / (double)(half - 1), log_hi - log_lo, log_lo));
      im = j >= half ? v : -v;
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
  double log_lo = 0, log_hi = 0;
  if (spacing == GF_SPACING_LOG_ABS_IM) {
    log_lo = log(im_abs_min);
    log_hi = log(im_max);
  }
  long long blocks = (total + 255) / 256;
  if (blocks > 148LL * 16) blocks = 148LL * 16;  // grid-stride: 16 CTAs per SM
  make_grid_kernel<<<(unsigned)blocks, 256, 0, stream>>>(re_min, re_max, d_re, n_re, im_min, im_max, d_im, n_im,
                                                         spacing, log_lo, log_hi, im_abs_min, row_first, n_rows, d_x);
  return check_cuda(cudaGetLastError(), "make_grid launch");
}

}  // namespace gf
