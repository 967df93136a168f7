// gf_diag.cu -- diagnostics for bench.py: the measured FP64-pipe peak (the roofline denominator
// MEASURED_PEAKS.json does not carry) and the raw MUFU.RCP64H seed.  Not on the hot path.
#include "gf_internal.h"

namespace gf {
namespace {

// 8 independent DFMA chains per thread: 16 flops x 8 = 8 DFMA per inner round.
__global__ void __launch_bounds__(1024) fp64_peak_kernel(long long iters, double* __restrict__ sink) {
  const double m = 1.0 + 1e-9 * threadIdx.x, c = 1e-12;
  double a0 = 1.0, a1 = 1.1, a2 = 1.2, a3 = 1.3, a4 = 1.4, a5 = 1.5, a6 = 1.6, a7 = 1.7;
#pragma unroll 4
  for (long long k = 0; k < iters; ++k) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  sink[blockIdx.x * (long long)blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

__global__ void rcp_seed_kernel(const double* __restrict__ in, double* __restrict__ out, long long n) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(in[i]));
    out[i] = r;
  }
}

}  // namespace

int launch_fp64_peak(int blocks, int threads, long long iters, double* d_sink, cudaStream_t stream) {
  fp64_peak_kernel<<<blocks, threads, 0, stream>>>(iters, d_sink);
  return check_cuda(cudaGetLastError(), "fp64_peak launch");
}

int launch_rcp_seed(const double* d_in, double* d_out, long long n, cudaStream_t stream) {
  long long blocks = (n + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  if (blocks < 1) blocks = 1;
  rcp_seed_kernel<<<(unsigned)blocks, 256, 0, stream>>>(d_in, d_out, n);
  return check_cuda(cudaGetLastError(), "rcp_seed launch");
}

}  // namespace gf
