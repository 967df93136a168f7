// gf_diag.cu -- diagnostics for bench.py: the measured FP64-pipe peak (the roofline denominator
// MEASURED_PEAKS.json does not carry) and the issue cadence of DFMA streams by the number of distinct
// register operands.  Not on the hot path.
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

// DFMA issue cadence.  Every mode runs 8 independent chains per thread, 8 DFMA per round and chain-step, so the
// dependent-issue latency is covered and only the operand traffic differs:
//   0  a_j = fma(a_j, m, c)        one varying register pair per instruction (m, c loop-invariant)
//   1  a_j = fma(a_j, b_j, c)      two varying pairs
//   2  a_j = fma(a_j, b_j, c_j)    three varying pairs: what a recurrence with its own multiplier, state and
//                                  coefficient issues
//   3  the second-order (Goertzel) recurrence of the series routes with coefficients in registers, four chains
//      (two nodes x two polynomials): t = fma(ns, p2, c); p2 = fma(r, p1, t)  -- 8 DFMA per round as well
template <int MODE>
__global__ void __launch_bounds__(1024) dfma_issue_kernel(long long iters, double* __restrict__ sink) {
  const double m = 1.0 + 1e-9 * threadIdx.x, c = 1e-12;
  double a[8], b[8], cc[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    a[j] = 1.0 + 0.1 * j;
    b[j] = 1.0 + 1e-9 * (threadIdx.x + 3 * j);
    cc[j] = 1e-12 * (1 + j + threadIdx.x);
  }
  if (MODE == 3) {
    const double r0 = 0.3 + 1e-6 * threadIdx.x, q0 = -0.05 - 1e-7 * threadIdx.x, r1 = 1.01 * r0, q1 = 0.99 * q0;
    double p1 = 0, p2 = 0, n1 = 0, n2 = 0, u1 = 0, u2 = 0, v1 = 0, v2 = 0;
    // four terms per trip with four different coefficient pairs, as the series loop sees them (the roles of
    // (p1, p2) alternate from term to term, as in goertzel_pair)
#pragma unroll 1
    for (long long k = 0; k < iters; k += 4) {
#pragma unroll
      for (int t = 0; t < 4; t += 2) {
        p2 = fma(r0, p1, fma(q0, p2, cc[2 * t])); n2 = fma(r0, n1, fma(q0, n2, cc[2 * t + 1]));
        u2 = fma(r1, u1, fma(q1, u2, cc[2 * t])); v2 = fma(r1, v1, fma(q1, v2, cc[2 * t + 1]));
        p1 = fma(r0, p2, fma(q0, p1, cc[2 * t + 2])); n1 = fma(r0, n2, fma(q0, n1, cc[2 * t + 3]));
        u1 = fma(r1, u2, fma(q1, u1, cc[2 * t + 2])); v1 = fma(r1, v2, fma(q1, v1, cc[2 * t + 3]));
      }
    }
    a[0] = p1 + p2; a[1] = n1 + n2; a[2] = u1 + u2; a[3] = v1 + v2;
  } else {
#pragma unroll 4
    for (long long k = 0; k < iters; ++k) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = MODE == 0 ? fma(a[j], m, c) : MODE == 1 ? fma(a[j], b[j], c) : fma(a[j], b[j], cc[j]);
    }
  }
  sink[blockIdx.x * (long long)blockDim.x + threadIdx.x] = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
}

}  // namespace

int launch_fp64_peak(int blocks, int threads, long long iters, double* d_sink, cudaStream_t stream) {
  fp64_peak_kernel<<<blocks, threads, 0, stream>>>(iters, d_sink);
  return check_cuda(cudaGetLastError(), "fp64_peak launch");
}

int launch_dfma_issue(int mode, int blocks, int threads, long long iters, double* d_sink, cudaStream_t stream) {
  switch (mode) {
    case 0: dfma_issue_kernel<0><<<blocks, threads, 0, stream>>>(iters, d_sink); break;
    case 1: dfma_issue_kernel<1><<<blocks, threads, 0, stream>>>(iters, d_sink); break;
    case 2: dfma_issue_kernel<2><<<blocks, threads, 0, stream>>>(iters, d_sink); break;
    default: dfma_issue_kernel<3><<<blocks, threads, 0, stream>>>(iters, d_sink); break;
  }
  return check_cuda(cudaGetLastError(), "dfma_issue launch");
}

}  // namespace gf
