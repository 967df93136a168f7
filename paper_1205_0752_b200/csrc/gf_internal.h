// gf_internal.h -- declarations shared by the translation units of libgf_b200 (CUDA path only;
// the CPU oracle under oracle/ includes nothing from here).
#pragma once
#include <cuda_runtime.h>

#include "gf.h"

namespace gf {

// D2(u) = sum_r R_r / (u + mu_r): one term for a massive line, two for a rational line
// (partial fractions of (u+M2)/(u^2+au+b)).
struct PoleTerm {
  double R_re, R_im;
  double mu_re, mu_im;
};

constexpr int kMaxTerms = 2;
constexpr int kBlockThreads = 256;

// Everything the evaluation kernel needs, passed by value as a __grid_constant__.
struct EvalArgs {
  const double* rad_nodes;
  const double* rad_weights;
  const double* ang_nodes;
  const double* ang_weights;
  const double2* x;
  void* out;
  long long n_points;
  int n_rad, n_ang, n_pairs;
  int n_terms;
  PoleTerm term[kMaxTerms];
  gf_propagator line_k;
  double cutoff2, s0, c0;
  double line2_scale;  // |m2^2| or the largest pole modulus: sizes the deformed contours
  int contour;         // gf_contour
  int thread_ok;       // THREAD applicable (equal real masses)
  int split_log2;      // lanes per grid point = 1 << split_log2
};

struct LaunchPlan {
  int block_threads;
  long long grid_blocks;
  int split_log2;
  size_t smem_bytes;
  bool shared_nodes;  // REAL: per-node tables staged once per CTA
};

// host-side helpers (gf_api.cu)
void set_error(const char* fmt, ...);
int check_cuda(cudaError_t e, const char* what);

// gf_tables.cpp
int make_rule_host(int kind, int n, double step, int measure, double* nodes, double* weights);

// gf_grid.cu
int launch_make_grid(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
                     int spacing, double im_abs_min, int row_first, int n_rows, double2* d_x,
                     cudaStream_t stream);

// gf_eval.cu
int plan_eval(const EvalArgs& a, int precision, LaunchPlan* plan);
int launch_eval(const EvalArgs& a, int precision, cudaStream_t stream);
void eval_inst_counts(const EvalArgs& a, int precision, const LaunchPlan& plan, double* fp64_inst,
                      double* fp32_inst, double* flops);

// gf_diag.cu
int launch_fp64_peak(int blocks, int threads, long long iters, double* d_sink, cudaStream_t stream);
int launch_rcp_seed(const double* d_in, double* d_out, long long n, cudaStream_t stream);

}  // namespace gf
