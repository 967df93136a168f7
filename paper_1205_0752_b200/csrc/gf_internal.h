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
  double mu_re_lo, mu_im_lo;   // mu = (mu_re + mu_re_lo) + i (mu_im + mu_im_lo): the roots of a rational line are made
                               // in binary128 on the host; where a deformed contour passes next to the pole of D2(y)
                               // at y = -mu, y + mu must be accurate to an ulp of ITSELF (reading G18)
};

constexpr int kMaxTerms = 2;
constexpr int kBlkMaxLev = 4;    // levels of the tree of blocks of a split angular rule (gf_routes.cuh)
constexpr int kMaxTaylor = 4;   // largest order n of the Taylor subtraction t^n (gf_taylor.cu)
#ifndef GF_BLOCK_THREADS
#define GF_BLOCK_THREADS 256
#endif
constexpr int kBlockThreads = GF_BLOCK_THREADS;
constexpr int kKreqBins = 256;
#ifndef GF_TAIL_N
#define GF_TAIL_N 32
#endif
#ifndef GF_TAIL_FACTOR
#define GF_TAIL_FACTOR 4.0
#endif
constexpr int kTailN = GF_TAIL_N;  // terms of the large-y tail series (gf_eval.cu)
// the tail takes over at y >= kTailFactor x (the extent of the cut in the y-plane); term n of its series is below
// kTailFactor^-n there, and 4^-32 is 5e-20 (longer series with a lower threshold were measured slower: the series is one dependent chain per point)
constexpr double kTailFactor = GF_TAIL_FACTOR;

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
  PoleTerm kroot[2];   // rational line 1: y^2 + a y + b = (y + nu_1)(y + nu_2), nu in mu_re.. (deformed contours
                       // evaluate the denominator in this form: accurate next to a root)
  double cutoff2, s0, c0;
  double ypow;         // radial measure dy y^ypow: (d - 2)/2, 1 in d = 4
  double Llog_hi, Llog_lo;  // ln((Lambda^2 + s0)/s0) as a double-double (host, binary128)
  double line2_scale;  // |m2^2| or the largest pole modulus: sizes the deformed contours
  int contour;         // gf_contour
  int routing;         // 0: eq. (19) (lines k, p-k); 1: symmetric (lines k + p/2, k - p/2)
  int thread_ok;       // THREAD applicable (equal real masses)
  int same_mass;       // line 1 is 1/(y + mu_0) with the one pole of line 2: D1(y)/(y + mu) = 1/(y + mu)^2
  double parab_c2;     // (Re sqrt(mu))^2, the smallest over the poles of line 2: REAL is the continuation inside the
                       // parabola Re x > (Im x)^2/(4 c2) - c2 (AUTO's first test)
  int rung_lo;         // ladder index of the first tabulated contour radius (deformed contours)
  int split_log2;      // lanes per grid point = 1 << split_log2
  int taylor_order;    // n of the Taylor subtraction t^n (eq. (13)); n > 0 runs gf_taylor.cu
  int* status;         // mapped host word the kernels report bad input to (gf.h "Errors"); may be null
  double ws_tag;       // hash of (params, orders, layout version) as a double in [1, 2): the preparation kernel writes
                       // it into the workspace header, the evaluation kernels refuse a workspace that carries another
};
// codes a kernel leaves in *status (the next API call of the device returns GF_ERR_ARG and describes it)
enum { kStatusAsymmetricRule = 1, kStatusRadialNodes = 2, kStatusWorkspace = 4 };
constexpr int kLayoutVersion = 13;   // bump when a BlobLayout or the meaning of a table changes

// Offsets (in doubles) of the prepared tables, as the preparation kernel writes them and every CTA of the
// evaluation kernel copies them to shared memory (one 16-byte header first).
struct BlobLayout {
  int npad;                     // n_pairs rounded up to 4
  int kmc;                      // series coefficients k = 0 .. kmc-1 (even)
  int off_t, off_tlo, off_w;    // folded angular rule: t = z^2 (hi, lo), weight
  int off_mom, off_cheb;        // double2 (P_k, N_k)[kmc]: centred-moment series, Chebyshev series
  int off_kreq;                 // int Kreq[kKreqBins]: entry 0 "no series", entry 1 + b the Chebyshev terms needed in bin b of log2(rho)
  int n_rad_pad;                // n_rad rounded up to 32: padding repeats the last node with prefactor 0
  int off_y, off_q4;            // radial nodes y_i, 1/(4 y_i), n_rad_pad each
  int n_pref;                   // rows of node prefactors: n_terms, + 1 for the symmetric routing's second tail table
  int off_pref;                 // double2 pref[n_pref][n_rad_pad]
  int off_sf;                   // float2 mom[kmc], cheb[kmc]: the series tables in float (high-order terms run in FP32)
  int off_f32;                  // FP32 variant: float t[npad], w[npad]; or -1
  int off_rt, off_rw, n_tab;    // point-dependent contours: the radial rule pyramid (nodes, weights) or -1
  int n_doubles;                // doubles every CTA stages (even)
  int off_gam;                  // tail series: gamma_{n,k}, row n = 1..kTailN at n(n-1)/2, staged; or -1 (no tail)
  int off_gam2;                 // symmetric routing: kappa_{n,k} = mu_k C(n+k, n-1-k), same shape; or -1
  int off_tail;                 // NOT staged (global): double2 Rhat[n_pref][n_rad + 1][kTailN]
  int off_scratch;              // preparation-only scratch: T_k(s_j) [npad][kmc]; tail: q_i^n (hi, lo) [kTailN][n_rad] x 2
  int off_scratch2;
  int off_scratch3;             // tail: Q_c(i) [kTailN][n_rad], run starts (double-double)
  // deformed contours: one row of tables per contour radius R_k of the ladder (kRungs rungs + the cap Lambda^2/2),
  // NOT staged.  Row k starts at off_rung + k rung_stride; inside a row (offsets in doubles):
  //   rg_r, rg_q4 [n_rad/2]            ray |y| = r_i in [0, R_k] (shifted-log, correctly rounded), 1/(4 r_i)
  //   rg_w [n_rad/2]                   c0 r_i dr_i  (dr_i = rule weight x dr/dt)
  //   rg_y, rg_yq4 [n4p]               real tail y_i in [R_k, Lambda^2], 1/(4 y_i)     (n4p = n_rad/4 rounded up to even)
  //   rg_pref double2 [n_terms][n4p]   node prefactors of the tail, as off_pref
  //   rg_tail double2 [n_terms][n_rad/4 + 1][kTailN]   Rhat of the tail segment
  //   rg_s2, rg_s3                     preparation-only scratch of the row
  long long off_rung, rung_stride;
  int n_rungs;                  // rows (kRungs + 1) or 0
  int n4p, rg_r, rg_q4, rg_w, rg_y, rg_yq4, rg_pref, rg_tail, rg_s2, rg_s3;
  long long n_total;            // doubles to allocate
  // Taylor order n > 0 (gf_taylor.cu): n_poly = n + 2 series tables per family, [k][n_poly], and 1/(y_i + mu_r)
  int n_poly, off_momA, off_chebA, off_ic;
  // blocks of the folded rule for the direct routes (gf_routes.cuh, angular_blocked), staged: n_blk x (c, 1/h) and
  // n_blk x kBlkTerms Chebyshev moments; n_blk = 0: the rule is not split
  int n_blk, off_blk, off_blkM;
  // the blocks form a binary tree: level l joins 2^l leaves (kBlkPairs 2^l pairs); lev_off[l] = index of level l's first
  // block in the tables, n_lev levels, n_blk_all blocks over all levels (tables: n_blk_all entries)
  int n_lev, n_blk_all, lev_off[kBlkMaxLev];
  long long off_blkS;           // preparation-only scratch of the block tables: double2 [n_lev][n_pairs][kBlkTerms]
};
constexpr int kRungs = 64;      // tabulated contour radii above the first (deformed contours); then Lambda^2/2

struct LaunchPlan {
  int block_threads;
  long long grid_blocks;
  int split_log2;
  size_t smem_bytes;
  bool shared_nodes;  // REAL: per-node tables prepared once per launch
  BlobLayout layout;
};

// host-side helpers (gf_api.cu)
void set_error(const char* fmt, ...);
int check_cuda(cudaError_t e, const char* what);
int scratch_alloc(void** ptr, size_t bytes, cudaStream_t stream);  // from the library's own stream-ordered pool
int attach_status(EvalArgs* a);   // a->status = the current device's status word (allocated on first use)
int take_status(const char* where);   // GF_ERR_ARG (and the word cleared) if a kernel of the current device reported bad input

// gf_tables.cpp
int make_rule_host(int kind, int n, double step, int measure, double* nodes, double* weights);
int make_rule_dim_host(int kind, int n, double step, double dim, double* nodes, double* weights);
void log_ratio_dd(double a, double b, double s0, double* hi, double* lo);  // ln((b+s0)/(a+s0)), binary128 -> (hi, lo)

// gf_grid.cu
int launch_make_grid(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
                     int spacing, double im_abs_min, int row_first, int n_rows, double2* d_x,
                     cudaStream_t stream);

// gf_eval.cu
int plan_eval(const EvalArgs& a, int precision, LaunchPlan* plan);
int launch_eval(const EvalArgs& a, int precision, unsigned long long* d_counters, cudaStream_t stream);
int launch_prepare(const EvalArgs& a, int precision, double* blob, cudaStream_t stream);
int launch_prepared(const EvalArgs& a, int precision, const double* blob, unsigned long long* d_counters,
                    cudaStream_t stream);
// gf_contour.cu: evaluation kernel for contours that depend on the grid point (RAY_ARC, THREAD, AUTO)
int launch_contour(const EvalArgs& a, const LaunchPlan& plan, const double* blob, unsigned long long* d_counters,
                   cudaStream_t stream);
int launch_prepare_rungs(const EvalArgs& a, const LaunchPlan& plan, double* blob, cudaStream_t stream);
int launch_contour_nodes(const EvalArgs& a, const LaunchPlan& plan, const double* blob, double x_re, double x_im,
                         int* d_policy, double2* d_y, double2* d_wy, cudaStream_t stream);
int launch_radial_map(double Llog_hi, double Llog_lo, double s0, const double* d_nodes, int n, double* d_y,
                      cudaStream_t stream);

// gf_taylor.cu: Taylor subtraction of order n > 0 on the REAL contour
int plan_taylor(const EvalArgs& a, LaunchPlan* plan);
int launch_taylor_prepare(const EvalArgs& a, const LaunchPlan& plan, double* blob, cudaStream_t stream);
int launch_taylor(const EvalArgs& a, const LaunchPlan& plan, const double* blob, cudaStream_t stream);

// gf_cut.cu: the paper's Kernels 3 and 4 (a.x holds the y array / the x array, a.out the result)
BlobLayout make_blob_layout(int n_rad, int n_pairs, int n_terms, bool f32, bool pyramid, bool tail,
                            bool sym = false, int taylor_order = 0);  // gf_eval.cu; pyramid: the layout of the deformed-contour kernel
int launch_angular(const EvalArgs& a, double x_re, double x_im, cudaStream_t stream);
int launch_cut_crossings(const EvalArgs& a, int n_z, int* d_out, cudaStream_t stream);

// gf_diag.cu
int launch_fp64_peak(int blocks, int threads, long long iters, double* d_sink, cudaStream_t stream);
int launch_dfma_issue(int mode, int blocks, int threads, long long iters, double* d_sink, cudaStream_t stream);

}  // namespace gf
