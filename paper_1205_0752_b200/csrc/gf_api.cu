// gf_api.cu -- the C ABI of include/gf.h: argument validation, host-side preparation (pole
// decomposition of line 2, launch plan) and kernel launches.  No torch types, no exceptions.
#include <quadmath.h>

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdarg>
#include <cstdio>
#include <exception>
#include <mutex>
#include <vector>

#include "gf_internal.h"

namespace gf {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

int check_cuda(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return GF_OK;
  set_error("%s: %s", what, cudaGetErrorString(e));
  return GF_ERR_CUDA;
}

// Scratch comes from a stream-ordered memory pool of the library's own (one per device) that keeps freed
// blocks for the next call instead of returning them to the driver at every synchronisation (the default
// pool does that, and mapping ~200 MB again costs milliseconds per call); gf_trim_scratch() empties it.
static cudaMemPool_t g_pool[64] = {};
static std::mutex g_pool_mutex;

static int scratch_pool(cudaMemPool_t* pool) {
  int dev = 0;
  int rc = check_cuda(cudaGetDevice(&dev), "cudaGetDevice");
  if (rc) return rc;
  if (dev < 0 || dev >= 64) { set_error("device ordinal %d out of range", dev); return GF_ERR_CUDA; }
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (!g_pool[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    if ((rc = check_cuda(cudaMemPoolCreate(&g_pool[dev], &props), "cudaMemPoolCreate"))) { g_pool[dev] = nullptr; return rc; }
    unsigned long long keep = ~0ULL;
    cudaMemPoolSetAttribute(g_pool[dev], cudaMemPoolAttrReleaseThreshold, &keep);
  }
  *pool = g_pool[dev];
  return GF_OK;
}

int scratch_alloc(void** ptr, size_t bytes, cudaStream_t stream) {
  cudaMemPool_t pool;
  int rc = scratch_pool(&pool);
  if (rc) return rc;
  return check_cuda(cudaMallocFromPoolAsync(ptr, bytes, pool, stream), "cudaMallocFromPoolAsync(scratch)");
}

// One mapped host word per device that kernels report bad input to (an asymmetric angular rule, radial tables that are
// not ascending inside (-1,1), a workspace prepared for other parameters): zero-copy, so reading it needs no
// synchronisation.  Allocated on first use, kept for the life of the process (4 bytes of pinned host memory).
static int* g_status[64] = {};

static int status_word(int** word) {
  int dev = 0;
  int rc = check_cuda(cudaGetDevice(&dev), "cudaGetDevice");
  if (rc) return rc;
  if (dev < 0 || dev >= 64) { set_error("device ordinal %d out of range", dev); return GF_ERR_CUDA; }
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (!g_status[dev]) {
    int* h = nullptr;
    if ((rc = check_cuda(cudaHostAlloc(reinterpret_cast<void**>(&h), sizeof(int), cudaHostAllocMapped), "cudaHostAlloc(status word)"))) return rc;
    *h = 0;
    g_status[dev] = h;
  }
  *word = g_status[dev];
  return GF_OK;
}

int attach_status(EvalArgs* a) {
  int* h = nullptr;
  int rc = status_word(&h);
  if (rc) return rc;
  int* d = nullptr;
  if ((rc = check_cuda(cudaHostGetDevicePointer(reinterpret_cast<void**>(&d), h, 0), "cudaHostGetDevicePointer(status word)"))) return rc;
  a->status = d;
  return GF_OK;
}

int take_status(const char* where) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return GF_OK; }
  int* h;
  {
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    h = g_status[dev];
  }
  if (!h) return GF_OK;
  const int code = __atomic_exchange_n(h, 0, __ATOMIC_ACQ_REL);
  if (!code) return GF_OK;
  set_error("%s: a kernel of this device was given bad input:%s%s%s", where,
            (code & kStatusAsymmetricRule) ? " an angular rule that is not symmetric (z[n-1-j] = -z[j], equal weights);" : "",
            (code & kStatusRadialNodes) ? " radial nodes that are not ascending strictly inside (-1,1);" : "",
            (code & kStatusWorkspace) ? " a workspace prepared with other parameters, orders or precision;" : "");
  return GF_ERR_ARG;
}

namespace {

// FNV-1a over the parameter block and the orders -> a double in [1, 2) (EvalArgs::ws_tag)
double workspace_tag(const gf_params* p, int n_rad, int n_ang) {
  unsigned long long h = 1469598103934665603ULL;
  auto mix = [&](const void* ptr, size_t n) {
    const unsigned char* b = static_cast<const unsigned char*>(ptr);
    for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ULL; }
  };
  // field by field: the struct's padding bytes are not the caller's to define
  const gf_propagator* pr[2] = {&p->line_k, &p->line_pk};
  for (int k = 0; k < 2; ++k) {
    mix(&pr[k]->kind, sizeof(int)); mix(&pr[k]->m2_re, sizeof(double)); mix(&pr[k]->m2_im, sizeof(double));
    mix(&pr[k]->M2, sizeof(double)); mix(&pr[k]->a, sizeof(double)); mix(&pr[k]->b, sizeof(double));
  }
  mix(&p->cutoff2, sizeof(double)); mix(&p->sub_re, sizeof(double)); mix(&p->sub_im, sizeof(double));
  mix(&p->taylor_order, sizeof(int)); mix(&p->prefactor, sizeof(double)); mix(&p->map_scale, sizeof(double));
  mix(&p->contour, sizeof(int)); mix(&p->precision, sizeof(int)); mix(&p->routing, sizeof(int)); mix(&p->dim, sizeof(double));
  const int extra[3] = {n_rad, n_ang, kLayoutVersion};
  mix(extra, sizeof(extra));
  return 1.0 + (double)(h >> 12) * 0x1p-52;
}

// per (point, node, pole) FP64-pipe instructions of each route's set-up + finish (SASS of eval_real_kernel<double>)
constexpr double kNodeNearDfma = 12, kNodeNearOther = 13, kNodeMomentDfma = 21, kNodeMomentOther = 15,
                 kNodeChebDfma = 31, kNodeChebOther = 28;

bool finite_prop(const gf_propagator& p) {
  return std::isfinite(p.m2_re) && std::isfinite(p.m2_im) && std::isfinite(p.M2) && std::isfinite(p.a) &&
         std::isfinite(p.b);
}

int check_prop(const gf_propagator& p, const char* name) {
  if (p.kind != GF_PROP_MASSIVE && p.kind != GF_PROP_RATIONAL) {
    set_error("%s: unknown propagator kind %d", name, p.kind);
    return GF_ERR_ARG;
  }
  if (!finite_prop(p)) { set_error("%s: non-finite propagator parameter", name); return GF_ERR_ARG; }
  return GF_OK;
}

// index of the smallest rung >= v of the ladder {2^k, 1.5 2^k}: rung I is 2^(I/2) for even I, 1.5 2^((I-1)/2) for odd I
int rung_index(double v) {
  int e;
  const double m = std::frexp(v, &e);   // v = m 2^e, 0.5 <= m < 1
  if (m == 0.5) return 2 * (e - 1);
  if (m <= 0.75) return 2 * (e - 1) + 1;
  return 2 * e;
}

// The roots u_1 = (-a + sqrt(a^2-4b))/2, u_2 = (-a - sqrt(a^2-4b))/2 of u^2 + a u + b and the residues
// R_r = (u_r + M2)/(u_r - u_s) of (u + M2)/(u^2 + a u + b), in binary128 (the smaller real root from b/q: no
// cancellation), returned as poles -mu_r with mu_r split into hi + lo.
void rational_poles(double M2, double a, double b, PoleTerm* t) {
  const __float128 A = a, B = b, disc = A * A - 4 * B;
  __float128 ur[2], ui[2] = {0, 0};
  if (disc >= 0) {
    const __float128 sq = sqrtq(disc);
    if (A >= 0) { ur[1] = -(A + sq) / 2; ur[0] = ur[1] != 0 ? B / ur[1] : (__float128)0; }
    else { ur[0] = (sq - A) / 2; ur[1] = B / ur[0]; }
  } else {
    ur[0] = ur[1] = -A / 2;
    ui[0] = sqrtq(-disc) / 2;
    ui[1] = -ui[0];
  }
  for (int r = 0; r < 2; ++r) {
    const int s = 1 - r;
    // R_r = (u_r + M2)/(u_r - u_s)
    const __float128 nr = ur[r] + (__float128)M2, ni = ui[r], dr = ur[r] - ur[s], di = ui[r] - ui[s];
    const __float128 dn = dr * dr + di * di;
    t[r].R_re = (double)((nr * dr + ni * di) / dn);
    t[r].R_im = (double)((ni * dr - nr * di) / dn);
    t[r].mu_re = (double)(-ur[r]);
    t[r].mu_re_lo = (double)(-ur[r] - (__float128)t[r].mu_re);
    t[r].mu_im = (double)(-ui[r]);
    t[r].mu_im_lo = (double)(-ui[r] - (__float128)t[r].mu_im);
  }
}

// validate everything that does not need a pointer, and build the kernel arguments
int build_args(const gf_params* p, int n_rad, int n_ang, long long n_points, EvalArgs* a) {
  if (!p) { set_error("eval_grid: params is null"); return GF_ERR_NULL; }
  int rc;
  if ((rc = check_prop(p->line_k, "line_k"))) return rc;
  if ((rc = check_prop(p->line_pk, "line_pk"))) return rc;
  if (n_rad < 1 || n_ang < 1) { set_error("eval_grid: n_rad=%d, n_ang=%d must be >= 1", n_rad, n_ang); return GF_ERR_ARG; }
  if (n_points < 0) { set_error("eval_grid: n_points < 0"); return GF_ERR_ARG; }
  if (!(p->cutoff2 > 0) || !(p->cutoff2 <= 1e60)) { set_error("eval_grid: cutoff2 must be in (0, 1e60]"); return GF_ERR_ARG; }
  if (!(p->map_scale > 0) || !std::isfinite(p->map_scale)) { set_error("eval_grid: map_scale must be > 0"); return GF_ERR_ARG; }
  if (!std::isfinite(p->prefactor)) { set_error("eval_grid: prefactor not finite"); return GF_ERR_ARG; }
  if (p->precision != 64 && p->precision != 32) { set_error("eval_grid: precision must be 64 or 32"); return GF_ERR_ARG; }
  if (p->contour < GF_CONTOUR_REAL || p->contour > GF_CONTOUR_AUTO) { set_error("eval_grid: unknown contour %d", p->contour); return GF_ERR_ARG; }
  if (p->taylor_order < 0 || p->taylor_order > kMaxTaylor) { set_error("eval_grid: taylor_order %d outside [0, %d] (eq. (13))", p->taylor_order, kMaxTaylor); return GF_ERR_UNSUPPORTED; }
  if (p->taylor_order > 0 && (p->routing != 0 || p->precision != 64)) {
    set_error("eval_grid: taylor_order > 0 is built for the paper's routing and precision 64");
    return GF_ERR_UNSUPPORTED;
  }
  if (p->sub_re != 0 || p->sub_im != 0) { set_error("eval_grid: subtraction point must be 0 (eq. (13))"); return GF_ERR_UNSUPPORTED; }
  if (p->routing != 0 && p->routing != 1) { set_error("eval_grid: unknown routing %d", p->routing); return GF_ERR_ARG; }
  if (p->routing == 1 && !(p->line_k.kind == GF_PROP_MASSIVE && p->line_pk.kind == GF_PROP_MASSIVE &&
                           p->line_k.m2_re == p->line_pk.m2_re && p->line_k.m2_im == p->line_pk.m2_im)) {
    set_error("eval_grid: symmetric routing needs two equal massive lines");
    return GF_ERR_UNSUPPORTED;
  }
  if (!(p->dim == 0 || (p->dim >= 1 && p->dim <= 8))) { set_error("eval_grid: dim=%g outside [1, 8] (0 = 4)", p->dim); return GF_ERR_ARG; }
  if (p->contour != GF_CONTOUR_REAL && n_rad % 8 != 0) { set_error("eval_grid: deformed contours need n_rad %% 8 == 0"); return GF_ERR_ARG; }

  *a = EvalArgs{};
  a->n_points = n_points;
  a->n_rad = n_rad;
  a->n_ang = n_ang;
  a->n_pairs = (n_ang + 1) / 2;
  a->line_k = p->line_k;
  a->cutoff2 = p->cutoff2;
  a->s0 = p->map_scale;
  a->c0 = p->prefactor;
  a->ypow = (p->dim == 0 || p->dim == 4) ? 1.0 : 0.5 * (p->dim - 2.0);
  log_ratio_dd(0.0, p->cutoff2, p->map_scale, &a->Llog_hi, &a->Llog_lo);  // REAL contour: [0, Lambda^2]
  a->contour = p->contour;
  a->routing = p->routing;
  a->taylor_order = p->taylor_order;
  a->ws_tag = workspace_tag(p, n_rad, n_ang);

  // line 2 as a sum of simple poles R_r/(u + mu_r)
  const gf_propagator& q = p->line_pk;
  if (q.kind == GF_PROP_MASSIVE) {
    a->n_terms = 1;
    a->term[0] = PoleTerm{1.0, 0.0, q.m2_re, q.m2_im, 0.0, 0.0};
    a->line2_scale = std::hypot(q.m2_re, q.m2_im);
  } else {
    const double disc = q.a * q.a - 4.0 * q.b;
    if (disc == 0.0) {
      set_error("line_pk: rational propagator with a double pole (a^2 = 4b) is unsupported");
      return GF_ERR_UNSUPPORTED;
    }
    a->n_terms = 2;
    rational_poles(q.M2, q.a, q.b, a->term);
    // size of the singular structure of line 2 in the y-plane, the largest pole modulus: sqrt(b) for a
    // complex-conjugate pair (|u_r|^2 = b), else max |(-a +- sqrt(disc))/2|
    a->line2_scale = disc < 0 ? std::sqrt(q.b)
                              : std::fmax(std::fabs(-q.a + std::sqrt(disc)), std::fabs(-q.a - std::sqrt(disc))) / 2.0;
  }
  if (p->line_k.kind == GF_PROP_RATIONAL) rational_poles(p->line_k.M2, p->line_k.a, p->line_k.b, a->kroot);
  a->thread_ok = p->line_k.kind == GF_PROP_MASSIVE && q.kind == GF_PROP_MASSIVE && p->line_k.m2_im == 0 &&
                 q.m2_im == 0 && p->line_k.m2_re == q.m2_re && q.m2_re > 0;
  a->same_mass = p->line_k.kind == GF_PROP_MASSIVE && q.kind == GF_PROP_MASSIVE && p->line_k.m2_re == q.m2_re &&
                 p->line_k.m2_im == q.m2_im;
  // AUTO's parabola: (Re sqrt(mu))^2 = (|mu| + Re mu)/2, the smallest over the poles -mu of line 2 (gf.h, gf_contour)
  {
    auto c2 = [](double mr, double mi) { return 0.5 * (std::sqrt(std::fma(mr, mr, mi * mi)) + mr); };
    if (q.kind == GF_PROP_MASSIVE) a->parab_c2 = c2(q.m2_re, q.m2_im);
    else {
      const double disc = q.a * q.a - 4.0 * q.b;
      if (disc >= 0.0) {
        const double r = std::sqrt(disc);
        a->parab_c2 = std::fmin(c2(0.5 * (q.a - r), 0.0), c2(0.5 * (q.a + r), 0.0));
      } else {
        a->parab_c2 = c2(0.5 * q.a, 0.5 * std::sqrt(-disc));
      }
    }
  }
  // the ladder of contour radii {2^k, 1.5 2^k} starts one rung below the smallest rung >= 1.5 sc (gf.h, gf_contour)
  a->rung_lo = rung_index(1.5 * a->line2_scale) - 1;
  if (p->contour == GF_CONTOUR_THREAD && !a->thread_ok) {
    set_error("eval_grid: the THREAD contour needs equal real positive masses on both lines");
    return GF_ERR_UNSUPPORTED;
  }
  return GF_OK;
}

long long radial_table_size(int contour, int n_rad) {
  if (n_rad < 1) return -1;
  if (contour == GF_CONTOUR_REAL) return n_rad;
  if (contour < GF_CONTOUR_REAL || contour > GF_CONTOUR_AUTO || n_rad % 8 != 0) return -1;
  return (long long)n_rad + n_rad / 2 + n_rad / 4 + n_rad / 8;
}

}  // namespace
}  // namespace gf

using namespace gf;

// gf_tables.cpp allocates (std::vector) and may start threads: nothing may propagate across the C ABI
template <typename F>
static int no_throw(const char* what, F&& f) {
  try {
    return f();
  } catch (const std::exception& e) {
    set_error("%s: %s", what, e.what());
  } catch (...) {
    set_error("%s: unknown C++ exception", what);
  }
  return GF_ERR_ARG;
}

extern "C" {

const char* gf_last_error(void) { return g_err; }
int gf_trim_scratch(void) {
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  int rc = GF_OK;
  for (int dev = 0; dev < 64; ++dev)
    if (g_pool[dev]) {
      int r = check_cuda(cudaMemPoolTrimTo(g_pool[dev], 0), "cudaMemPoolTrimTo");
      if (r) rc = r;
    }
  return rc;
}

const char* gf_version(void) { return "gf_b200 0.3 (sm_100a)"; }
#ifndef GF_BUILD_ID
#define GF_BUILD_ID ""
#endif
const char* gf_build_id(void) { return GF_BUILD_ID; }

static int make_grid_rows(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
                          int spacing, double im_abs_min, int row_first, int n_rows, void* d_x, void* stream) {
  if (n_re < 1 || n_im < 1) { set_error("make_grid: n_re=%d, n_im=%d must be >= 1", n_re, n_im); return GF_ERR_ARG; }
  if (row_first < 0 || n_rows < 0 || (long long)row_first + n_rows > n_im) {
    set_error("make_grid: rows [%d, %d+%d) outside the grid of %d rows", row_first, row_first, n_rows, n_im);
    return GF_ERR_ARG;
  }
  if (!d_x && n_rows > 0) { set_error("make_grid: d_x is null"); return GF_ERR_NULL; }
  if (!std::isfinite(re_min) || !std::isfinite(re_max) || !std::isfinite(im_min) || !std::isfinite(im_max)) {
    set_error("make_grid: non-finite box");
    return GF_ERR_ARG;
  }
  if (spacing == GF_SPACING_LOG_ABS_IM) {
    if (n_im % 2 != 0 || !(im_abs_min > 0) || !(im_max > im_abs_min) || im_min != -im_max) {
      set_error("make_grid: LOG_ABS_IM needs n_im even, im_min == -im_max, 0 < im_abs_min < im_max");
      return GF_ERR_ARG;
    }
  } else if (spacing != GF_SPACING_UNIFORM) {
    set_error("make_grid: unknown spacing %d", spacing);
    return GF_ERR_ARG;
  }
  return launch_make_grid(re_min, re_max, n_re, im_min, im_max, n_im, spacing, im_abs_min, row_first, n_rows,
                          static_cast<double2*>(d_x), static_cast<cudaStream_t>(stream));
}

int gf_make_grid(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im, int spacing,
                 double im_abs_min, void* d_x, void* stream) {
  if (!d_x) { set_error("make_grid: d_x is null"); return GF_ERR_NULL; }
  return make_grid_rows(re_min, re_max, n_re, im_min, im_max, n_im, spacing, im_abs_min, 0, n_im, d_x, stream);
}

int gf_make_grid_rows(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im, int spacing,
                      double im_abs_min, int row_first, int n_rows, void* d_x, void* stream) {
  return make_grid_rows(re_min, re_max, n_re, im_min, im_max, n_im, spacing, im_abs_min, row_first, n_rows, d_x,
                        stream);
}

int gf_make_quadrature_host(int kind, int n, double step, int measure, double* h_nodes, double* h_weights) {
  return no_throw("make_quadrature_host", [&] { return make_rule_host(kind, n, step, measure, h_nodes, h_weights); });
}

int gf_make_quadrature(int kind, int n, double step, int measure, double* d_nodes, double* d_weights, void* stream) {
  if (!d_nodes || !d_weights) { set_error("make_quadrature: null device pointer"); return GF_ERR_NULL; }
  if (n < 1 || n > (1 << 20)) { set_error("make_quadrature: n=%d out of range", n); return GF_ERR_ARG; }
  return no_throw("make_quadrature", [&] {
    std::vector<double> x(n), w(n);
    int rc = make_rule_host(kind, n, step, measure, x.data(), w.data());
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // pageable source: the runtime stages the data before returning, so x, w may go out of scope
    if ((rc = check_cuda(cudaMemcpyAsync(d_nodes, x.data(), sizeof(double) * n, cudaMemcpyHostToDevice, s), "copy nodes"))) return rc;
    return check_cuda(cudaMemcpyAsync(d_weights, w.data(), sizeof(double) * n, cudaMemcpyHostToDevice, s), "copy weights");
  });
}

int gf_make_quadrature_dim_host(int kind, int n, double step, double dim, double* h_nodes, double* h_weights) {
  return no_throw("make_quadrature_dim_host", [&] { return make_rule_dim_host(kind, n, step, dim, h_nodes, h_weights); });
}

int gf_make_quadrature_dim(int kind, int n, double step, double dim, double* d_nodes, double* d_weights, void* stream) {
  if (!d_nodes || !d_weights) { set_error("make_quadrature_dim: null device pointer"); return GF_ERR_NULL; }
  if (n < 1 || n > (1 << 20)) { set_error("make_quadrature_dim: n=%d out of range", n); return GF_ERR_ARG; }
  return no_throw("make_quadrature_dim", [&] {
    std::vector<double> x(n), w(n);
    int rc = make_rule_dim_host(kind, n, step, dim, x.data(), w.data());
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if ((rc = check_cuda(cudaMemcpyAsync(d_nodes, x.data(), sizeof(double) * n, cudaMemcpyHostToDevice, s), "copy nodes"))) return rc;
    return check_cuda(cudaMemcpyAsync(d_weights, w.data(), sizeof(double) * n, cudaMemcpyHostToDevice, s), "copy weights");
  });
}

long long gf_radial_table_size(int contour, int n_rad) { return radial_table_size(contour, n_rad); }

static int eval_grid_impl(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                          const double* d_ang_nodes, const double* d_ang_weights, int n_ang, const void* d_x,
                          long long n_points, void* d_out, unsigned long long* d_counters, void* stream) {
  EvalArgs a;
  int rc = build_args(p, n_rad, n_ang, n_points, &a);
  if (rc) return rc;
  if (!d_rad_nodes || !d_rad_weights || !d_ang_nodes || !d_ang_weights) { set_error("eval_grid: null table pointer"); return GF_ERR_NULL; }
  if (n_points > 0 && (!d_x || !d_out)) { set_error("eval_grid: null grid/output pointer"); return GF_ERR_NULL; }
  if ((rc = take_status("eval_grid")) || (rc = attach_status(&a))) return rc;
  a.rad_nodes = d_rad_nodes;
  a.rad_weights = d_rad_weights;
  a.ang_nodes = d_ang_nodes;
  a.ang_weights = d_ang_weights;
  a.x = static_cast<const double2*>(d_x);
  a.out = d_out;
  return launch_eval(a, p->precision, d_counters, static_cast<cudaStream_t>(stream));
}

int gf_eval_grid(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                 const double* d_ang_nodes, const double* d_ang_weights, int n_ang, const void* d_x,
                 long long n_points, void* d_out, void* stream) {
  return eval_grid_impl(p, d_rad_nodes, d_rad_weights, n_rad, d_ang_nodes, d_ang_weights, n_ang, d_x, n_points,
                        d_out, nullptr, stream);
}

int gf_eval_grid_counted(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                         const double* d_ang_nodes, const double* d_ang_weights, int n_ang, const void* d_x,
                         long long n_points, void* d_out, unsigned long long* d_counters, void* stream) {
  if (!d_counters) { set_error("eval_grid_counted: d_counters is null"); return GF_ERR_NULL; }
  return eval_grid_impl(p, d_rad_nodes, d_rad_weights, n_rad, d_ang_nodes, d_ang_weights, n_ang, d_x, n_points,
                        d_out, d_counters, stream);
}

long long gf_eval_workspace_size(const gf_params* p, int n_rad, int n_ang) {
  EvalArgs a;
  if (build_args(p, n_rad, n_ang, 1, &a)) return -1;
  LaunchPlan plan;
  if (plan_eval(a, p->precision, &plan)) return -1;
  return (long long)plan.layout.n_total * (long long)sizeof(double);
}

int gf_eval_prepare(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                    const double* d_ang_nodes, const double* d_ang_weights, int n_ang, void* d_workspace,
                    void* stream) {
  EvalArgs a;
  int rc = build_args(p, n_rad, n_ang, 1, &a);
  if (rc) return rc;
  if (!d_rad_nodes || !d_rad_weights || !d_ang_nodes || !d_ang_weights) { set_error("eval_prepare: null table pointer"); return GF_ERR_NULL; }
  if (!d_workspace) { set_error("eval_prepare: d_workspace is null"); return GF_ERR_NULL; }
  if ((rc = take_status("eval_prepare")) || (rc = attach_status(&a))) return rc;
  a.rad_nodes = d_rad_nodes;
  a.rad_weights = d_rad_weights;
  a.ang_nodes = d_ang_nodes;
  a.ang_weights = d_ang_weights;
  return launch_prepare(a, p->precision, static_cast<double*>(d_workspace), static_cast<cudaStream_t>(stream));
}

int gf_eval_grid_prepared(const gf_params* p, int n_rad, int n_ang, const void* d_workspace, const void* d_x,
                          long long n_points, void* d_out, unsigned long long* d_counters, void* stream) {
  EvalArgs a;
  int rc = build_args(p, n_rad, n_ang, n_points, &a);
  if (rc) return rc;
  if (!d_workspace) { set_error("eval_grid_prepared: d_workspace is null"); return GF_ERR_NULL; }
  if (n_points > 0 && (!d_x || !d_out)) { set_error("eval_grid_prepared: null grid/output pointer"); return GF_ERR_NULL; }
  if ((rc = take_status("eval_grid_prepared")) || (rc = attach_status(&a))) return rc;
  a.x = static_cast<const double2*>(d_x);
  a.out = d_out;
  return launch_prepared(a, p->precision, static_cast<const double*>(d_workspace), d_counters,
                         static_cast<cudaStream_t>(stream));
}

int gf_eval_grid_host(const gf_params* p, const double* h_rad_nodes, const double* h_rad_weights, int n_rad,
                      const double* h_ang_nodes, const double* h_ang_weights, int n_ang, const void* h_x,
                      long long n_points, void* h_out, void* stream) {
  EvalArgs a;
  int rc = build_args(p, n_rad, n_ang, n_points, &a);
  if (rc) return rc;
  if (!h_rad_nodes || !h_rad_weights || !h_ang_nodes || !h_ang_weights) { set_error("eval_grid_host: null table pointer"); return GF_ERR_NULL; }
  if (n_points > 0 && (!h_x || !h_out)) { set_error("eval_grid_host: null grid/output pointer"); return GF_ERR_NULL; }
  // the tables are in host memory here: what the kernels can only answer with NaN (gf_eval_grid) is an error code
  for (int j = 0; j < (n_ang + 1) / 2; ++j) {
    const int jm = n_ang - 1 - j;
    const double zp = h_ang_nodes[jm], zm = h_ang_nodes[j], wp = h_ang_weights[jm], wm = h_ang_weights[j];
    const double tol = 16.0 * 2.220446049250313e-16;
    const bool ok = jm == j ? std::fabs(zp) <= 1e-15
                            : (std::fabs(zp + zm) <= tol * std::fabs(zp) && std::fabs(wp - wm) <= tol * std::fabs(wp));
    if (!ok) { set_error("eval_grid_host: the angular rule is not symmetric at node %d (z[n-1-j] = -z[j], equal weights)", j); return GF_ERR_ARG; }
  }
  {
    int off = 0, n = n_rad;
    for (int l = 0; l < (p->contour == GF_CONTOUR_REAL ? 1 : 4); ++l, off += n, n >>= 1)
      for (int i = 0; i < n; ++i) {
        const double t = h_rad_nodes[off + i];
        if (!(t > -1.0 && t < 1.0) || (i > 0 && !(t > h_rad_nodes[off + i - 1]))) {
          set_error("eval_grid_host: radial nodes must be ascending strictly inside (-1,1) (level %d, node %d)", l, i);
          return GF_ERR_ARG;
        }
      }
  }
  if (n_points == 0) return GF_OK;
  if ((rc = take_status("eval_grid_host")) || (rc = attach_status(&a))) return rc;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const size_t n_radtab = (size_t)radial_table_size(p->contour, n_rad);
  const size_t out_elem = p->precision == 32 ? 8 : 16;
  const size_t tab_bytes = (2 * n_radtab + 2 * (size_t)n_ang) * sizeof(double);
  const size_t x_bytes = (size_t)n_points * 16, out_bytes = (size_t)n_points * out_elem;
  // one scratch allocation: [tables | prepared workspace | x | out], each part 256-byte aligned
  auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
  LaunchPlan plan0;
  if ((rc = plan_eval(a, p->precision, &plan0))) return rc;
  const size_t ws_bytes = (size_t)plan0.layout.n_total * sizeof(double);
  const size_t off_ws = up(tab_bytes), off_x = off_ws + up(ws_bytes), off_out = off_x + up(x_bytes),
               total = off_out + up(out_bytes);
  unsigned char* d = nullptr;
  if ((rc = scratch_alloc(reinterpret_cast<void**>(&d), total, s))) return rc;
  double* d_tab = reinterpret_cast<double*>(d);
  double* d_rn = d_tab;
  double* d_rw = d_rn + n_radtab;
  double* d_an = d_rw + n_radtab;
  double* d_aw = d_an + n_ang;
  cudaError_t e = cudaSuccess;
  auto cp = [&](void* dst, const void* src, size_t n, cudaMemcpyKind k, cudaStream_t st) { if (e == cudaSuccess) e = cudaMemcpyAsync(dst, src, n, k, st); };
  cp(d_rn, h_rad_nodes, n_radtab * 8, cudaMemcpyHostToDevice, s);
  cp(d_rw, h_rad_weights, n_radtab * 8, cudaMemcpyHostToDevice, s);
  cp(d_an, h_ang_nodes, (size_t)n_ang * 8, cudaMemcpyHostToDevice, s);
  cp(d_aw, h_ang_weights, (size_t)n_ang * 8, cudaMemcpyHostToDevice, s);
  rc = check_cuda(e, "host->device copies (tables)");
  a.rad_nodes = d_rn; a.rad_weights = d_rw; a.ang_nodes = d_an; a.ang_weights = d_aw;
  double* d_ws = reinterpret_cast<double*>(d + off_ws);
  if (!rc) rc = launch_prepare(a, p->precision, d_ws, s);

  // x in, kernel, G out as a pipeline of chunks: copies in both directions overlap the evaluation
  // (pinned host buffers; with pageable ones the copies serialise but the result is the same)
  const int kMaxChunks = 8;
  const long long min_chunk = 1 << 18;
  int n_chunks = (int)std::min<long long>(kMaxChunks, std::max<long long>(1, n_points / min_chunk));
  cudaStream_t s_in = nullptr, s_out = nullptr, s_k2 = nullptr;   // copies in / out, second compute stream
  cudaEvent_t ev_ready = nullptr, ev_in[kMaxChunks] = {}, ev_k[kMaxChunks] = {}, ev_done = nullptr;
  auto ok = [&](cudaError_t err, const char* what) { if (!rc) rc = check_cuda(err, what); };
  if (!rc && n_chunks > 1) {
    ok(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking), "cudaStreamCreate");
    ok(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking), "cudaStreamCreate");
    ok(cudaStreamCreateWithFlags(&s_k2, cudaStreamNonBlocking), "cudaStreamCreate");
    ok(cudaEventCreateWithFlags(&ev_ready, cudaEventDisableTiming), "cudaEventCreate");
    ok(cudaEventCreateWithFlags(&ev_done, cudaEventDisableTiming), "cudaEventCreate");
    for (int c = 0; c < n_chunks; ++c) {
      ok(cudaEventCreateWithFlags(&ev_in[c], cudaEventDisableTiming), "cudaEventCreate");
      ok(cudaEventCreateWithFlags(&ev_k[c], cudaEventDisableTiming), "cudaEventCreate");
    }
    if (!rc) {
      ok(cudaEventRecord(ev_ready, s), "cudaEventRecord");          // the scratch exists in stream order of s
      ok(cudaStreamWaitEvent(s_in, ev_ready, 0), "cudaStreamWaitEvent");
      ok(cudaStreamWaitEvent(s_out, ev_ready, 0), "cudaStreamWaitEvent");
      ok(cudaStreamWaitEvent(s_k2, ev_ready, 0), "cudaStreamWaitEvent");
    }
  }
  for (int c = 0; c < n_chunks && !rc; ++c) {
    // boundaries on multiples of the CTA size: every warp holds the same points as in one launch over all of x,
    // so the chunked result is bit-identical to gf_eval_grid's (the series loop runs to the warp's longest series)
    // With the full eight chunks the first and the last are small (1/32 of the points, then 3/32, the middle four 6/32
    // each): the copy in of the first chunk and the copy out of the last are the only ones nothing overlaps
    static const int kRamp[kMaxChunks + 1] = {0, 1, 4, 10, 16, 22, 28, 31, 32};
    auto cut = [&](int k) {
      if (k >= n_chunks) return n_points;
      const long long at = n_chunks == kMaxChunks ? n_points * kRamp[k] / 32 : n_points * k / n_chunks;
      return at / kBlockThreads * kBlockThreads;
    };
    const long long p0 = cut(c), p1 = cut(c + 1), np = p1 - p0;
    // odd chunks are evaluated on a second stream, so that the last, partly filled wave of CTAs of one chunk
    // overlaps the first waves of the next
    cudaStream_t sin = n_chunks > 1 ? s_in : s, sout = n_chunks > 1 ? s_out : s, sk = (c & 1) ? s_k2 : s;
    ok(cudaMemcpyAsync(d + off_x + (size_t)p0 * 16, static_cast<const char*>(h_x) + (size_t)p0 * 16, (size_t)np * 16,
                       cudaMemcpyHostToDevice, sin), "host->device copy (x)");
    if (n_chunks > 1) {
      ok(cudaEventRecord(ev_in[c], s_in), "cudaEventRecord");
      ok(cudaStreamWaitEvent(sk, ev_in[c], 0), "cudaStreamWaitEvent");
    }
    if (!rc) {
      a.x = reinterpret_cast<const double2*>(d + off_x) + p0;
      a.out = d + off_out + (size_t)p0 * out_elem;
      a.n_points = np;
      rc = launch_prepared(a, p->precision, d_ws, nullptr, sk);
    }
    if (n_chunks > 1) {
      ok(cudaEventRecord(ev_k[c], sk), "cudaEventRecord");
      ok(cudaStreamWaitEvent(s_out, ev_k[c], 0), "cudaStreamWaitEvent");
    }
    ok(cudaMemcpyAsync(static_cast<char*>(h_out) + (size_t)p0 * out_elem, d + off_out + (size_t)p0 * out_elem,
                       (size_t)np * out_elem, cudaMemcpyDeviceToHost, sout), "device->host copy");
  }
  if (rc) {
    // a call failed part-way: work already enqueued on the side streams has no event edge to s, so drain them before
    // the scratch goes back to the pool
    if (s_in) cudaStreamSynchronize(s_in);
    if (s_k2) cudaStreamSynchronize(s_k2);
    if (s_out) cudaStreamSynchronize(s_out);
  } else if (n_chunks > 1 && ev_done && s_out) {
    cudaEventRecord(ev_done, s_out);
    cudaStreamWaitEvent(s, ev_done, 0);   // the scratch is freed in stream order of s after the last copy out
  }
  cudaFreeAsync(d, s);
  int rc2 = check_cuda(cudaStreamSynchronize(s), "stream synchronize");
  if (!rc && !rc2) rc2 = take_status("eval_grid_host");   // the call has synchronised: report what its kernels found
  if (s_in) { cudaStreamSynchronize(s_in); cudaStreamDestroy(s_in); }
  if (s_out) { cudaStreamSynchronize(s_out); cudaStreamDestroy(s_out); }
  if (s_k2) { cudaStreamSynchronize(s_k2); cudaStreamDestroy(s_k2); }
  if (ev_ready) cudaEventDestroy(ev_ready);
  if (ev_done) cudaEventDestroy(ev_done);
  for (int c = 0; c < kMaxChunks; ++c) {
    if (ev_in[c]) cudaEventDestroy(ev_in[c]);
    if (ev_k[c]) cudaEventDestroy(ev_k[c]);
  }
  return rc ? rc : rc2;
}

int gf_eval_angular(const gf_params* p, double x_re, double x_im, const double* d_ang_nodes,
                    const double* d_ang_weights, int n_ang, const void* d_y, long long n_y, void* d_out, void* stream) {
  EvalArgs a;
  int rc = build_args(p, 8, n_ang, n_y, &a);   // the radial order plays no part
  if (rc) return rc;
  if (!std::isfinite(x_re) || !std::isfinite(x_im)) { set_error("eval_angular: x is not finite"); return GF_ERR_ARG; }
  if (p->routing != 0) { set_error("eval_angular: defined for the paper's routing (eq. (22)) only"); return GF_ERR_UNSUPPORTED; }
  if (!d_ang_nodes || !d_ang_weights) { set_error("eval_angular: null table pointer"); return GF_ERR_NULL; }
  if (n_y > 0 && (!d_y || !d_out)) { set_error("eval_angular: null y/output pointer"); return GF_ERR_NULL; }
  if ((rc = take_status("eval_angular")) || (rc = attach_status(&a))) return rc;
  a.ang_nodes = d_ang_nodes;
  a.ang_weights = d_ang_weights;
  a.x = static_cast<const double2*>(d_y);
  a.out = d_out;
  return launch_angular(a, x_re, x_im, static_cast<cudaStream_t>(stream));
}

int gf_cut_crossings(const gf_params* p, const void* d_x, long long n_points, int n_z, int* d_out, void* stream) {
  EvalArgs a;
  int rc = build_args(p, 8, 2, n_points, &a);  // neither quadrature order plays a part
  if (rc) return rc;
  if (p->routing != 0) { set_error("cut_crossings: defined for the paper's routing (eq. (23)-(25)) only"); return GF_ERR_UNSUPPORTED; }
  if (n_z < 2 || n_z > (1 << 24)) { set_error("cut_crossings: n_z=%d out of range [2, 2^24]", n_z); return GF_ERR_ARG; }
  if (n_points > 0 && (!d_x || !d_out)) { set_error("cut_crossings: null grid/output pointer"); return GF_ERR_NULL; }
  a.x = static_cast<const double2*>(d_x);
  return launch_cut_crossings(a, n_z, d_out, static_cast<cudaStream_t>(stream));
}

int gf_eval_launch_info(const gf_params* p, int n_rad, int n_ang, long long n_points, gf_launch_info* out) {
  if (!out) { set_error("eval_launch_info: out is null"); return GF_ERR_NULL; }
  EvalArgs a;
  int rc = build_args(p, n_rad, n_ang, n_points, &a);
  if (rc) return rc;
  LaunchPlan plan;
  if ((rc = plan_eval(a, p->precision, &plan))) return rc;
  out->block_threads = plan.block_threads;
  out->grid_blocks = plan.grid_blocks;
  out->split = 1 << plan.split_log2;
  out->smem_bytes = (int)plan.smem_bytes;
  out->n_pairs = a.n_pairs;
  out->n_terms = a.n_terms;
  out->series_terms_max = plan.layout.kmc;
  out->evals = (double)n_points * n_rad * n_ang;
  if (a.taylor_order > 0) {   // gf_taylor.cu has no instruction model: launch shape only, the per-unit counts stay 0
    out->near_pair_dfma = out->near_pair_other = out->near_pair_fp32 = out->series_term_dfma = out->series_term_other =
        out->series_term_fp32 = out->exact_pair_dfma = out->exact_pair_other = out->node_near_dfma = out->node_near_other =
            out->node_moment_dfma = out->node_moment_other = out->node_cheb_dfma = out->node_cheb_other =
                out->node_exact_dfma = out->node_exact_other = out->tail_dfma = out->tail_other = 0.0;
    out->blk_series_dfma = out->blk_series_other = out->blk_term_dfma = out->blk_term_other = 0.0;
    return GF_OK;
  }
  // FP64-pipe instructions per unit of each route, counted per SASS region in the ncu source page of
  // eval_real_kernel<double, false, 1, true, false> (profiles/r02c_eval_ncu_full.md; DSETP not counted: no flops):
  //   pair of the plain direct loop 5 DFMA + 1 DMUL + 2 DADD, of the double-double loop 5 + 1 + 4;
  //   series term (P and N): 4 DFMA;
  //   every node-term: zeta, delta (5 DFMA + 3 DMUL + 1 DADD) and the accumulation into G (4 DFMA);
  //   MOMENT adds 4 + 5 (set-up) and 8 + 4 (finish), CHEB 14 + 18 and 8 + 4, both 2 DADD (2 Re s at the head of the
  //   FP32 and of the FP64 phase of the series loop), the direct loops 3 + 9,
  //   EXACT lanes the double-double zeta (29 + 217);
  //   tail per (point, pole): 2 DFMA per coefficient (kTailN (kTailN + 1)), 8 + 9 per n, the per-point set-up.
  const bool f32 = p->precision == 32;
  out->near_pair_dfma = f32 ? 0 : 5; out->near_pair_other = f32 ? 0 : 3; out->near_pair_fp32 = f32 ? 5 : 0;
  out->series_term_dfma = f32 ? 0 : 4; out->series_term_other = 0; out->series_term_fp32 = 4;  // per term run in FP32 (counter [9]; the FP32 variant: counter [1])
  out->exact_pair_dfma = 5; out->exact_pair_other = 5;
  out->node_near_dfma = kNodeNearDfma; out->node_near_other = kNodeNearOther;
  out->node_moment_dfma = kNodeMomentDfma; out->node_moment_other = kNodeMomentOther;
  out->node_cheb_dfma = kNodeChebDfma; out->node_cheb_other = kNodeChebOther;
  out->node_exact_dfma = kNodeNearDfma + 29; out->node_exact_other = kNodeNearOther + 217;
  out->tail_dfma = kTailN * (kTailN + 1) + 8.0 * kTailN + 45; out->tail_other = 9.0 * kTailN + 34;
  // a far block of a split rule (angular_blocked): w', its complex square root, s, the finish: 27 DFMA + 24 DMUL/DADD;
  // 2 DFMA per term of its series
  out->blk_series_dfma = 27; out->blk_series_other = 24;
  out->blk_term_dfma = 2; out->blk_term_other = 0;
  return GF_OK;
}

int gf_diag_fp64_peak(int blocks, int threads, long long iters, double* d_sink, void* stream) {
  if (!d_sink) { set_error("diag_fp64_peak: d_sink is null"); return GF_ERR_NULL; }
  if (blocks < 1 || threads < 1 || threads > 1024 || iters < 0) { set_error("diag_fp64_peak: bad launch shape"); return GF_ERR_ARG; }
  return launch_fp64_peak(blocks, threads, iters, d_sink, static_cast<cudaStream_t>(stream));
}

int gf_diag_radial_map(double cutoff2, double map_scale, const double* d_nodes, int n, double* d_y, void* stream) {
  if (!d_nodes || !d_y) { set_error("diag_radial_map: null pointer"); return GF_ERR_NULL; }
  if (n < 1 || !(cutoff2 > 0) || !(map_scale > 0)) { set_error("diag_radial_map: bad argument"); return GF_ERR_ARG; }
  double hi, lo;
  log_ratio_dd(0.0, cutoff2, map_scale, &hi, &lo);
  return launch_radial_map(hi, lo, map_scale, d_nodes, n, d_y, static_cast<cudaStream_t>(stream));
}

int gf_diag_contour_nodes(const gf_params* p, int n_rad, int n_ang, const void* d_workspace, const double* d_rad_nodes,
                          const double* d_rad_weights, double x_re, double x_im, int* d_policy, void* d_y, void* d_wy,
                          void* stream) {
  EvalArgs a;
  int rc = build_args(p, n_rad, n_ang, 1, &a);
  if (rc) return rc;
  if (p->contour == GF_CONTOUR_REAL) { set_error("diag_contour_nodes: a deformed contour policy (or AUTO) is needed"); return GF_ERR_ARG; }
  if (!d_workspace || !d_rad_nodes || !d_rad_weights || !d_policy || !d_y || !d_wy) { set_error("diag_contour_nodes: null pointer"); return GF_ERR_NULL; }
  if ((rc = attach_status(&a))) return rc;
  if (!std::isfinite(x_re) || !std::isfinite(x_im)) { set_error("diag_contour_nodes: x is not finite"); return GF_ERR_ARG; }
  LaunchPlan plan;
  if ((rc = plan_eval(a, p->precision, &plan))) return rc;
  a.rad_nodes = d_rad_nodes;
  a.rad_weights = d_rad_weights;
  return launch_contour_nodes(a, plan, static_cast<const double*>(d_workspace), x_re, x_im, d_policy,
                              static_cast<double2*>(d_y), static_cast<double2*>(d_wy), static_cast<cudaStream_t>(stream));
}

int gf_diag_dfma_issue(int mode, int blocks, int threads, long long iters, double* d_sink, void* stream) {
  if (!d_sink) { set_error("diag_dfma_issue: d_sink is null"); return GF_ERR_NULL; }
  if (mode < 0 || mode > 3 || blocks < 1 || threads < 1 || threads > 1024 || iters < 0) { set_error("diag_dfma_issue: bad mode or launch shape"); return GF_ERR_ARG; }
  return launch_dfma_issue(mode, blocks, threads, iters, d_sink, static_cast<cudaStream_t>(stream));
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// gf_eval_grid_static: gf_eval_grid for callers that cannot allocate (code under CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  The workspace of the prepared tables is a file-scope device array of
// GF_STATIC_WORKSPACE_BYTES that every GPU loading this library holds until the process exits; the entry point calls
// no cudaMalloc / cudaFree / pool routine and no mapped host word (status = NULL: bad tables show as NaN results only).
// In host code the array's NAME is a host-side stand-in, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_static_workspace[GF_STATIC_WORKSPACE_BYTES / sizeof(double)];

// Device code may name the array directly.  The header (status bits of the tables, hash tag) is what a kernel reads
// first from a workspace: it starts every call at zero, whatever the last call left there.
static __global__ void static_workspace_reset_kernel() {
  g_static_workspace[0] = 0.0;
  g_static_workspace[1] = 0.0;
}

static double* g_static_ptr[64] = {};
static std::mutex g_static_mutex;

static int static_workspace(double** ptr) {
  int dev = 0;
  int rc = check_cuda(cudaGetDevice(&dev), "cudaGetDevice");
  if (rc) return rc;
  if (dev < 0 || dev >= 64) { set_error("device ordinal %d out of range", dev); return GF_ERR_CUDA; }
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    double* d = nullptr;
    if ((rc = check_cuda(cudaGetSymbolAddress(reinterpret_cast<void**>(&d), g_static_workspace),
                         "cudaGetSymbolAddress(static workspace)")))
      return rc;
    if (!d) { set_error("eval_grid_static: the static workspace has no device address"); return GF_ERR_CUDA; }
    g_static_ptr[dev] = d;
  }
  *ptr = g_static_ptr[dev];
  return GF_OK;
}

extern "C" int gf_eval_grid_static(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                                   const double* d_ang_nodes, const double* d_ang_weights, int n_ang, const void* d_x,
                                   long long n_points, void* d_out, void* stream) {
  return no_throw("eval_grid_static", [&] {
    EvalArgs a;
    int rc = build_args(p, n_rad, n_ang, n_points, &a);
    if (rc) return rc;
    if (!d_rad_nodes || !d_rad_weights || !d_ang_nodes || !d_ang_weights) { set_error("eval_grid_static: null table pointer"); return (int)GF_ERR_NULL; }
    if (n_points > 0 && (!d_x || !d_out)) { set_error("eval_grid_static: null grid/output pointer"); return (int)GF_ERR_NULL; }
    LaunchPlan plan;
    if ((rc = plan_eval(a, p->precision, &plan))) return rc;
    const long long need = (long long)plan.layout.n_total * (long long)sizeof(double);
    if (need > (long long)GF_STATIC_WORKSPACE_BYTES) {
      set_error("eval_grid_static: these parameters and orders need a workspace of %lld bytes; the static workspace "
                "holds GF_STATIC_WORKSPACE_BYTES = %lld (use gf_eval_grid, or gf_eval_prepare with a workspace of the caller's)",
                need, (long long)GF_STATIC_WORKSPACE_BYTES);
      return (int)GF_ERR_ARG;
    }
    if (n_points == 0) return (int)GF_OK;
    double* blob = nullptr;
    if ((rc = static_workspace(&blob))) return rc;
    a.status = nullptr;
    a.rad_nodes = d_rad_nodes;
    a.rad_weights = d_rad_weights;
    a.ang_nodes = d_ang_nodes;
    a.ang_weights = d_ang_weights;
    a.x = static_cast<const double2*>(d_x);
    a.out = d_out;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    static_workspace_reset_kernel<<<1, 1, 0, s>>>();
    if ((rc = check_cuda(cudaGetLastError(), "static workspace reset launch"))) return rc;
    if ((rc = launch_prepare(a, p->precision, blob, s))) return rc;
    return launch_prepared(a, p->precision, blob, nullptr, s);
  });
}
