/* gf.h -- C ABI of libgf_b200: complex-plane scans of regularised one-loop integrals on B200.
 *
 * The data-parallel hot path of arXiv:1205.0752 (Windisch, Alkofer, Haase, Liebmann,
 * "Examining the Analytic Structure of Green's Functions: Massive Parallel Complex Integration
 * using GPUs"), citations are lines of the paper text PAPER.md:
 *
 *   for every point x = p^2 of a grid in the complex plane (Step 4) evaluate
 *
 *     G(x) = c0 * int_C dy y  int_-1^1 dz sqrt(1-z^2)  F_sub(x, y, sqrt(x) sqrt(y) z)     eq. (14)/(15)
 *
 *   by non-adaptive quadrature (Step 5), where F = D1(y) D2(u),
 *   u = x + y - 2 sqrt(x) sqrt(y) z = (p-k)^2 (eq. (10),(19)), and F_sub = (1 - t^0) F is the
 *   BPHZ-like Taylor-subtracted integrand (eq. (12),(13),(20)).  Every grid point is independent.
 *
 * Conventions
 *   - All entry points are extern "C", return a gf_status, and never throw.
 *   - "d_" arguments are DEVICE pointers (CUDA global memory of the current device), "h_"
 *     arguments are HOST pointers.  `stream` is a cudaStream_t passed as void* (NULL = the
 *     legacy default stream).  Unless stated otherwise a call only ENQUEUES work on `stream`
 *     and returns; the caller synchronises.
 *   - Ownership: the caller owns every buffer.  Scratch a call needs is taken from, and returned
 *     (in stream order, before the call returns) to, a stream-ordered memory pool of the library's
 *     own, one per device; the pool keeps freed blocks for the next call until gf_trim_scratch().
 *     Nothing else outlives a call.
 *   - Complex arrays are interleaved (re, im) pairs: complex<double> = 2 doubles (16 bytes,
 *     16-byte aligned), complex<float> = 2 floats (8 bytes, 8-byte aligned).
 *   - Grids are stored [n_im][n_re], the real index fastest (the paper's X(M,N) with M along
 *     the real axis, Fortran order).
 *   - Errors: GF_ERR_NULL for a null pointer, GF_ERR_ARG for a value out of range,
 *     GF_ERR_UNSUPPORTED for a combination the method does not define or that is not built (taylor_order outside
 *     [0, 4], taylor_order > 0 with the symmetric routing or with precision 32, a
 *     subtraction point other than 0, the symmetric routing with unequal or rational lines, the THREAD contour
 *     with unequal or complex masses, a rational propagator with a double pole, precision 32 on a
 *     contour other than REAL), GF_ERR_CUDA when the CUDA runtime reports an error (no device,
 *     launch failure).  gf_last_error() describes the last failure of the
 *     calling thread.  A denominator that vanishes at a quadrature node yields IEEE inf/NaN in
 *     that output entry, not an error (the paper has no convention).
 *   - Bad input that only a kernel can see (tables in DEVICE memory: an angular rule that is not symmetric, radial
 *     nodes that are not ascending strictly inside (-1,1); a workspace that was prepared for other parameters): the
 *     kernel fills every output of that call with NaN and leaves a code in a mapped host word of the device; the
 *     NEXT call of gf_eval_grid / _counted / _host, gf_eval_prepare, gf_eval_grid_prepared or gf_eval_angular on
 *     that device (after the kernel has run) does nothing, returns GF_ERR_ARG and names the cause, once.
 *     gf_eval_grid_host checks its (host) tables before it launches anything and reports what its own kernels found
 *     before it returns.
 */
#ifndef GF_B200_H_
#define GF_B200_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { GF_OK = 0, GF_ERR_NULL = 1, GF_ERR_ARG = 2, GF_ERR_UNSUPPORTED = 3, GF_ERR_CUDA = 4 } gf_status;

/* Quadrature rules on [-1,1]: Gauss-Legendre (the paper's radial rule, and the
 * angular rule of BASELINE.json's configs), Gauss-Chebyshev of the 2nd kind (the paper's check
 * rule; the exact Gauss rule for the d=4 angular measure), tanh-sinh (the paper's angular rule). */
typedef enum { GF_QUAD_GAUSS_LEGENDRE = 0, GF_QUAD_GAUSS_CHEB2 = 1, GF_QUAD_TANH_SINH = 2,
               GF_QUAD_GAUSS_CHEB1 = 3 /* first kind: the exact Gauss rule of the d = 2 angular measure */ } gf_quad_kind;

/* Which measure the returned weights integrate against: dz (radial rules), or the d=4
 * hyperspherical angular measure sqrt(1-z^2) dz of eq. (9)/(11). */
typedef enum { GF_MEASURE_PLAIN = 0, GF_MEASURE_SQRT1MZ2 = 1 } gf_measure;

/* Propagators.  MASSIVE: 1/(u + m2), m2 complex (the paper's example uses m2 = +-i/2, eq. (19)).
 * RATIONAL: (u + M2)/(u^2 + a u + b) with real M2, a, b (BASELINE.json config 4). */
typedef enum { GF_PROP_MASSIVE = 0, GF_PROP_RATIONAL = 1 } gf_prop_kind;
typedef struct {
  int kind;            /* gf_prop_kind */
  double m2_re, m2_im; /* MASSIVE */
  double M2, a, b;     /* RATIONAL */
} gf_propagator;

/* Radial contour C of eq. (15) (Step 3), chosen per grid point inside the
 * evaluation kernel like the IF-THEN-ELSE of the paper's Kernel 2:
 *   REAL     the positive real axis [0, Lambda^2] of eq. (14);
 *   RAY_ARC  ray along arg x, arc back to the real axis, real tail (generalises the paper's
 *            region-2/5 contour);
 *   THREAD   polyline through the opening of the cut for Re x < -4 m^2 next to the negative
 *            axis, equal real masses only (analogue of the region-3/4 contours);
 *   AUTO     per-point choice among the three.
 * Geometry (no angle is ever formed; every operation below is one correctly rounded +, -, *, /, sqrt in the order
 * written, so the nodes are the same doubles on any IEEE machine).  sc = |m2^2| of line 2 (largest pole modulus for
 * a rational line); dir = x/|x| with x scaled by a power of two first (two divisions); tau = tan(phi/4) of dir =
 * (cos phi, sin phi) by half-angle formulas (ch = sqrt((1+c)/2), sh = (s/2)/ch for c >= 0, else sh = +-sqrt((1-c)/2),
 * ch = (|s|/2)/|sh|; tau = sh/(1+ch)).  Ladder of contour radii: {2^k, 1.5 2^k}, starting one rung below the smallest
 * rung >= 1.5 sc; rung(v) = the smallest rung >= v, or Lambda^2/2 when that rung is more than 64 rungs up the ladder
 * or not below Lambda^2/2.
 *   RAY_ARC  = ray r dir, r in [0,R] shifted-log, n_rad/2 nodes; arc y(v) = R ((1 + i tau v)/(1 - i tau v))^2,
 *              v = 1 - u: 1 -> 0, with dy/du = -4 i tau y/(1 + tau^2 v^2), n_rad/4; real [R, Lambda^2] shifted-log,
 *              n_rad/4; R = rung(1.5 (sqrt|x| + sqrt(|x|+sc))^2).
 *   THREAD   (Im x >= 0, mirrored otherwise; s = |x|, |A| = (sqrt s - m)^2, |B| = (sqrt s + m)^2, r0 = |x + m^2|)
 *              straight pieces 0 -> -m^2 + i(|A|-m^2)/2 -> (|A|+m^2)/2 dir -> -(|A|+r0)/2 - i(r0-|A|)/2
 *              -> r0 dir -> R e^{3 pi i/4} (the arc's v = 1 end with tau = tan(3 pi/16)), arc to R, n_rad/8 nodes
 *              each; real [R, Lambda^2], n_rad/4; R = rung(1.5 |B|).
 *   AUTO     with c2 = min over the poles -mu of line 2 of (Re sqrt(mu))^2 = (|mu| + Re mu)/2 and the parabola
 *              P(c) = {Re x + c > 0, (Im x)^2 < 4 c (Re x + c)} (REAL is the continuation exactly inside P(c2),
 *              PAPER.md:270), tested in this order:
 *              1. x in P(c2/2): REAL (exact there and the cheapest);
 *              2. Re x < 0, |Im x| n_rad < 80 |Re x| and x in P(c2): REAL (next to the negative axis the ray of
 *                 RAY_ARC passes the pole of line 1 closer than the radial rule resolves);
 *              3. x in the wedge W = {Re x < -sc, |Im x| n_ang sc < 5 |x|^2}: THREAD if it applies and
 *                 Re x <= -4.1 sc, else REAL;
 *              4. RAY_ARC.
 *            Limitation: in case 3 with REAL (next to the negative axis between the parabola and -4.1 sc, e.g. the
 *            strip -4 m^2 < Re x < -m^2 of the equal-mass bubble, and for lines THREAD does not apply to) the value
 *            is bounded and reproducible but NOT the analytic continuation: no contour of this library reaches it.
 * Every piece carries the Gauss-Legendre rule of its order from the pyramid of gf_radial_table_size().
 * The restructured evaluation (pole sum, folded angular sum, series) needs propagators that are sums of simple
 * poles, which MASSIVE and RATIONAL are; it does not extend to a general integrand F(x, y, z) of PAPER.md:43. */
typedef enum { GF_CONTOUR_REAL = 0, GF_CONTOUR_RAY_ARC = 1, GF_CONTOUR_THREAD = 2, GF_CONTOUR_AUTO = 3 } gf_contour;

typedef enum { GF_SPACING_UNIFORM = 0, GF_SPACING_LOG_ABS_IM = 1 } gf_spacing;

typedef struct {
  gf_propagator line_k;  /* D1(y): the line carrying k      (eq. (19)) */
  gf_propagator line_pk; /* D2(u): the line carrying p - k */
  double cutoff2;        /* Lambda^2 in (0, 1e60], upper limit of the radial integral */
  double sub_re, sub_im; /* subtraction point x0 of t^n; only 0 is supported (eq. (13)) */
  int taylor_order;      /* n of the Taylor subtraction t^n of eq. (12),(13), 0 <= n <= 4.  0 is the
                            paper's worked example (log-divergent integrals).  "x = 0" in eq. (13) is
                            p = 0 (eq. (20) sets the scalar product to zero with x): t^n is the Taylor operator in the
                            external momentum, x^i standing for the order 2i in p, so (1 - t^n) F is F minus every
                            term of its expansion in p up to the order 2n and G_n = G - sum_{i<=n} x^i G^(i)(0)/i! =
                            O(x^(n+1)).  n > 0: any contour policy, the paper's routing, precision 64 (any dim on REAL) */
  double prefactor;      /* c0; 1/(2 pi)^3 is eq. (14), 2/pi the rescaled eq. (21) */
  double map_scale;      /* s0 > 0 of the shifted-log radial map y(u) = a + (a+s0) expm1(u L) */
  int contour;           /* gf_contour */
  int precision;         /* 64: complex<double> output (the contract); 32: the FP32 comparison
                            variant, complex<float> output */
  int routing;           /* 0: the paper's eq. (19), the lines carry k and p - k.  1: symmetric, the lines carry
                            k + p/2 and k - p/2 (the integral is shift invariant, eq. (4)): equal massive
                            lines only, taylor_order 0; G agrees up to O(x/Lambda^2), and REAL is the
                            continuation inside the parabola through the threshold, Re x > (Im x)^2/(16 m^2) - 4 m^2,
                            instead of Re x > (Im x)^2/(4 m^2) - m^2.  Its cut in the y-plane is the paper
                            routing's at x/4, so the deformed contours (RAY_ARC, THREAD, AUTO) are those of x/4 */
  double dim;            /* space-time dimension d in [1, 8], 0 meaning 4 ("arbitrary dimensions by
                            trivial modifications"): the radial measure becomes dy y^((d-2)/2); the angular measure
                            (1-z^2)^((d-3)/2) is the caller's, in the angular weights (gf_make_quadrature_dim makes them;
                            GF_MEASURE_PLAIN is d = 3).
                            On a deformed contour y^((d-2)/2) is taken on the branch continued along the contour
                            from y = 0 (|y|^p e^(i p arg y), arg y = arg x on the ray, running past pi on THREAD's
                            pieces under the negative real axis).  Constants of the d-dimensional measure go into
                            `prefactor` (d^dk = 1/2 y^((d-2)/2) dy dOmega_d). */
} gf_params;

/* Step 4 / Kernel 1: fill d_x[n_im][n_re] (complex<double>) with the
 * homogeneous, endpoint-inclusive distribution of points over [re_min,re_max] x [im_min,im_max].
 * Each axis is two-sided: v_i = min + i*d for 2i <= n-1 and max - (n-1-i)*d above, d = (max-min)/(n-1),
 * each with one fused multiply-add, so a range symmetric about 0 is mirrored exactly.  n = 1 gives min.
 * GF_SPACING_LOG_ABS_IM (n_im even, im_min == -im_max, 0 < im_abs_min < im_max): |Im x| takes n_im/2
 * log-spaced values from im_abs_min to im_max on each side of the real axis, ascending in Im x.
 * Asynchronous on `stream`. */
int gf_make_grid(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
                 int spacing, double im_abs_min, void* d_x, void* stream);

/* Rows [row_first, row_first + n_rows) of the same grid into d_x[n_rows][n_re], bit-identical to the
 * corresponding rows of gf_make_grid.  This is the multi-GPU partition: grid
 * points are independent, each rank owns a contiguous block of rows, no exchange.
 * n_rows = 0 is a no-op. */
int gf_make_grid_rows(double re_min, double re_max, int n_re, double im_min, double im_max, int n_im,
                      int spacing, double im_abs_min, int row_first, int n_rows, void* d_x, void* stream);

/* "Preparation": nodes t_i in (-1,1), ascending, and weights of an n-point rule
 * into caller-allocated DEVICE arrays of n doubles each.  Tables are computed on the host in extended
 * precision (as in the paper) and copied with cudaMemcpyAsync on `stream`; the host staging copy is
 * complete on return.  `step` is the tanh-sinh step h (0 = default 2.9/((n-1)/2)); ignored otherwise.
 * `measure` is a gf_measure.  Rules are exactly symmetric: t[n-1-i] == -t[i], w[n-1-i] == w[i]. */
int gf_make_quadrature(int kind, int n, double step, int measure, double* d_nodes, double* d_weights,
                       void* stream);

/* The same tables into HOST arrays (no CUDA call is made). */
int gf_make_quadrature_host(int kind, int n, double step, int measure, double* h_nodes, double* h_weights);

/* The angular rule of `dim` space-time dimensions ("arbitrary dimensions by trivial modifications"): nodes
 * of rule `kind` and weights that integrate against (1 - z^2)^((dim-3)/2) dz, dim in [1, 8] -- what gf_params.dim
 * expects in the angular weights.  The paper uses "Gauss-Chebyshev ... polynomials of the first and second kind ...
 * depending on the dimension": GF_QUAD_GAUSS_CHEB1 is the exact Gauss rule of dim = 2 (z_j =
 * cos((2j-1) pi/2n), weights pi/n), GF_QUAD_GAUSS_CHEB2 of dim = 4, GF_QUAD_GAUSS_LEGENDRE of dim = 3; for another dim
 * the remaining power of (1 - z^2) = sin^2(theta) goes into the weights.  dim = 3 and dim = 4 give the tables of
 * gf_make_quadrature with GF_MEASURE_PLAIN and GF_MEASURE_SQRT1MZ2 bit for bit.  Otherwise as gf_make_quadrature. */
int gf_make_quadrature_dim(int kind, int n, double step, double dim, double* d_nodes, double* d_weights, void* stream);
int gf_make_quadrature_dim_host(int kind, int n, double step, double dim, double* h_nodes, double* h_weights);

/* Doubles needed for the radial tables of a contour policy: n_rad for REAL; for the other policies
 * the pyramid n_rad + n_rad/2 + n_rad/4 + n_rad/8 (rules of those orders back to back -- the paper's
 * "n arrays for the radial nodes"), which requires n_rad % 8 == 0.  Returns -1 on error. */
long long gf_radial_table_size(int contour, int n_rad);

/* Step 5 / Kernel 2: G at every point of d_x.
 *   d_rad_nodes/d_rad_weights  radial rule(s), measure PLAIN, gf_radial_table_size() doubles each;
 *                              nodes ascending, strictly inside (-1,1) (every level of the pyramid; the tail series
 *                              and its binary search rely on the order)
 *   d_ang_nodes/d_ang_weights  angular rule of n_ang nodes whose weights include the measure
 *                              sqrt(1-z^2) (GF_MEASURE_SQRT1MZ2).  The rule must be symmetric
 *                              (z[n-1-j] = -z[j], equal weights): the kernel folds +-z pairs.  A rule
 *                              that is not makes every output NaN (and see "Bad input" above).
 *   d_x      n_points complex<double>
 *   d_out    n_points complex<double> (precision 64) or complex<float> (precision 32; REAL contour only)
 * Domain: x = 0 gives exactly 0; |x| up to 1e100.  Asynchronous on `stream`; n_points = 0 is a no-op. */
int gf_eval_grid(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                 const double* d_ang_nodes, const double* d_ang_weights, int n_ang, const void* d_x,
                 long long n_points, void* d_out, void* stream);

/* gf_eval_grid for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same arguments, the same kernels, the same results, but the workspace of the prepared tables
 * is a static device array of GF_STATIC_WORKSPACE_BYTES inside the library instead of stream-ordered scratch.  It calls
 * no cudaMalloc, cudaFree, memory-pool or host-allocation routine.
 *   Limit: parameters and orders whose gf_eval_workspace_size() exceeds GF_STATIC_WORKSPACE_BYTES are refused with
 *          GF_ERR_ARG and a message that names both sizes (the configs of this repository need 0.2 to 26 MiB).
 *   Cost:  every GPU that loads the library holds the array until the process exits.
 *   First call: looks up the array's device address (cudaGetSymbolAddress, once per device) and may set a kernel's
 *          shared-memory attribute; make one call per device outside a stream capture before capturing calls.
 *   Sharing: every call on a device uses the same array, which keeps the last call's tables (each call rewrites all
 *          it reads and resets the header first).  Calls that OVERLAP on the GPU (two streams, two host threads) race on
 *          it: issue them on one stream, or order them with events.  Other devices have their own copy.
 *   Errors: as gf_eval_grid, except that bad TABLES (an asymmetric angular rule, radial nodes out of order) show as NaN
 *          results only: this entry point does not use the mapped status word of "Bad input" above (it would have to
 *          allocate it).  precision 32 / 64, every contour policy, routing, dim and taylor_order as gf_eval_grid. */
#define GF_STATIC_WORKSPACE_BYTES (32ll << 20)
int gf_eval_grid_static(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                        const double* d_ang_nodes, const double* d_ang_weights, int n_ang, const void* d_x,
                        long long n_points, void* d_out, void* stream);

/* The two halves of gf_eval_grid, for callers that evaluate several grids with the same parameters and rules
 * (and for benchmarks that time the evaluation kernel alone).  gf_eval_prepare makes every table that does not
 * depend on x (folded angular rule, series coefficients, radial nodes and prefactors, tail tables) into the
 * caller's DEVICE workspace of gf_eval_workspace_size() bytes (256-byte aligned; -1 on a bad argument; it does not
 * depend on the number of points).  gf_eval_grid_prepared evaluates d_x from such a workspace; params, n_rad and
 * n_ang must be the ones it was prepared with: the workspace header carries a hash of them, and the kernels read
 * nothing else from a workspace whose hash differs (outputs NaN, "Bad input" above).  d_counters may be NULL (else as in
 * gf_eval_grid_counted).  gf_eval_grid == workspace from cudaMallocAsync + these two + cudaFreeAsync. */
long long gf_eval_workspace_size(const gf_params* p, int n_rad, int n_ang);
int gf_eval_prepare(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                    const double* d_ang_nodes, const double* d_ang_weights, int n_ang, void* d_workspace,
                    void* stream);
int gf_eval_grid_prepared(const gf_params* p, int n_rad, int n_ang, const void* d_workspace, const void* d_x,
                          long long n_points, void* d_out, unsigned long long* d_counters, void* stream);

/* The same call on HOST buffers (the end-to-end path): allocates device scratch on `stream`, copies
 * tables and x host->device, runs the kernels, copies the result device->host and synchronises
 * `stream` before returning.  Pinned host memory makes the copies asynchronous but is not required. */
int gf_eval_grid_host(const gf_params* p, const double* h_rad_nodes, const double* h_rad_weights, int n_rad,
                      const double* h_ang_nodes, const double* h_ang_weights, int n_ang, const void* h_x,
                      long long n_points, void* h_out, void* stream);

/* Paper Kernel 3 (Fig. 1): the angular integral B of eq. (22) for ONE x = (x_re, x_im) at
 * n_y complex y (d_y, interleaved),
 *     B(x, y) = sum_j w'_j [ D2(u_j) - D2(y) ] / D2(y),   u_j = x + y - 2 sqrt(x) sqrt(y) z_j,
 * which for a massive line 2 is eq. (22)'s  int dz sqrt(1-z^2) (-x + 2 sqrt(x) sqrt(y) z)/(u + m2^2).  Only
 * p->line_pk is used (line_k, cutoff2, contour play no part but must be valid); the angular rule as in
 * gf_eval_grid.  d_out: n_y complex<double>.  x = 0 gives exactly 0; y = 0 is the limit value; where 4 x y
 * overflows or underflows the entry is IEEE inf/NaN.  Accuracy: 1e-11 relative where |B| is of the order of the sum
 * of the weights; where B is small by cancellation (|x|, |y| >> |m2|: the rule nearly integrates the numerator to
 * zero) the error is absolute, about 1e-14 of the sum of the weights (2e-10 relative was the worst of 8 000 random
 * (x, y, line 2, rule) against the oracle in binary128).  FP64 only.  Asynchronous on `stream`. */
int gf_eval_angular(const gf_params* p, double x_re, double x_im, const double* d_ang_nodes,
                    const double* d_ang_weights, int n_ang, const void* d_y, long long n_y, void* d_out, void* stream);

/* Paper Kernel 4 (Fig. 2): for every x of d_x (n_points complex<double>), how often the branch
 * cut(s) that the angular integral induces in the y-plane cross the original contour (0, Lambda^2] of the real
 * y-axis; 0 means the contour "remains unharmed".  Procedure (reading G19; the paper does not give
 * one): per pole -mu of line 2 the cut y(z) = (sqrt(x) z + i s(z))^2, s(z) = sqrt(x (1 - z^2) + mu) (eq. (23)-(25)),
 * sampled at n_z equidistant z in [-1, 1] with s continued from sample to sample; a crossing is counted where
 * Im y changes sign between neighbours and the linearly interpolated Re y is in (0, Lambda^2].  Every step is a
 * correctly rounded real operation in a fixed order: the result is bit-identical to the oracle's.
 * d_out: n_points 32-bit integers.  Asynchronous on `stream`. */
int gf_cut_crossings(const gf_params* p, const void* d_x, long long n_points, int n_z, int* d_out, void* stream);

/* The same evaluation, also counting the work by route for the roofline accounting.
 * d_counters: 13 unsigned 64-bit DEVICE counters the kernel ADDS to (zero them first):
 *   [0] pairs of the plain direct loop  [1] series terms EXECUTED in FP64 (every lane of a warp runs its warp's
 *   longest series; the FP64 kernel runs the high-order terms of a series, whose sum is below 2^-24 of the budget,
 *   in FP32: those are counter [9])  [2] pairs of the double-double direct loop (EXACT lanes, and the NEAR lanes of their warps)
 *   [3] [4] [5] [6] (point, radial node, pole) triples taken by the NEAR / MOMENT / EXACT / CHEB
 *   route (the triples of the large-y tail are not among them)  [7] series terms NEEDED (the sum over series
 *   triples of their own K)  [8] tail series evaluated, one per (point, pole)  [9] series terms executed in
 *   FP32 by the FP64 kernel  [10] far blocks of the angular rule summed by their own series on the NEAR / EXACT
 *   routes (rules of 128 and more folded pairs, 192 on the deformed contours, are split into a binary tree of blocks
 *   whose leaves hold 32 pairs; counters [0] and [2] then count only the pairs of the leaves next to zeta)  [11] terms
 *   of those block series  [12] leaves covered by them (a block of level l covers 2^l).  Results are identical to
 *   gf_eval_grid. */
int gf_eval_grid_counted(const gf_params* p, const double* d_rad_nodes, const double* d_rad_weights, int n_rad,
                         const double* d_ang_nodes, const double* d_ang_weights, int n_ang, const void* d_x,
                         long long n_points, void* d_out, unsigned long long* d_counters, void* stream);

/* How gf_eval_grid would launch, and the FP64-pipe instructions per unit of work of each route (for benchmarks
 * and roofline numbers; makes no CUDA call).  Per unit: *_dfma counts DFMA (2 flops each), *_other counts
 * DMUL + DADD (1 flop each), *_fp32 FP32-pipe instructions (precision 32); they follow the SASS of the loops
 * (DESIGN.md "Instruction counts").  Executed instructions per launch = sum over routes of
 * (gf_eval_grid_counted's counters) x (these). */
typedef struct {
  int block_threads;      /* threads per CTA */
  long long grid_blocks;  /* CTAs */
  int split;              /* lanes sharing one grid point (radial nodes dealt round-robin) */
  int smem_bytes;         /* dynamic shared memory per CTA */
  int n_pairs;            /* folded angular nodes: ceil(n_ang/2) */
  int n_terms;            /* simple-pole terms of line 2 (1 massive, 2 rational) */
  int series_terms_max;   /* longest series (coefficients staged per table) */
  double evals;           /* nominal integrand evaluations: n_points * n_rad * n_ang */
  double near_pair_dfma, near_pair_other, near_pair_fp32;         /* per NEAR pair */
  double series_term_dfma, series_term_other, series_term_fp32;   /* per executed series term */
  double exact_pair_dfma, exact_pair_other;                       /* per EXACT pair */
  double node_near_dfma, node_near_other;                         /* per (point, node, pole) by route: set-up + finish */
  double node_moment_dfma, node_moment_other;
  double node_cheb_dfma, node_cheb_other;
  double node_exact_dfma, node_exact_other;
  double tail_dfma, tail_other;                                   /* per tail series (point, pole) */
  double blk_series_dfma, blk_series_other;                       /* per far block: set-up + finish of its series */
  double blk_term_dfma, blk_term_other;                           /* per term of a block series */
} gf_launch_info;
int gf_eval_launch_info(const gf_params* p, int n_rad, int n_ang, long long n_points, gf_launch_info* out);

/* Diagnostics used by bench.py to measure the denominators it reports against (not on the hot path).
 * gf_diag_fp64_peak: enqueue a kernel of `blocks` x `threads` threads, each running `iters` rounds of 8
 *   independent DFMA chains (16*iters flops per thread per round... see DESIGN.md); writes one double
 *   per thread to d_sink (blocks*threads doubles) so the work cannot be removed.
 * gf_diag_dfma_issue: the same launch shape and sink, 8 DFMA per thread and round as well, with the operand pattern
 *   `mode` selects: 0 one varying register pair per DFMA (a = fma(a, m, c), m and c loop-invariant), 1 two varying
 *   pairs, 2 three varying pairs (a_j = fma(a_j, b_j, c_j)), 3 the second-order recurrence of the series routes
 *   (t = fma(ns, p2, c); p2 = fma(r, p1, t)) on four chains.  The ratio of the measured times is the issue cadence
 *   of each pattern relative to the peak stream. */
int gf_diag_fp64_peak(int blocks, int threads, long long iters, double* d_sink, void* stream);
int gf_diag_dfma_issue(int mode, int blocks, int threads, long long iters, double* d_sink, void* stream);
/* The radial nodes y_i = s0 expm1(u_i L), u_i = (t_i + 1)/2, L = ln((cutoff2 + s0)/s0), of the REAL contour
 * exactly as the evaluation kernel makes them (double-double, correctly rounded), for the n rule nodes in
 * d_nodes; tests compare them bit for bit with the oracle's. */
int gf_diag_radial_map(double cutoff2, double map_scale, const double* d_nodes, int n, double* d_y, void* stream);
/* The n_rad nodes of the contour of the one point x = (x_re, x_im) under a deformed policy (RAY_ARC, THREAD, AUTO)
 * exactly as the evaluation kernel walks them, read from the workspace gf_eval_prepare() made for the same
 * (p, rules, orders): d_policy[0] = the policy taken (gf_contour), d_y[g] = y_g, d_wy[g] = (rule weight) x dy/dt
 * (complex<double>, n_rad each; the weights are re-derived and good to a few ulp).  Tests compare y bit for bit with
 * the oracle's. */
int gf_diag_contour_nodes(const gf_params* p, int n_rad, int n_ang, const void* d_workspace, const double* d_rad_nodes,
                          const double* d_rad_weights, double x_re, double x_im, int* d_policy, void* d_y, void* d_wy,
                          void* stream);

/* Return the cached scratch of every device's pool to the driver (blocks still in use by enqueued work stay). */
int gf_trim_scratch(void);

const char* gf_last_error(void);
const char* gf_version(void);
/* Hash of the sources this binary was compiled from (paper_1205_0752_b200/build.py source_id()); the Python binding
 * refuses a library whose id differs from that of the sources beside it.  "" when built by other means. */
const char* gf_build_id(void);

#ifdef __cplusplus
}
#endif
#endif /* GF_B200_H_ */
