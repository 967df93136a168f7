// gf_dd.cuh -- double-double arithmetic for the two places of the CUDA path that need more than 53
// bits: the radial map y_i = s0 expm1(u_i L) of the REAL contour (correctly rounded, so that the node
// positions do not depend on the device's libm; reading G18) and the accurate evaluation of
// zeta - t next to a singularity of the integrand.  Error-free transformations after Dekker/Knuth;
// every rounding that matters is written with the _rn intrinsics so that no contraction can touch it.
#pragma once

namespace gf {

struct dd {
  double hi, lo;
};

__device__ __forceinline__ dd two_sum(double a, double b) {
  const double s = __dadd_rn(a, b);
  const double bb = __dadd_rn(s, -a);
  const double e = __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb));
  return {s, e};
}
// requires |a| >= |b| (or a == 0)
__device__ __forceinline__ dd quick_two_sum(double a, double b) {
  const double s = __dadd_rn(a, b);
  const double e = __dadd_rn(b, -__dadd_rn(s, -a));
  return {s, e};
}
__device__ __forceinline__ dd two_prod(double a, double b) {
  const double p = __dmul_rn(a, b);
  return {p, __fma_rn(a, b, -p)};
}
__device__ __forceinline__ dd dd_neg(dd a) { return {-a.hi, -a.lo}; }
__device__ __forceinline__ dd dd_add(dd a, dd b) {
  dd s = two_sum(a.hi, b.hi);
  const dd t = two_sum(a.lo, b.lo);
  s.lo = __dadd_rn(s.lo, t.hi);
  s = quick_two_sum(s.hi, s.lo);
  s.lo = __dadd_rn(s.lo, t.lo);
  return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_add_d(dd a, double b) {
  dd s = two_sum(a.hi, b);
  s.lo = __dadd_rn(s.lo, a.lo);
  return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
  dd p = two_prod(a.hi, b.hi);
  p.lo = __dadd_rn(p.lo, __fma_rn(a.hi, b.lo, __dmul_rn(a.lo, b.hi)));
  return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b) {
  dd p = two_prod(a.hi, b);
  p.lo = __fma_rn(a.lo, b, p.lo);
  return quick_two_sum(p.hi, p.lo);
}
// exact scaling by a power of two
__device__ __forceinline__ dd dd_scale2(dd a, double pow2) { return {a.hi * pow2, a.lo * pow2}; }
__device__ __forceinline__ dd dd_div_d(dd a, double b) {
  const double q1 = __ddiv_rn(a.hi, b);
  dd r = dd_add(a, dd_neg(two_prod(q1, b)));
  const double q2 = __ddiv_rn(r.hi, b);
  r = dd_add(r, dd_neg(two_prod(q2, b)));
  const double q3 = __ddiv_rn(r.hi, b);
  return dd_add_d(quick_two_sum(q1, q2), q3);
}
__device__ __forceinline__ dd dd_div(dd a, dd b) {
  const double q1 = __ddiv_rn(a.hi, b.hi);
  dd r = dd_add(a, dd_neg(dd_mul_d(b, q1)));
  const double q2 = __ddiv_rn(r.hi, b.hi);
  r = dd_add(r, dd_neg(dd_mul_d(b, q2)));
  const double q3 = __ddiv_rn(r.hi, b.hi);
  return dd_add_d(quick_two_sum(q1, q2), q3);
}

// expm1(v) for a double-double 0 <= v < 700, relative error ~1e-30:
// v = k ln2 + r, |r| <= ln2/2; exp(r/512) - 1 by its Taylor series (10 terms), nine squarings in the
// expm1 form p <- 2p + p^2, then 2^k (1 + p) - 1.
__device__ inline dd dd_expm1(dd v) {
  const dd ln2 = {6.93147180559945286227e-01, 2.31904681384629955842e-17};
  const double k = rint(v.hi * 1.4426950408889634074);
  dd r = dd_add(v, dd_neg(dd_mul_d(ln2, k)));
  r = dd_scale2(r, 1.0 / 512.0);
  dd p = dd_div_d(r, 10.0);
  for (int n = 9; n >= 1; --n) p = dd_div_d(dd_mul(dd_add_d(p, 1.0), r), (double)n);
  for (int s = 0; s < 9; ++s) p = dd_add(dd_scale2(p, 2.0), dd_mul(p, p));
  if (k == 0.0) return p;
  const double sc = scalbn(1.0, (int)k);
  return dd_add_d(dd_scale2(dd_add_d(p, 1.0), sc), -1.0);
}

}  // namespace gf
