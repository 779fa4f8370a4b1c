// dd_arith.cuh — double-double arithmetic for the precision-fallback kernel (O8, step a8;
// PAPER.md:91 "arithmetic with different precisions"). Error-free transformations with FMA
// (two_sum / two_prod); ~106-bit significand. Device only.
#pragma once
#include <cuda_runtime.h>

struct dd {
  double hi, lo;
  __device__ __forceinline__ dd() {}
  __device__ __forceinline__ dd(double h) : hi(h), lo(0.0) {}
  __device__ __forceinline__ dd(double h, double l) : hi(h), lo(l) {}
};

__device__ __forceinline__ dd dd_two_sum(double a, double b) {
  double s = __dadd_rn(a, b), bb = __dadd_rn(s, -a);
  double e = __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb));
  return dd(s, e);
}
__device__ __forceinline__ dd dd_quick_two_sum(double a, double b) {  // |a| >= |b|
  double s = __dadd_rn(a, b);
  return dd(s, __dadd_rn(b, -__dadd_rn(s, -a)));
}
__device__ __forceinline__ dd dd_two_prod(double a, double b) {
  double p = __dmul_rn(a, b);
  return dd(p, __fma_rn(a, b, -p));
}
__device__ __forceinline__ dd operator+(dd a, dd b) {   // accurate (IEEE-style) addition
  dd s = dd_two_sum(a.hi, b.hi), t = dd_two_sum(a.lo, b.lo);
  s.lo = __dadd_rn(s.lo, t.hi);
  s = dd_quick_two_sum(s.hi, s.lo);
  s.lo = __dadd_rn(s.lo, t.lo);
  return dd_quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd operator-(dd a) { return dd(-a.hi, -a.lo); }
__device__ __forceinline__ dd operator-(dd a, dd b) { return a + (-b); }
__device__ __forceinline__ dd operator*(dd a, dd b) {
  const double p = __dmul_rn(a.hi, b.hi);
  double e = __fma_rn(a.hi, b.hi, -p);
  e = __fma_rn(a.hi, b.lo, e);
  e = __fma_rn(a.lo, b.hi, e);
  return dd_quick_two_sum(p, e);
}
__device__ __forceinline__ dd operator*(dd a, double b) {
  dd p = dd_two_prod(a.hi, b);
  p.lo = __fma_rn(a.lo, b, p.lo);
  return dd_quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd operator/(dd a, dd b) {
  double q1 = __ddiv_rn(a.hi, b.hi);
  dd r = a - b * q1;
  double q2 = __ddiv_rn(r.hi, b.hi);
  r = r - b * q2;
  double q3 = __ddiv_rn(r.hi, b.hi);
  dd q = dd_quick_two_sum(q1, q2);
  return q + dd(q3);
}
__device__ __forceinline__ dd &operator+=(dd &a, dd b) { a = a + b; return a; }
__device__ __forceinline__ dd &operator-=(dd &a, dd b) { a = a - b; return a; }
__device__ __forceinline__ dd &operator*=(dd &a, dd b) { a = a * b; return a; }

// generic helpers so that one templated evaluator serves binary64 and double-double
__device__ __forceinline__ double mq_fma(double a, double b, double c) { return fma(a, b, c); }
// Pair arithmetic (no renormalisation of the result): a*b + c in 12 flops. The product of the high parts and the sum
// of the two high parts are exact (error-free transformations); every low-order term is binary64. The pair
// (s, lo) need not satisfy |lo| <= ulp(s)/2: after cancellation of the high parts |lo| may even exceed |s|, so
// nothing downstream may assume an ordering (two_sum, never quick_two_sum, on values that come from here).
// Error <= ~2^-103 (|a b| + |c|): the bound is relative to the operands, which is all a renormalising a*b + c gives
// after a cancellation as well; the evaluator renormalises once per family (mq_norm in account()).
// Error-free sum of two binary64 numbers in 3 FP64 instructions instead of 6 (MQ_DD_FAST2SUM = 1): FastTwoSum is exact when
// exponent(x) >= exponent(y); the operands are ordered by comparing their high words without the sign with INTEGER compare and
// selects, which run on the ALU pipe. MEASURED AND REJECTED on B200 (32 graphs of configs[4]): k_batch_dd 204 -> 236 ms. The
// kernel is at 73 % FP64 pipe activity but the ordering adds 7 ALU instructions to the dependency chain of every sum, and two
// warps per scheduler cannot hide it. Kept behind the switch for the record; default 0 = Knuth's branch-free two_sum.
#ifndef MQ_DD_FAST2SUM
#define MQ_DD_FAST2SUM 0
#endif
__device__ __forceinline__ dd dd_two_sum_ord(double a, double b) {
#if MQ_DD_FAST2SUM
  const bool sw = (unsigned)(__double2hiint(a) & 0x7fffffff) < (unsigned)(__double2hiint(b) & 0x7fffffff);
  const double x = sw ? b : a, y = sw ? a : b;
  const double s = __dadd_rn(x, y);
  return dd(s, __dadd_rn(y, -__dadd_rn(s, -x)));
#else
  return dd_two_sum(a, b);
#endif
}
__device__ __forceinline__ dd mq_fma(dd a, dd b, dd c) {
  const double p = __dmul_rn(a.hi, b.hi);
  double e = __fma_rn(a.hi, b.hi, -p);
  e = __fma_rn(a.hi, b.lo, e);
  e = __fma_rn(a.lo, b.hi, e);
  const dd st = dd_two_sum_ord(p, c.hi);
  return dd(st.hi, __dadd_rn(__dadd_rn(e, c.lo), st.lo));
}
__device__ __forceinline__ double mq_fma_c(double coef, double x, double c0, double) { return fma(coef, x, c0); }   // coef*x + c0
__device__ __forceinline__ dd mq_fma_c(double coef, dd x, double c0, dd) {   // coef*x + c0, coef and c0 binary64 (exact table entries); 10 flops
  const double p = __dmul_rn(coef, x.hi);
  double e = __fma_rn(coef, x.hi, -p);
  e = __fma_rn(coef, x.lo, e);
  const dd st = dd_two_sum_ord(p, c0);
  return dd(st.hi, __dadd_rn(st.lo, e));
}
// product of two pairs without renormalisation (5 flops); same remark as mq_fma
__device__ __forceinline__ dd mq_mul(dd a, dd b) {
  const double p = __dmul_rn(a.hi, b.hi);
  double e = __fma_rn(a.hi, b.hi, -p);
  e = __fma_rn(a.hi, b.lo, e);
  e = __fma_rn(a.lo, b.hi, e);
  return dd(p, e);
}
__device__ __forceinline__ double mq_mul(double a, double b) { return a * b; }
__device__ __forceinline__ dd mq_norm(dd a) { return dd_two_sum(a.hi, a.lo); }
__device__ __forceinline__ double mq_norm(double a) { return a; }
__device__ __forceinline__ double mq_to_double(double a) { return a; }
__device__ __forceinline__ double mq_to_double(dd a) { return a.hi + a.lo; }
__device__ __forceinline__ double mq_abs(double a) { return fabs(a); }
__device__ __forceinline__ dd mq_abs(dd a) { return a.hi < 0 ? -a : a; }
__device__ __forceinline__ bool mq_lt0(double a) { return a < 0; }
__device__ __forceinline__ bool mq_lt0(dd a) { return a.hi < 0; }
