// iv_arith.cuh — binary64 interval arithmetic with directed rounding, the value type of the interval tier (kern_iv.cu).
// Product code (libmcqed.so). Device only.
//
// the paper controls round-off "by interval arithmetic with different precisions and speeds": a value is
// accepted when its rigorous enclosure is narrow enough, else the point is re-evaluated in a slower, wider arithmetic. This
// header makes the templated evaluator of mcqed_kernels.cuh run on intervals [lo, hi]: every operation rounds the lower
// bound down and the upper bound up (__dadd_rd/_ru, __dmul_rd/_ru, __fma_rd/_ru, __ddiv_rd/_ru), so the TRUE value of the
// integrand at the given binary64 coordinates lies in the result — an enclosure, not an estimate.
// Table coefficients are exact binary64 numbers, so coefficient * interval + coefficient needs two directed FMAs only.
#pragma once
#include <cuda_runtime.h>

struct iv {
  double lo, hi;
  __device__ __forceinline__ iv() {}
  __device__ __forceinline__ iv(double x) : lo(x), hi(x) {}
  __device__ __forceinline__ iv(double l, double h) : lo(l), hi(h) {}
};
__device__ __forceinline__ iv operator+(iv a, iv b) { return iv(__dadd_rd(a.lo, b.lo), __dadd_ru(a.hi, b.hi)); }
__device__ __forceinline__ iv operator-(iv a) { return iv(-a.hi, -a.lo); }
__device__ __forceinline__ iv operator-(iv a, iv b) { return iv(__dadd_rd(a.lo, -b.hi), __dadd_ru(a.hi, -b.lo)); }
__device__ __forceinline__ iv operator*(iv a, iv b) {
  // the four corner products, each rounded both ways; a NaN (0 * inf) poisons the result, which the caller treats as "no enclosure"
  const double l = fmin(fmin(__dmul_rd(a.lo, b.lo), __dmul_rd(a.lo, b.hi)), fmin(__dmul_rd(a.hi, b.lo), __dmul_rd(a.hi, b.hi)));
  const double h = fmax(fmax(__dmul_ru(a.lo, b.lo), __dmul_ru(a.lo, b.hi)), fmax(__dmul_ru(a.hi, b.lo), __dmul_ru(a.hi, b.hi)));
  return iv(l, h);
}
__device__ __forceinline__ iv operator/(iv a, iv b) {
  if (!(b.lo > 0.0 || b.hi < 0.0)) return iv(-__longlong_as_double(0x7ff0000000000000ll), __longlong_as_double(0x7ff0000000000000ll));   // 0 in the divisor: no enclosure
  const iv r(__ddiv_rd(1.0, b.hi), __ddiv_ru(1.0, b.lo));      // 1/b is decreasing on either side of 0
  return a * r;
}
__device__ __forceinline__ iv &operator+=(iv &a, iv b) { a = a + b; return a; }
__device__ __forceinline__ iv &operator*=(iv &a, iv b) { a = a * b; return a; }

// generic helpers of the templated evaluator (dd_arith.cuh has the binary64 / double-double ones)
__device__ __forceinline__ iv mq_fma(iv a, iv b, iv c) { return a * b + c; }
__device__ __forceinline__ iv mq_fma_c(double coef, iv x, double c0, iv) {   // coef * x + c0 with exact coef, c0: two directed FMAs
  const bool pos = coef >= 0.0;
  return iv(__fma_rd(coef, pos ? x.lo : x.hi, c0), __fma_ru(coef, pos ? x.hi : x.lo, c0));
}
__device__ __forceinline__ iv mq_mul(iv a, iv b) { return a * b; }
__device__ __forceinline__ iv mq_norm(iv a) { return a; }
__device__ __forceinline__ double mq_to_double(iv a) { return 0.5 * a.lo + 0.5 * a.hi; }
__device__ __forceinline__ double mq_mag(iv a) { return 0.5 * a.lo + 0.5 * a.hi; }                  // the value as a magnitude: its midpoint
__device__ __forceinline__ double mq_absd(iv a) { return fmax(fabs(a.lo), fabs(a.hi)); }            // largest |x| in the interval
__device__ __forceinline__ iv mq_abs(iv a) { return a.lo >= 0.0 ? a : a.hi <= 0.0 ? -a : iv(0.0, fmax(-a.lo, a.hi)); }
__device__ __forceinline__ bool mq_lt0(iv a) { return a.hi < 0.0; }
