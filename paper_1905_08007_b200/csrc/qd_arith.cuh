// qd_arith.cuh — quad-double arithmetic (four non-overlapping binary64 words, ~212 bits) for the third
// precision tier: points whose cancellation exceeds what double-double can resolve (O8;
// PAPER.md:91 "arithmetic with different precisions"). Renormalisation-based algorithms in the style of
// Hida-Li-Bailey's QD, restated here; speed is irrelevant (a few per mille of the points). Device only.
#pragma once
#include "dd_arith.cuh"

struct qd {
  double x[4];
  __device__ __forceinline__ qd() {}
  __device__ __forceinline__ qd(double a) { x[0] = a; x[1] = x[2] = x[3] = 0.0; }
  __device__ __forceinline__ qd(double a, double b, double c, double d) { x[0] = a; x[1] = b; x[2] = c; x[3] = d; }
};

namespace qdi {
__device__ __forceinline__ double qts(double a, double b, double &e) { double s = __dadd_rn(a, b); e = __dadd_rn(b, -__dadd_rn(s, -a)); return s; }   // |a| >= |b|
__device__ __forceinline__ double ts(double a, double b, double &e) {
  double s = __dadd_rn(a, b), bb = __dadd_rn(s, -a);
  e = __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb));
  return s;
}
__device__ __forceinline__ double tp(double a, double b, double &e) { double p = __dmul_rn(a, b); e = __fma_rn(a, b, -p); return p; }
__device__ __forceinline__ void three_sum(double &a, double &b, double &c) {
  double t1, t2, t3;
  t1 = ts(a, b, t2); a = ts(c, t1, t3); b = ts(t2, t3, c);
}
__device__ __forceinline__ void three_sum2(double &a, double &b, double c) {
  double t1, t2, t3;
  t1 = ts(a, b, t2); a = ts(c, t1, t3); b = __dadd_rn(t2, t3);
}
__device__ __forceinline__ qd renorm(double c0, double c1, double c2, double c3, double c4) {
  double s0, s1, s2 = 0.0, s3 = 0.0;
  s0 = qts(c3, c4, c4); s0 = qts(c2, s0, c3); s0 = qts(c1, s0, c2); c0 = qts(c0, s0, c1);
  s0 = c0; s1 = c1;
  if (s1 != 0.0) {
    s1 = qts(s1, c2, s2);
    if (s2 != 0.0) { s2 = qts(s2, c3, s3); if (s3 != 0.0) s3 = __dadd_rn(s3, c4); else s2 = qts(s2, c4, s3); }
    else { s1 = qts(s1, c3, s2); if (s2 != 0.0) s2 = qts(s2, c4, s3); else s1 = qts(s1, c4, s2); }
  } else {
    s0 = qts(s0, c2, s1);
    if (s1 != 0.0) { s1 = qts(s1, c3, s2); if (s2 != 0.0) s2 = qts(s2, c4, s3); else s1 = qts(s1, c4, s2); }
    else { s0 = qts(s0, c3, s1); if (s1 != 0.0) s1 = qts(s1, c4, s2); else s0 = qts(s0, c4, s1); }
  }
  return qd(s0, s1, s2, s3);
}
}  // namespace qdi

__device__ __forceinline__ qd operator-(qd a) { return qd(-a.x[0], -a.x[1], -a.x[2], -a.x[3]); }
static __device__ __noinline__ qd operator+(qd a, qd b) {
  using namespace qdi;
  double s0, s1, s2, s3, t0, t1, t2, t3;
  s0 = ts(a.x[0], b.x[0], t0); s1 = ts(a.x[1], b.x[1], t1); s2 = ts(a.x[2], b.x[2], t2); s3 = ts(a.x[3], b.x[3], t3);
  s1 = ts(s1, t0, t0);
  three_sum(s2, t0, t1);
  three_sum2(s3, t0, t2);
  t0 = __dadd_rn(__dadd_rn(t0, t1), t3);
  return renorm(s0, s1, s2, s3, t0);
}
__device__ __forceinline__ qd operator-(qd a, qd b) { return a + (-b); }
static __device__ __noinline__ qd operator*(qd a, qd b) {
  using namespace qdi;
  double p0, p1, p2, p3, p4, p5, q0, q1, q2, q3, q4, q5, t0, t1, s0, s1, s2;
  p0 = tp(a.x[0], b.x[0], q0);
  p1 = tp(a.x[0], b.x[1], q1); p2 = tp(a.x[1], b.x[0], q2);
  p3 = tp(a.x[0], b.x[2], q3); p4 = tp(a.x[1], b.x[1], q4); p5 = tp(a.x[2], b.x[0], q5);
  three_sum(p1, p2, q0);
  three_sum(p2, q1, q2); three_sum(p3, p4, p5);
  s0 = ts(p2, p3, t0); s1 = ts(q1, p4, t1); s2 = __dadd_rn(q2, p5);
  s1 = ts(s1, t0, t0); s2 = __dadd_rn(s2, __dadd_rn(t0, t1));
  double o3 = __fma_rn(a.x[0], b.x[3], __fma_rn(a.x[1], b.x[2], __fma_rn(a.x[2], b.x[1], __dmul_rn(a.x[3], b.x[0]))));
  s1 = __dadd_rn(s1, __dadd_rn(__dadd_rn(o3, q0), __dadd_rn(__dadd_rn(q3, q4), q5)));
  return renorm(p0, p1, s0, s1, s2);
}
__device__ __forceinline__ qd operator*(qd a, double b) { return a * qd(b); }
static __device__ __noinline__ qd operator/(qd a, qd b) {   // long division, five quotient words
  double q0 = __ddiv_rn(a.x[0], b.x[0]);
  qd r = a - b * q0;
  double q1 = __ddiv_rn(r.x[0], b.x[0]); r = r - b * q1;
  double q2 = __ddiv_rn(r.x[0], b.x[0]); r = r - b * q2;
  double q3 = __ddiv_rn(r.x[0], b.x[0]); r = r - b * q3;
  double q4 = __ddiv_rn(r.x[0], b.x[0]);
  return qdi::renorm(q0, q1, q2, q3, q4);
}
__device__ __forceinline__ qd &operator+=(qd &a, qd b) { a = a + b; return a; }

__device__ __forceinline__ qd mq_fma(qd a, qd b, qd c) { return a * b + c; }
__device__ __forceinline__ qd mq_fma_c(double coef, qd x, double c0, qd) { return x * qd(coef) + qd(c0); }
__device__ __forceinline__ qd mq_mul(qd a, qd b) { return a * b; }
__device__ __forceinline__ qd mq_norm(qd a) { return a; }
__device__ __forceinline__ double mq_to_double(qd a) { return __dadd_rn(__dadd_rn(a.x[0], a.x[1]), __dadd_rn(a.x[2], a.x[3])); }
__device__ __forceinline__ double mq_mag(qd a) { return mq_to_double(a); }
__device__ __forceinline__ double mq_absd(qd a) { return fabs(a.x[0]); }
__device__ __forceinline__ qd mq_abs(qd a) { return a.x[0] < 0 ? -a : a; }
__device__ __forceinline__ bool mq_lt0(qd a) { return a.x[0] < 0; }
