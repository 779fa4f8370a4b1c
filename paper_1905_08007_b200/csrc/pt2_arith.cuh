// pt2_arith.cuh — "N sample points per lane" value type of the binary64 tier (ptn<N>, N = 2 or 4), and the magnitude
// traits that let one templated evaluator (mcqed_kernels.cuh) serve double, ptn<N> (N x binary64), dd and qd.
// Product code (libmcqed.so). Device only.
//
// Why (measured on B200, profiles/r2_microbench.md): a shared-memory load returns 8 bytes per lane per cycle per SM whether
// or not the lanes read the same address, and the FP64 pipe retires 2 warp-DFMA per cycle per SM. With lanes = sample points
// every table coefficient is a broadcast load feeding ONE DFMA per lane: the load path allows at most 50 % of the FP64 peak
// before any operand gather is counted (round 1: L1/TEX 71 %, FP64 pipe 37 %). A lane that carries N points uses every loaded
// coefficient, header field and index byte N times: 1/N of the table-side bytes and instructions per DFMA, and N independent
// FMA chains per lane.
#pragma once
#include <cuda_runtime.h>

#include "dd_arith.cuh"

template <int N> struct ptn {
  double v[N];
  __device__ __forceinline__ ptn() {}
  __device__ __forceinline__ ptn(double x) {
#pragma unroll
    for (int i = 0; i < N; i++) v[i] = x;
  }
};
using pt2 = ptn<2>;
using pt4 = ptn<4>;
#define MQ_PTN_OP2(name, expr)                                                      \
  template <int N> __device__ __forceinline__ ptn<N> name(ptn<N> x, ptn<N> y) {     \
    ptn<N> r;                                                                       \
    _Pragma("unroll") for (int i = 0; i < N; i++) r.v[i] = (expr);                  \
    return r;                                                                       \
  }
MQ_PTN_OP2(operator+, x.v[i] + y.v[i])
MQ_PTN_OP2(operator-, x.v[i] - y.v[i])
MQ_PTN_OP2(operator*, x.v[i] * y.v[i])
MQ_PTN_OP2(operator/, x.v[i] / y.v[i])
MQ_PTN_OP2(mq_mul, x.v[i] * y.v[i])
MQ_PTN_OP2(mq_mmin, fmin(x.v[i], y.v[i]))
#undef MQ_PTN_OP2
#define MQ_PTN_OP1(name, expr)                                                      \
  template <int N> __device__ __forceinline__ ptn<N> name(ptn<N> x) {               \
    ptn<N> r;                                                                       \
    _Pragma("unroll") for (int i = 0; i < N; i++) r.v[i] = (expr);                  \
    return r;                                                                       \
  }
MQ_PTN_OP1(operator-, -x.v[i])
MQ_PTN_OP1(mq_abs, fabs(x.v[i]))
MQ_PTN_OP1(mq_absd, fabs(x.v[i]))
MQ_PTN_OP1(mq_mmax1, fmax(1.0, x.v[i]))
MQ_PTN_OP1(mq_norm, x.v[i])
MQ_PTN_OP1(mq_mag, x.v[i])
#undef MQ_PTN_OP1
// mixed operand forms (a binary64 constant on one side) so that template deduction never has to convert
template <int N> __device__ __forceinline__ ptn<N> operator+(ptn<N> x, double y) { return x + ptn<N>(y); }
template <int N> __device__ __forceinline__ ptn<N> operator-(double x, ptn<N> y) { return ptn<N>(x) - y; }
template <int N> __device__ __forceinline__ ptn<N> operator*(ptn<N> x, double y) { return x * ptn<N>(y); }
template <int N> __device__ __forceinline__ ptn<N> operator/(double x, ptn<N> y) { return ptn<N>(x) / y; }
template <int N> __device__ __forceinline__ ptn<N> &operator+=(ptn<N> &x, ptn<N> y) { x = x + y; return x; }
template <int N> __device__ __forceinline__ ptn<N> &operator*=(ptn<N> &x, ptn<N> y) { x = x * y; return x; }
template <int N> __device__ __forceinline__ ptn<N> mq_fma(ptn<N> x, ptn<N> y, ptn<N> z) {
  ptn<N> r;
#pragma unroll
  for (int i = 0; i < N; i++) r.v[i] = fma(x.v[i], y.v[i], z.v[i]);
  return r;
}
template <int N> __device__ __forceinline__ ptn<N> mq_fma_c(double coef, ptn<N> x, double c0, ptn<N>) {   // coef*x + c0
  ptn<N> r;
#pragma unroll
  for (int i = 0; i < N; i++) r.v[i] = fma(coef, x.v[i], c0);
  return r;
}
template <int N> __device__ __forceinline__ ptn<N> mq_mfma(ptn<N> a, double l, ptn<N> c) {                 // a*l + c on magnitudes
  ptn<N> r;
#pragma unroll
  for (int i = 0; i < N; i++) r.v[i] = fma(a.v[i], l, c.v[i]);
  return r;
}

// Magnitude type M of a value type T: what round-off bounds, pivot ratios and the like are carried in.
// double for double, dd and qd (one point per lane); ptn<N> for ptn<N> (one bound per point). M also is the type of the
// coordinates z handed to the evaluator.
template <class T> struct MagOf { using type = double; };
template <int N> struct MagOf<ptn<N>> { using type = ptn<N>; };
template <class T> struct PtsOf { static constexpr int n = 1; };       // sample points per lane
template <int N> struct PtsOf<ptn<N>> { static constexpr int n = N; };

__device__ __forceinline__ double mq_absd(double a) { return fabs(a); }
__device__ __forceinline__ double mq_absd(dd a) { return fabs(a.hi); }
__device__ __forceinline__ double mq_mag(double a) { return a; }
__device__ __forceinline__ double mq_mag(dd a) { return a.hi + a.lo; }
__device__ __forceinline__ double mq_mfma(double a, double l, double c) { return fma(a, l, c); }
__device__ __forceinline__ double mq_mmin(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ double mq_mmax1(double a) { return fmax(1.0, a); }
// component k of a per-lane value (k < PtsOf<T>::n)
__device__ __forceinline__ double mq_comp(double x, int) { return x; }
__device__ __forceinline__ void mq_setc(double &x, int, double v) { x = v; }
template <int N> __device__ __forceinline__ double mq_comp(const ptn<N> &x, int k) {
  double r = x.v[0];
#pragma unroll
  for (int i = 1; i < N; i++) r = (k == i) ? x.v[i] : r;
  return r;
}
template <int N> __device__ __forceinline__ void mq_setc(ptn<N> &x, int k, double v) {
#pragma unroll
  for (int i = 0; i < N; i++) x.v[i] = (k == i) ? v : x.v[i];
}
