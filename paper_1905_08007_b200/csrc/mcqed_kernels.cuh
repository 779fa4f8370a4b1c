// mcqed_kernels.cuh — device code of the hot path (steps a1-a8 of DESIGN.md §2), sm_100a.
// Product code (libmcqed.so); shares nothing with oracle/.
//
// Mapping: lanes = sample points of ONE diagram (MQ_WL lanes share a point and evaluate the MQ_WL families of a
// stream entry side by side: "lane split" below). All threads of a CTA work on the same diagram, so every table
// read (entry headers, coefficients, Z/invDeg rows) is warp-uniform and control flow never diverges inside the
// integrand. Per-point operands that the tables address by index (r_t, A_t, A'_t/g_t, beta_tu/(g_t g_u)) live in
// shared memory laid out [index][point] (conflict-free); everything with static indexing lives in registers.
// The quad-double tier works entry-parallel instead (one point per CTA). FP64 FMA pipe is the roofline.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "dd_arith.cuh"
#include "pt2_arith.cuh"
#include "device_layout.h"

// Device-side bounds checks of the library's own (build with MCQED_DEFS=-DMQ_DEVICE_ASSERTS=1; compute-sanitizer is not
// available on every pool). Every run-time index into shared memory, the per-thread arrays and the scratch lists is checked;
// a violation prints its place and traps, which the host sees as a launch failure. Off (no code) in the normal build.
#ifndef MQ_DEVICE_ASSERTS
#define MQ_DEVICE_ASSERTS 0
#endif
#if MQ_DEVICE_ASSERTS
#include <cstdio>
#define MQ_DASSERT(c) do { if (!(c)) { printf("MQ_DASSERT %s:%d: %s (block %d thread %d)\n", __FILE__, __LINE__, #c, (int)blockIdx.x, (int)threadIdx.x); __trap(); } } while (0)
#else
#define MQ_DASSERT(c) ((void)0)
#endif

namespace mqk {

// value types whose family code keeps the outer pairing levels (c >= 3) and the halves of a kd = 6 block in real loops:
// everything but plain binary64 (double-double: code size; N points per lane: registers)
#define MQ_LOOPED(T) (!std::is_same<T, double>::value)
#ifndef MQ_DUAL
#define MQ_DUAL 1     // binary64: evaluate two consecutive same-shape entries together (independent chains)
#endif

struct DiagView {
  const uint64_t *blob; const DevHeader *h; const double *Z, *invdeg;
  const DevGeom *geom; const DevTable *tab; const DevNode *node; const DevTerm *term;
};
__device__ __forceinline__ DiagView make_view(const uint64_t *blob) {
  DiagView v; v.blob = blob; v.h = reinterpret_cast<const DevHeader *>(blob);
  v.Z = reinterpret_cast<const double *>(blob + v.h->off_Z);
  v.invdeg = reinterpret_cast<const double *>(blob + v.h->off_invdeg);
  v.geom = reinterpret_cast<const DevGeom *>(blob + v.h->off_geom);
  v.tab = reinterpret_cast<const DevTable *>(blob + v.h->off_table);
  v.node = reinterpret_cast<const DevNode *>(blob + v.h->off_node);
  v.term = reinterpret_cast<const DevTerm *>(blob + v.h->off_term);
  return v;
}

// ------------------------------------------------------------------ a1: Philox4x32-10
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; r++) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ __forceinline__ double u01(uint32_t x, uint32_t y) {   // 52 random bits, strictly inside (0,1), exact
  return __dmul_rn(__dadd_rn(__dadd_rn(__dmul_rn((double)(x >> 6), 67108864.0), (double)(y >> 6)), 0.5), 1.0 / 4503599627370496.0);
}

// ------------------------------------------------------------------ a1': MRG32k3a ("Calc 1"; S1b)
// x1_n = (1403580 x1_{n-2} - 810728 x1_{n-3}) mod m1, x2_n = (527612 x2_{n-1} - 1370589 x2_{n-3}) mod m2, w_n = (x1_n - x2_n) mod m1,
// m1 = 2^32 - 209, m2 = 2^32 - 22853. Used counter-style: sample idx of diagram id owns the 64 outputs from position
// (id * 2^38 + idx) * 64 on; the position is reached with the stored powers A^(2^k) of the two companion matrices (pw: [2][64][9]
// uint32 in the diagram blob, host_prepare.cpp), one 3x3 matrix-vector product mod m per set bit. Reduction mod 2^32 - c by folding
// the high word twice (hi * c + lo), no division.
#define MQ_MRG_M1 4294967087u
#define MQ_MRG_M2 4294944443u
template <uint32_t CC> __device__ __forceinline__ uint32_t mrg_red(uint64_t p) {      // p mod (2^32 - CC), any p < 2^64, CC < 2^15
  p = (p >> 32) * CC + (p & 0xffffffffull);
  p = (p >> 32) * CC + (p & 0xffffffffull);                                             // < 2^32 + 2^30
  const uint64_t m = 4294967296ull - CC;
  return (uint32_t)(p >= m ? p - m : p);
}
template <uint32_t CC> __device__ __forceinline__ uint32_t mrg_addmod(uint32_t a, uint32_t b) {
  const uint64_t m = 4294967296ull - CC, t = (uint64_t)a + b;
  return (uint32_t)(t >= m ? t - m : t);
}
template <uint32_t CC> __device__ __forceinline__ void mrg_matvec(const uint32_t *__restrict__ P, uint32_t s[3]) {
  uint32_t t[3];
#pragma unroll
  for (int i = 0; i < 3; i++) {
    uint32_t acc = mrg_red<CC>((uint64_t)__ldg(P + 3 * i) * s[0]);
    acc = mrg_addmod<CC>(acc, mrg_red<CC>((uint64_t)__ldg(P + 3 * i + 1) * s[1]));
    t[i] = mrg_addmod<CC>(acc, mrg_red<CC>((uint64_t)__ldg(P + 3 * i + 2) * s[2]));
  }
  s[0] = t[0]; s[1] = t[1]; s[2] = t[2];
}
// the first nu uniforms of the sample: uniform r from outputs 2r, 2r+1. Not inlined: it runs once per point, and its registers
// stay out of the evaluator's allocation.
static __device__ __noinline__ void mrg32k3a_uniforms(const uint32_t *__restrict__ pw, uint64_t seed, uint64_t skip, int nu, double *u) {
  const uint32_t lo = (uint32_t)seed, hi = (uint32_t)(seed >> 32);
  uint32_t s1[3] = {1u + lo % (MQ_MRG_M1 - 1u), 1u + hi % (MQ_MRG_M1 - 1u), 12345u};
  uint32_t s2[3] = {1u + lo % (MQ_MRG_M2 - 1u), 1u + hi % (MQ_MRG_M2 - 1u), 12345u};
  for (int k = 0; skip; k++, skip >>= 1)
    if (skip & 1) { mrg_matvec<209u>(pw + 9 * k, s1); mrg_matvec<22853u>(pw + 9 * (64 + k), s2); }
  uint32_t w[2];
  for (int r = 0; r < nu; r++) {
#pragma unroll
    for (int j = 0; j < 2; j++) {
      const uint32_t x1 = mrg_addmod<209u>(mrg_red<209u>(1403580ull * s1[1]), mrg_red<209u>((uint64_t)(MQ_MRG_M1 - 810728u) * s1[0]));
      const uint32_t x2 = mrg_addmod<22853u>(mrg_red<22853u>(527612ull * s2[2]), mrg_red<22853u>((uint64_t)(MQ_MRG_M2 - 1370589u) * s2[0]));
      s1[0] = s1[1]; s1[1] = s1[2]; s1[2] = x1; s2[0] = s2[1]; s2[1] = s2[2]; s2[2] = x2;
      w[j] = x1 >= x2 ? x1 - x2 : x1 + (MQ_MRG_M1 - x2);       // (x1 - x2) mod m1 (x2 < m2 < m1)
    }
    u[r] = u01(w[0], w[1]);
  }
}

// ------------------------------------------------------------------ a3: deterministic pow (S4)
// explicit round-to-nearest mul/add only (never contracted) so that the bits equal the oracle's
__device__ __forceinline__ double det_log2(double u) {
  uint64_t bits = (uint64_t)__double_as_longlong(u);
  int ex = (int)((bits >> 52) & 0x7FF) - 1023;
  double m = __longlong_as_double((long long)((bits & 0x000FFFFFFFFFFFFFull) | 0x3FF0000000000000ull));
  if (m > 1.4142135623730951) { m = __dmul_rn(m, 0.5); ex += 1; }
  double s = __ddiv_rn(__dadd_rn(m, -1.0), __dadd_rn(m, 1.0)), s2 = __dmul_rn(s, s);
  double P = 1.0 / 23.0;
#define MQ_H(c) P = __dadd_rn(__dmul_rn(P, s2), (c))
  MQ_H(1.0 / 21.0); MQ_H(1.0 / 19.0); MQ_H(1.0 / 17.0); MQ_H(1.0 / 15.0); MQ_H(1.0 / 13.0); MQ_H(1.0 / 11.0);
  MQ_H(1.0 / 9.0); MQ_H(1.0 / 7.0); MQ_H(1.0 / 5.0); MQ_H(1.0 / 3.0); MQ_H(1.0);
#undef MQ_H
  double lnm = __dmul_rn(__dmul_rn(2.0, s), P);
  return __dadd_rn((double)ex, __dmul_rn(lnm, 1.4426950408889634));
}
__device__ __forceinline__ double det_exp2(double y) {
  if (y < -1020.0) return 0.0;
  double n = floor(__dadd_rn(y, 0.5)), r = __dadd_rn(y, -n), w = __dmul_rn(r, 0.6931471805599453);
  double P = 1.0 / 87178291200.0;
#define MQ_H(c) P = __dadd_rn(__dmul_rn(P, w), (c))
  MQ_H(1.0 / 6227020800.0); MQ_H(1.0 / 479001600.0); MQ_H(1.0 / 39916800.0); MQ_H(1.0 / 3628800.0); MQ_H(1.0 / 362880.0);
  MQ_H(1.0 / 40320.0); MQ_H(1.0 / 5040.0); MQ_H(1.0 / 720.0); MQ_H(1.0 / 120.0); MQ_H(1.0 / 24.0); MQ_H(1.0 / 6.0);
  MQ_H(0.5); MQ_H(1.0); MQ_H(1.0);
#undef MQ_H
  double sc = __longlong_as_double((long long)((uint64_t)((long long)n + 1023) << 52));
  return __dmul_rn(P, sc);
}

// ------------------------------------------------------------------ a2+a3: sector walk, coordinates, density (Eq.(1))
// z[] is written by line index; order[] (optional) gets the sector j_1..j_M; returns p(z)
template <bool WANT_ORDER>
__device__ __forceinline__ double draw_point(const DiagView &v, uint64_t idx, uint64_t seed, double *z, int32_t *order_out) {
  const int M = v.h->M;
  const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32), i0 = (uint32_t)idx, i1 = (uint32_t)(idx >> 32), dg = (uint32_t)v.h->diag_id;
  uint32_t mask = (1u << M) - 1;
  double r[MQ_MAXM]; int8_t ord[MQ_MAXM];
  double rl = 1.0, pu = 1.0;
  uint32_t ws[4], wr[4];
  const bool mrg = v.h->rng != 0;                      // the same for every point of a launch: no divergence
  double um[2 * MQ_MAXM];
  // defensive mixture (S5b): uniform number 2(M-1) picks the channel that draws the point; the other channel's density at
  // the point is prod t_l^Deg_other, accumulated in pq. The same for every point of a launch when off (alpha = 0): no divergence.
  const double alpha = v.h->mix_alpha;
  const bool mix = alpha > 0.0;
  if (mrg) mrg32k3a_uniforms(reinterpret_cast<const uint32_t *>(v.blob + v.h->off_mrg), seed, (((uint64_t)dg << 38) + idx) << 6, 2 * (M - 1) + (mix ? 1 : 0), um);
  const double *Zt = v.Z, *idg = v.invdeg, *dgo = nullptr;
  double Cd = v.h->C, Co = 0.0, pq = 1.0;
  bool alt = false;
  if (mix) {
    double uc;
    if (mrg) uc = um[2 * (M - 1)];
    else { uint32_t wc[4]; philox4x32_10(i0, i1, (uint32_t)(M - 1), dg, k0, k1, wc); uc = u01(wc[0], wc[1]); }
    alt = uc < alpha;
    const double *b = reinterpret_cast<const double *>(v.blob);
    if (alt) { Zt = b + v.h->off_Z2; idg = b + v.h->off_invdeg2; dgo = b + v.h->off_deg1; Cd = v.h->C2; Co = v.h->C; }
    else { dgo = b + v.h->off_deg2; Co = v.h->C2; }
  }
  for (int l = 0; l < M; l++) {
    int x;
    if (l == M - 1) x = __ffs(mask) - 1;
    else {
      if (!mrg && (l & 1) == 0) philox4x32_10(i0, i1, (uint32_t)(l >> 1), dg, k0, k1, ws);
      double u = mrg ? um[l] : (l & 1) ? u01(ws[2], ws[3]) : u01(ws[0], ws[1]);
      double total = 0.0;
      for (uint32_t mm = mask; mm; mm &= mm - 1) { int y = __ffs(mm) - 1; total = __dadd_rn(total, __ldg(&Zt[mask & ~(1u << y)])); }
      double target = __dmul_rn(u, total), cum = 0.0;
      x = -1; int last = -1;
      for (uint32_t mm = mask; mm; mm &= mm - 1) {
        int y = __ffs(mm) - 1; cum = __dadd_rn(cum, __ldg(&Zt[mask & ~(1u << y)])); last = y;
        if (target < cum) { x = y; break; }
      }
      if (x < 0) x = last;
    }
    if (l >= 1) {
      int ru = (M - 1) + (l - 1);
      if (!mrg && ((ru & 1) == 0 || l == 1)) philox4x32_10(i0, i1, (uint32_t)(ru >> 1), dg, k0, k1, wr);
      double u = mrg ? um[ru] : (ru & 1) ? u01(wr[2], wr[3]) : u01(wr[0], wr[1]);
      const double lg = __dmul_rn(det_log2(u), __ldg(&idg[mask]));
      double t = det_exp2(lg);
      rl = __dmul_rn(rl, t); pu = __dmul_rn(pu, u);
      if (mix) pq = __dmul_rn(pq, det_exp2(__dmul_rn(lg, __ldg(&dgo[mask]))));
    }
    r[l] = rl; ord[l] = (int8_t)x;
    mask &= ~(1u << x);
  }
  double S = 0.0;
  for (int l = 0; l < M; l++) S = __dadd_rn(S, r[l]);
  double pz = 1.0;
  for (int l = 0; l < M; l++) { double zz = __ddiv_rn(r[l], S); z[ord[l]] = zz; pz = __dmul_rn(pz, zz); if (WANT_ORDER) order_out[l] = ord[l]; }
  const double p_drawn = __ddiv_rn(__dmul_rn(Cd, pu), pz);
  if (!mix) return p_drawn;
  const double p_other = __ddiv_rn(__dmul_rn(Co, pq), pz);
  const double p_main = alt ? p_other : p_drawn, p_alt = alt ? p_drawn : p_other;
  return __dadd_rn(__dmul_rn(__dadd_rn(1.0, -alpha), p_main), __dmul_rn(alpha, p_alt));
}

// ------------------------------------------------------------------ shared-memory helpers (explicit LDS) and the stream reader
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t lds_u64(uint32_t a) { uint64_t v; asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds_u8(uint32_t a) { uint32_t v; asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ double2 lds_f64x2(uint32_t a) { double2 v; asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a)); return v; }
__device__ __forceinline__ double lds_f64(uint32_t a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
template <class T> __device__ __forceinline__ T lds_T(uint32_t a);
template <> __device__ __forceinline__ double lds_T<double>(uint32_t a) { return lds_f64(a); }
template <> __device__ __forceinline__ dd lds_T<dd>(uint32_t a) { double2 v = lds_f64x2(a); return dd(v.x, v.y); }
// Access to the per-point scalar scratch S[index][slot] of a CTA (stride = slots per CTA; S = this lane's slot base).
// Scalar types: one element of sizeof(T) per (index, slot). ptn<N>: N/2 planes of 16-byte point pairs per index,
// [index][plane][slot], so that the lanes of a warp read consecutive 16-byte units (no bank conflicts for any N).
// lds(a, sstride): a = shared address of (index, this slot), sstride = bytes per index = stride * sizeof(T).
template <class T> struct SAcc {
  static constexpr int slot_bytes = sizeof(T);
  static __device__ __forceinline__ T lds(uint32_t a, uint32_t) { return lds_T<T>(a); }
  static __device__ __forceinline__ T ld(const unsigned char *S, int i, int stride) { return reinterpret_cast<const T *>(S)[(size_t)i * stride]; }
  static __device__ __forceinline__ void st(unsigned char *S, int i, int stride, T v) { reinterpret_cast<T *>(S)[(size_t)i * stride] = v; }
};
template <int N> struct SAcc<ptn<N>> {
  static constexpr int slot_bytes = 16, NPL = N / 2;
  static __device__ __forceinline__ ptn<N> lds(uint32_t a, uint32_t sstride) {
    ptn<N> r;
#pragma unroll
    for (int h = 0; h < NPL; h++) { const double2 v = lds_f64x2(a + h * (sstride / NPL)); r.v[2 * h] = v.x; r.v[2 * h + 1] = v.y; }
    return r;
  }
  static __device__ __forceinline__ ptn<N> ld(const unsigned char *S, int i, int stride) {
    ptn<N> r;
#pragma unroll
    for (int h = 0; h < NPL; h++) { const double2 v = reinterpret_cast<const double2 *>(S)[(size_t)(i * NPL + h) * stride]; r.v[2 * h] = v.x; r.v[2 * h + 1] = v.y; }
    return r;
  }
  static __device__ __forceinline__ void st(unsigned char *S, int i, int stride, ptn<N> x) {
#pragma unroll
    for (int h = 0; h < NPL; h++) reinterpret_cast<double2 *>(S)[(size_t)(i * NPL + h) * stride] = make_double2(x.v[2 * h], x.v[2 * h + 1]);
  }
};

// The family stream of a diagram is staged through shared memory in chunks of MQ_CHUNK_WORDS words by bulk
// asynchronous copies (cp.async.bulk + mbarrier, the TMA engine; SASS UBLKCP), two chunks in flight, so that
// headers, index bytes and coefficients are read at shared-memory latency by every warp of the CTA.
// All methods are CTA-collective: every thread of the CTA calls them in the same order.
struct StreamReader {
  const uint64_t *gsrc;   // first chunk in global memory
#if MQ_DEVICE_ASSERTS
  int dbg_scal_len;       // number of S indices of the point group (the bound of every index byte of the stream)
#endif
  uint32_t s_buf;         // shared address of the two chunk buffers
  uint32_t s_bar;         // shared address of the two mbarriers
  int nchunks, chunk, pos;
  uint32_t phase;         // bit b: parity the next wait on buffer b expects

  __device__ __forceinline__ void init(uint64_t *buf, uint64_t *bar) {
    s_buf = smem_u32(buf); s_bar = smem_u32(bar); phase = 0;
    if (threadIdx.x == 0) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s_bar));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s_bar + 8));
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
  }
  __device__ __forceinline__ void issue(int k) {   // thread 0 only
    const uint32_t bar = s_bar + 8 * (k & 1), dst = s_buf + (k & 1) * (MQ_CHUNK_WORDS * 8);
    const uint32_t bytes = MQ_CHUNK_WORDS * 8;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(gsrc + (size_t)k * MQ_CHUNK_WORDS), "r"(bytes), "r"(bar) : "memory");
  }
  __device__ __forceinline__ void wait(int k) {
    const uint32_t bar = s_bar + 8 * (k & 1), par = (phase >> (k & 1)) & 1u;
    uint32_t ok;
    do {
      asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(ok) : "r"(bar), "r"(par) : "memory");
    } while (!ok);
    phase ^= 1u << (k & 1);
  }
  __device__ __forceinline__ void begin(const uint64_t *src, int n) {
    gsrc = src; nchunks = n; chunk = 0; pos = 0;
    __syncthreads();                                   // nobody still reads the buffers of the previous point
    if (threadIdx.x == 0) { issue(0); if (n > 1) issue(1); }
    wait(0);
  }
  __device__ __forceinline__ void advance() {          // the current chunk is used up
    __syncthreads();
    if (threadIdx.x == 0 && chunk + 2 < nchunks) issue(chunk + 2);
    chunk++; pos = 0;
    wait(chunk);
  }
  __device__ __forceinline__ uint32_t addr() const { return s_buf + (chunk & 1) * (MQ_CHUNK_WORDS * 8) + pos * 8; }
};

// ------------------------------------------------------------------ a5: one family, static code per (c, kd)
// coefficients and index bytes come from the staged stream (shared memory, broadcast reads); the per-point
// operands r_t and beta~_tu are gathered once per family from S[index][thread] into registers
template <class T, int KD>
__device__ __forceinline__ T horner_raw(uint32_t &s_coef, const T *r) {
  if constexpr (KD == 0) { T v = T(lds_f64(s_coef)); s_coef += 8 * MQ_WL; return v; }   // the MQ_WL members of an entry are interleaved
  else if constexpr (KD == 6 && MQ_LOOPED(T)) {   // double-double: the two halves in a real loop (half the code; integer overhead is free here)
    T acc = T(0.0);
#pragma unroll 1
    for (int hh = 0; hh < 2; hh++) {
      const T lo = horner_raw<T, 4>(s_coef, r), hi = horner_raw<T, 4>(s_coef, r);
      const T t = mq_fma(hi, r[4], lo);
      acc = hh ? mq_fma(t, r[5], acc) : t;
    }
    return acc;
  } else if constexpr (KD > 4) {                     // two-stage: 2^(KD-4) sub-blocks of kd = 4, combined over the top variables
    constexpr int NS = 1 << (KD - 4);
    T s[NS];
#pragma unroll
    for (int q = 0; q < NS; q++) s[q] = horner_raw<T, 4>(s_coef, r);
#pragma unroll
    for (int i = 0; i < KD - 4; i++) {
#pragma unroll
      for (int j = 0; j < (NS >> (i + 1)); j++) s[j] = mq_fma(s[2 * j + 1], r[4 + i], s[2 * j]);
    }
    return s[0];
  } else {
    constexpr int H = 1 << (KD - 1);
    T v[H];
#pragma unroll
    for (int j = 0; j < H; j++) {
      const double2 cc = lds_f64x2(s_coef + 16 * MQ_WL * j);               // (c[j], c[j+H])
      v[j] = mq_fma_c(cc.y, r[KD - 1], cc.x, T());
    }
    s_coef += 16 * MQ_WL * H;
#pragma unroll
    for (int i = KD - 2; i >= 0; i--) {
#pragma unroll
      for (int j = 0; j < (1 << i); j++) v[j] = mq_fma(v[j + (1 << i)], r[i], v[j]);
    }
    return v[0];
  }
}
// one pairing block: its value, and l1 = sum |c| from the block's closing unit (kd = 0: |c| itself) for the round-off bound
template <class T, int KD>
__device__ __forceinline__ T horner(uint32_t &s_coef, const T *r, double &l1) {
  if constexpr (KD == 0) { const double c0 = lds_f64(s_coef); s_coef += 8 * MQ_WL; l1 = fabs(c0); return T(c0); }
  else if constexpr (KD == 1) {                    // small blocks carry no closing unit: add the |c| just loaded
    const double2 cc = lds_f64x2(s_coef); s_coef += 16 * MQ_WL;
    l1 = fabs(cc.x) + fabs(cc.y);
    return mq_fma_c(cc.y, r[0], cc.x, T());
  } else if constexpr (KD == 2) {
    const double2 c0 = lds_f64x2(s_coef), c1 = lds_f64x2(s_coef + 16 * MQ_WL); s_coef += 32 * MQ_WL;
    l1 = (fabs(c0.x) + fabs(c0.y)) + (fabs(c1.x) + fabs(c1.y));
    return mq_fma(mq_fma_c(c1.y, r[1], c1.x, T()), r[0], mq_fma_c(c0.y, r[1], c0.x, T()));
  } else {
    const T h = horner_raw<T, KD>(s_coef, r);
    l1 = lds_f64(s_coef); s_coef += 16 * MQ_WL;
    return h;
  }
}
// index of the pair (i<j) among the C(N2,2) gathered betas
template <int N2> __host__ __device__ constexpr int pair_index(int i, int j) { return i * N2 - i * (i + 1) / 2 + (j - i - 1); }
constexpr int ctz_c(unsigned x) { int n = 0; while (!(x & 1u)) { x >>= 1; n++; } return n; }

template <class T, int KD, int N2, unsigned USED, bool FIRST> struct PairRec;
template <class T, int KD, int N2, unsigned USED, bool FIRST, int F, int S> struct PairStep {
  static __device__ __forceinline__ void run(const T *b, T w, uint32_t &s_coef, const T *r, T &sum, typename MagOf<T>::type &asum) {
    if constexpr (S < N2) {
      if constexpr (!((USED >> S) & 1u)) {
        if constexpr (FIRST) PairRec<T, KD, N2, (USED | (1u << F) | (1u << S)), false>::run(b, b[pair_index<N2>(F, S)], s_coef, r, sum, asum);
        else PairRec<T, KD, N2, (USED | (1u << F) | (1u << S)), false>::run(b, mq_mul(w, b[pair_index<N2>(F, S)]), s_coef, r, sum, asum);
      }
      PairStep<T, KD, N2, USED, FIRST, F, S + 1>::run(b, w, s_coef, r, sum, asum);
    }
  }
};
// sum += w_pairing * block, asum += |w_pairing| * sum|c|  (the latter bounds the block by sum|c| prod max(1,|r|), applied by the caller)
template <class T, int KD, int N2, unsigned USED, bool FIRST> struct PairRec {
  static __device__ __forceinline__ void run(const T *b, T w, uint32_t &s_coef, const T *r, T &sum, typename MagOf<T>::type &asum) {
    if constexpr (USED == ((1u << N2) - 1u)) {
      double l1;
      T h = horner<T, KD>(s_coef, r, l1);
      if constexpr (FIRST) { sum = h; asum = typename MagOf<T>::type(l1); }   // FIRST at a leaf: no pairs, one block
      else { sum = mq_fma(w, h, sum); asum = mq_mfma(mq_absd(w), l1, asum); }
    } else {
      constexpr int F = ctz_c(~USED);
      PairStep<T, KD, N2, USED, FIRST, F, F + 1>::run(b, w, s_coef, r, sum, asum);
    }
  }
};

// ---- looped pairings for c >= 3 in double-double -------------------------------------------------------------------
// Fully unrolled, the (2c-1)!! pairings of c = 3, 4 make the double-double evaluator ~1 MB of straight-line code, far
// beyond the instruction caches (ncu: "no instruction" was its largest stall). In double-double one coefficient costs
// ~11 FP64 instructions, so a few integer instructions per pairing are free: the outer levels of the pairing recursion
// become real loops over "pair the first free slot with the j-th later one", each iteration gathers the beta~ it needs
// through a static position table (positions in the member's index bytes), and only the last level (three pairings of
// four slots) is unrolled. Same pairing order as the canonical recursion, so the coefficient layout is unchanged.
struct PairTbl3 { uint8_t p[5][7]; };            // c = 3: iteration j pairs slot 0 with slot j+1; [0] = that beta, [1..6] = ab ac ad bc bd cd of the other four
struct PairTbl4 { uint8_t o[7]; uint8_t p[7][5][7]; };
constexpr PairTbl3 make_tbl3() {
  PairTbl3 t{};
  for (int j = 0; j < 5; j++) {
    int rest[4] = {0, 0, 0, 0}, n = 0;
    for (int e = 1; e < 6; e++) if (e != j + 1) rest[n++] = e;
    t.p[j][0] = (uint8_t)pair_index<6>(0, j + 1);
    int k = 1;
    for (int x = 0; x < 4; x++) for (int y = x + 1; y < 4; y++) t.p[j][k++] = (uint8_t)pair_index<6>(rest[x], rest[y]);
  }
  return t;
}
constexpr PairTbl4 make_tbl4() {
  PairTbl4 t{};
  for (int j1 = 0; j1 < 7; j1++) {
    int r6[6] = {0, 0, 0, 0, 0, 0}, n = 0;
    for (int e = 1; e < 8; e++) if (e != j1 + 1) r6[n++] = e;
    t.o[j1] = (uint8_t)pair_index<8>(0, j1 + 1);
    for (int j2 = 0; j2 < 5; j2++) {
      int rest[4] = {0, 0, 0, 0}, m = 0;
      for (int e = 1; e < 6; e++) if (e != j2 + 1) rest[m++] = r6[e];
      t.p[j1][j2][0] = (uint8_t)pair_index<8>(r6[0], r6[j2 + 1]);
      int k = 1;
      for (int x = 0; x < 4; x++) for (int y = x + 1; y < 4; y++) t.p[j1][j2][k++] = (uint8_t)pair_index<8>(rest[x], rest[y]);
    }
  }
  return t;
}
__constant__ PairTbl3 c_tbl3 = make_tbl3();
__constant__ PairTbl4 c_tbl4 = make_tbl4();

// the three pairings of four slots a<b<c<d, each with prefix weight wp: g = (ab, ac, ad, bc, bd, cd)
template <class T, int KD>
__device__ __forceinline__ void pair_body4(T wp, const T *g, uint32_t &s_coef, const T *r, T &sum, typename MagOf<T>::type &asum) {
  double l1; T w;
  w = mq_mul(mq_mul(wp, g[0]), g[5]); sum = mq_fma(w, horner<T, KD>(s_coef, r, l1), sum); asum = mq_mfma(mq_absd(w), l1, asum);     // (ab)(cd)
  w = mq_mul(mq_mul(wp, g[1]), g[4]); sum = mq_fma(w, horner<T, KD>(s_coef, r, l1), sum); asum = mq_mfma(mq_absd(w), l1, asum);     // (ac)(bd)
  w = mq_mul(mq_mul(wp, g[2]), g[3]); sum = mq_fma(w, horner<T, KD>(s_coef, r, l1), sum); asum = mq_mfma(mq_absd(w), l1, asum);     // (ad)(bc)
}

// byte i (compile-time) of an array of 64-bit index words: one PRMT
template <int I> __device__ __forceinline__ uint32_t idx_byte(const uint64_t *iw) {
  const uint32_t w = (I & 4) ? (uint32_t)(iw[I >> 3] >> 32) : (uint32_t)iw[I >> 3];
  return __byte_perm(w, 0u, 0x4440u | (uint32_t)(I & 3));
}
template <class T, int N, int OFF, int I = 0> struct Gather {
  static __device__ __forceinline__ void run(const uint64_t *iw, uint32_t s_S, uint32_t sstride, T *out) {
    if constexpr (I < N) { out[I] = SAcc<T>::lds(s_S + idx_byte<OFF + I>(iw) * sstride, sstride); Gather<T, N, OFF, I + 1>::run(iw, s_S, sstride, out); }
  }
};

// value of a family and its round-off magnitude a = sum_pairings |w| sum|c|; times Rp = prod over the lines of the piece of
// max(1,|r_t|) (applied once per table) it bounds the sum of |monomial|
template <class T> struct FamRes { T v; typename MagOf<T>::type a; };
// s_idx: shared address of the index bytes; s_coef: of the coefficients; s_S: of this thread's S[0]; sstride: bytes per S index
template <class T, int C, int KD>
__device__ __forceinline__ FamRes<T> family_eval(uint64_t w0, uint64_t w1, uint32_t s_idx, uint32_t s_coef, uint32_t s_S, uint32_t sstride) {
  constexpr int N2 = 2 * C, NB = C * (2 * C - 1), NI = NB + KD, NW = (NI + 7) / 8;
  FamRes<T> res;
  if constexpr (C >= 3 && MQ_LOOPED(T)) {
    T r[KD > 0 ? KD : 1];
#pragma unroll
    for (int i = 0; i < KD; i++) r[i] = SAcc<T>::lds(s_S + lds_u8(s_idx + NB + i) * sstride, sstride);
    T sum = T(0.0); typename MagOf<T>::type asum(0.0);
    if constexpr (C == 3) {
#pragma unroll 1
      for (int j = 0; j < 5; j++) {
        T g[7];
#pragma unroll
        for (int k = 0; k < 7; k++) g[k] = SAcc<T>::lds(s_S + lds_u8(s_idx + c_tbl3.p[j][k]) * sstride, sstride);
        pair_body4<T, KD>(g[0], g + 1, s_coef, r, sum, asum);
      }
    } else {
#pragma unroll 1
      for (int j1 = 0; j1 < 7; j1++) {
        const T w1 = SAcc<T>::lds(s_S + lds_u8(s_idx + c_tbl4.o[j1]) * sstride, sstride);
#pragma unroll 1
        for (int j2 = 0; j2 < 5; j2++) {
          T g[7];
#pragma unroll
          for (int k = 0; k < 7; k++) g[k] = SAcc<T>::lds(s_S + lds_u8(s_idx + c_tbl4.p[j1][j2][k]) * sstride, sstride);
          pair_body4<T, KD>(mq_mul(w1, g[0]), g + 1, s_coef, r, sum, asum);
        }
      }
    }
    res.v = sum; res.a = asum;                       // the factor prod max(1,|r_inner|) is applied per piece (piece_scalars: Rp)
  } else {
    uint64_t iw[NW > 2 ? NW : 2];
    iw[0] = w0; iw[1] = w1;                          // the first 16 index bytes were prefetched with the header
#pragma unroll
    for (int k = 2; k < NW; k++) iw[k] = lds_u64(s_idx + 8 * k);
    T b[NB > 0 ? NB : 1], r[KD > 0 ? KD : 1];
    Gather<T, NB, 0>::run(iw, s_S, sstride, b);
    Gather<T, KD, NB>::run(iw, s_S, sstride, r);
    T sum = T(0.0); typename MagOf<T>::type asum(0.0);
    PairRec<T, KD, N2, 0u, true>::run(b, T(1.0), s_coef, r, sum, asum);
    res.v = sum; res.a = asum;                       // the factor prod max(1,|r_inner|) is applied per piece (piece_scalars: Rp)
  }
  return res;
}

// Entry-parallel family evaluation (quad-double tier): member m of the stream entry at ent (GLOBAL memory), scalars from
// S[index * stride] (shared). Loop-based (no unrolling); same arithmetic and pairing order as family_eval (the first free
// element pairs with every later one); the scalar factors are applied here and
// the accumulation key (output, pattern, grade) of the member is returned in key.
template <class T>
__device__ __noinline__ T family_spread(const uint64_t *ent, uint64_t hd, int m, const T *S, int stride, int &key, double &amag) {
  const int c = (int)(hd & 7), kd = (int)(hd >> 3 & 7), idxw = (int)(hd >> 16 & 0xFFFF);
  const uint64_t ml = ent[m];
  const uint8_t *idx = reinterpret_cast<const uint8_t *>(ent + MQ_WL + (size_t)idxw * m);
  const double *coef = reinterpret_cast<const double *>(ent + MQ_WL * (1 + idxw)) + (kd ? 2 : 1) * m;
  key = (int)((ml & 7) | ((ml >> 6 & 15) << 3) | ((ml >> 14 & 1) << 7));
  const int n2 = 2 * c, nb = c * (2 * c - 1), nblk = 1 << kd, ns = (int)(ml >> 10 & 15);
  T b[28], r[6], v[8];
  for (int i = 0; i < nb; i++) b[i] = S[(int)idx[i] * stride];
  for (int i = 0; i < kd; i++) r[i] = S[(int)idx[nb + i] * stride];
  auto block_at = [&](const double *a, int kk) -> T {      // one block of kk <= 4 inner variables
    if (kk == 0) return T(a[0]);
    const int H = 1 << (kk - 1);
    for (int j = 0; j < H; j++) v[j] = mq_fma_c(a[2 * MQ_WL * j + 1], r[kk - 1], a[2 * MQ_WL * j], T());
    for (int i = kk - 2; i >= 0; i--) for (int j = 0; j < (1 << i); j++) v[j] = mq_fma(v[j + (1 << i)], r[i], v[j]);
    return v[0];
  };
  const int blk = kd >= 3 ? MQ_WL * (nblk + 2) : MQ_WL * nblk;       // doubles per pairing block incl. the closing (sum |c|, 0) unit of kd >= 3
  auto l1_at = [&](const double *a) -> double {
    if (kd >= 3) return a[MQ_WL * nblk];
    if (kd == 0) return fabs(a[0]);
    double t = 0.0;
    for (int j = 0; j < nblk / 2; j++) t += fabs(a[2 * MQ_WL * j]) + fabs(a[2 * MQ_WL * j + 1]);
    return t;
  };
  auto horner_at = [&](const double *a) -> T {
    if (kd <= 4) return block_at(a, kd);
    T s[4];                                                 // kd = 5, 6: sub-blocks of kd = 4, combined over r[4], r[5]
    const int nsub = 1 << (kd - 4);
    for (int q = 0; q < nsub; q++) s[q] = block_at(a + 16 * MQ_WL * q, 4);
    for (int i = 0; i < kd - 4; i++) for (int j = 0; j < (nsub >> (i + 1)); j++) s[j] = mq_fma(s[2 * j + 1], r[4 + i], s[2 * j]);
    return s[0];
  };
  T sum = T(0.0); double asum = 0.0;
  if (c == 0) { sum = horner_at(coef); asum = l1_at(coef); }
  else {
    T w[5]; unsigned used[5]; int scur[5];
    int level = 0; used[0] = 0u; w[0] = T(1.0); scur[0] = -1;
    while (level >= 0) {
      const unsigned u = used[level]; const int f = __ffs(~u) - 1;
      int s2 = scur[level] < 0 ? f + 1 : scur[level] + 1;
      while (s2 < n2 && (u >> s2 & 1u)) s2++;
      if (s2 >= n2) { level--; continue; }
      scur[level] = s2;
      const T wn = w[level] * b[f * n2 - f * (f + 1) / 2 + (s2 - f - 1)];
      if (level == c - 1) { sum = sum + wn * horner_at(coef); asum += fabs(mq_to_double(wn)) * l1_at(coef); coef += blk; }
      else { level++; used[level] = u | 1u << f | 1u << s2; w[level] = wn; scur[level] = -1; }
    }
  }
  for (int i = 0; i < kd; i++) asum *= fmax(1.0, fabs(mq_to_double(r[i])));
  for (int i = 0; i < ns; i++) { const T sc = S[(int)idx[nb + kd + i] * stride]; sum = sum * sc; asum *= fabs(mq_to_double(sc)) + 0.125; }
  amag = asum;
  return sum;
}

// ------------------------------------------------------------------ a5: the entries of one table, run by run
// The entries of a table come in runs of equal shape (c, kd): host_prepare.cpp sorts shape-major and stores in every header
// the number of entries left in its run. The shape switch is taken once per RUN and each shape has its own loop over the
// run's entries, which carries a handful of values (stream position, count, accumulation key, run accumulator) next to the
// family body's registers. (Round 1 took the switch per entry through a call: its loop state lived in local memory and every
// entry paid a chain of local-memory round trips, ~1800 cycles per entry whatever the arithmetic inside.)
// A run of families with the same (output, pattern, grade) accumulates in registers; the accumulator is (re)loaded from N
// when the key changes, BEFORE the family is evaluated, so that the local-memory load has the whole evaluation to complete.
#ifndef MQ_RUNS
#define MQ_RUNS 1
#endif
template <class T> struct RunAcc { int key; T racc; typename MagOf<T>::type racca; };

template <class T, int C, int KD>
__device__ __forceinline__ void run_loop(StreamReader &rd, int count, int sub, uint32_t s_S, uint32_t sstride,
                                         T (*N)[MQ_MAXPAT][MQ_NGRADE], typename MagOf<T>::type (*Na)[MQ_MAXPAT][MQ_NGRADE], RunAcc<T> &ra) {
  using M = typename MagOf<T>::type;
  constexpr int NI = C * (2 * C - 1) + KD;
  int pos = rd.pos;
  uint32_t base = rd.addr() - 8u * (uint32_t)pos;              // shared address of word 0 of the current chunk
  int key = ra.key; T racc = ra.racc; M racca = ra.racca;
#pragma unroll 1
  for (int i = 0; i < count;) {
    if (pos == MQ_CHUNK_WORDS) { rd.pos = pos; rd.advance(); pos = 0; base = rd.addr(); }
    const uint32_t a0 = base + 8u * (uint32_t)pos;
    const uint64_t hd = lds_u64(a0);
    const uint32_t idxw = (uint32_t)(hd >> 16 & 0xFFFF);
    if ((int)(hd & 7) == MQ_PAD_MARK) { pos += 1 + (int)idxw; continue; }
    const uint64_t hl = lds_u64(a0 + 8u * (uint32_t)sub);
    MQ_DASSERT(pos >= 0 && pos + MQ_WL * (1 + (int)idxw) + (int)(hd >> 32 & 0xFFFF) <= MQ_CHUNK_WORDS);   // an entry never straddles a chunk
    MQ_DASSERT((int)(hd & 7) == C && (int)(hd >> 3 & 7) == KD && (int)idxw * 8 >= NI + (int)(hl >> 10 & 15));
    const uint32_t sidx = a0 + 8u * MQ_WL + 8u * idxw * (uint32_t)sub;
    const uint64_t w0 = lds_u64(sidx), w1 = lds_u64(sidx + 8);
    const uint32_t scoef = a0 + 8u * MQ_WL * (1u + idxw) + (KD ? 16u : 8u) * (uint32_t)sub;
    const int keyk = (int)((hl & 7) | ((hl >> 6 & 15) << 3) | ((hl >> 14 & 1) << 7));
    MQ_DASSERT((keyk & 7) < MQ_NGRADE && ((keyk >> 3) & 15) < MQ_MAXPAT && (keyk >> 7) < 2);
#if MQ_DEVICE_ASSERTS
    for (int j = 0; j < NI + (int)(hl >> 10 & 15); j++) MQ_DASSERT((int)lds_u8(sidx + j) < rd.dbg_scal_len);
#endif
    if (keyk != key) {
      if (key >= 0) { N[key >> 7][(key >> 3) & 15][key & 7] = racc; Na[key >> 7][(key >> 3) & 15][key & 7] = racca; }
      key = keyk; racc = N[key >> 7][(key >> 3) & 15][key & 7]; racca = Na[key >> 7][(key >> 3) & 15][key & 7];
    }
    const FamRes<T> fr = family_eval<T, C, KD>(w0, w1, sidx, scoef, s_S, sstride);
    T val = mq_norm(fr.v); M amag = fr.a;             // the family code works on unnormalised pairs (dd_arith.cuh)
    const int ns = (int)(hl >> 10 & 15);
#pragma unroll 1
    for (int j = 0; j < ns; j++) {                    // scalar factors; + 1/8: the factor's own absolute round-off (A_t = 1 - x_t may be tiny)
      const T sc = SAcc<T>::lds(s_S + lds_u8(sidx + NI + j) * sstride, sstride);
      val = val * sc; amag = amag * (mq_absd(sc) + M(0.125));
    }
    racc = racc + val; racca += amag;                 // racca: sum of |monomial| bounds, sees the cancellation inside a family too
    pos += MQ_WL * (1 + (int)idxw) + (int)(hd >> 32 & 0xFFFF);
    i++;
  }
  rd.pos = pos;
  ra.key = key; ra.racc = racc; ra.racca = racca;
}
template <class T>
__device__ __forceinline__ void run_dispatch(int ckd, StreamReader &rd, int count, int sub, uint32_t s_S, uint32_t sstride,
                                             T (*N)[MQ_MAXPAT][MQ_NGRADE], typename MagOf<T>::type (*Na)[MQ_MAXPAT][MQ_NGRADE], RunAcc<T> &ra) {
  switch (ckd) {     // key = c*8 + kd; the inner dimension kd is capped per c by mq_kd_max (device_layout.h)
#define MQ_CASE(C, K) case C * 8 + K: run_loop<T, C, K>(rd, count, sub, s_S, sstride, N, Na, ra); return;
#define MQ_ROW(C) MQ_CASE(C, 0) MQ_CASE(C, 1) MQ_CASE(C, 2)
    MQ_ROW(0) MQ_ROW(1) MQ_ROW(2) MQ_ROW(3) MQ_ROW(4)
    MQ_CASE(0, 3) MQ_CASE(0, 4) MQ_CASE(0, 5) MQ_CASE(0, 6) MQ_CASE(1, 3) MQ_CASE(1, 4) MQ_CASE(1, 5) MQ_CASE(1, 6)
    MQ_CASE(2, 3) MQ_CASE(2, 4) MQ_CASE(2, 5) MQ_CASE(2, 6) MQ_CASE(3, 3) MQ_CASE(3, 4)
#undef MQ_ROW
#undef MQ_CASE
  }
  __trap();          // a family shape the tables must never contain
}

// ------------------------------------------------------------------ a4: scalars of one piece
// accessors to the piece's scalar array S[index] of one point group: the whole element of type T, or (SComp) one binary64
// component of ptn<N> elements: the lane computes the scalars of ONE of the group's points in plain binary64
template <class T> struct SWhole {
  unsigned char *S; int stride;
  __device__ __forceinline__ void st(int i, T v) const { SAcc<T>::st(S, i, stride, v); }
  __device__ __forceinline__ T ld(int i) const { return SAcc<T>::ld(S, i, stride); }
};
template <int N> struct SComp {
  double *base; size_t istride;            // element i, point k of the group: plane k/2 of index i, half k&1 of the 16-byte unit
  __device__ __forceinline__ SComp(unsigned char *S, int stride, int k) : base(reinterpret_cast<double *>(S) + (size_t)(k >> 1) * stride * 2 + (k & 1)), istride((size_t)N * stride) {}
  __device__ __forceinline__ void st(int i, double v) const { base[(size_t)i * istride] = v; }
  __device__ __forceinline__ double ld(int i) const { return base[(size_t)i * istride]; }
};
// writes S = [ r_t | A_t | A'_t/g_t | beta_tu/(g_t g_u) (t<u) ] and returns U, V, G = prod_lines g_t, Rp = prod_lines max(1,|r_t|)
template <class T, class ACC>
__device__ __forceinline__ void piece_scalars(const DevGeom &g, const typename MagOf<T>::type *z, const ACC acc, bool wr, T &U, T &V, T &G,
                                              typename MagOf<T>::type &Rp, typename MagOf<T>::type &amin, typename MagOf<T>::type &xmin) {
  using M = typename MagOf<T>::type;
  const int n = g.nch, ns = g.nslot;
  T A[MQ_MAXL][MQ_MAXL], Inv[MQ_MAXL][MQ_MAXL];
#pragma unroll
  for (int i = 0; i < MQ_MAXL; i++)
#pragma unroll
    for (int j = 0; j < MQ_MAXL; j++) { A[i][j] = T(0.0); Inv[i][j] = T(i == j ? 1.0 : 0.0); }
  for (int s = 0; s < ns; s++) {
    if (g.slot[s].kind != MQ_SLOT_LINE) continue;
    const uint32_t e = g.slot[s].eps; const T zt = T(z[g.slot[s].zline]);
#pragma unroll
    for (int i = 0; i < MQ_MAXL; i++)
#pragma unroll
      for (int j = 0; j < MQ_MAXL; j++) if ((e >> i & 1u) && (e >> j & 1u)) A[i][j] = A[i][j] + zt;
  }
#pragma unroll
  for (int i = 0; i < MQ_MAXL; i++) if (i < n) A[i][i] = A[i][i] + T(z[g.chord_zline[i]]);
  // Gauss-Jordan without pivoting (A is symmetric positive definite); determinant = product of pivots.
  // pivot/original diagonal measures the relative accuracy lost in the Schur complements (O8).
  M d0[MQ_MAXL];
#pragma unroll
  for (int i = 0; i < MQ_MAXL; i++) d0[i] = mq_mag(A[i][i]);
  U = T(1.0);
#pragma unroll
  for (int c = 0; c < MQ_MAXL; c++) {
    if (c < n) {
      const T p = A[c][c]; U = U * p;
      xmin = mq_mmin(xmin, mq_mag(p) / d0[c]);
      const T ip = T(1.0) / p;
#pragma unroll
      for (int k = 0; k < MQ_MAXL; k++) { A[c][k] = A[c][k] * ip; Inv[c][k] = Inv[c][k] * ip; }
#pragma unroll
      for (int r = 0; r < MQ_MAXL; r++) if (r != c && r < n) {
        const T f = A[r][c];
#pragma unroll
        for (int k = 0; k < MQ_MAXL; k++) { A[r][k] = A[r][k] - f * A[c][k]; Inv[r][k] = Inv[r][k] - f * Inv[c][k]; }
      }
    }
  }
  // beta_su = eps_s^T Inv eps_u ; x_s = sum_lines z_u beta_su ; A'_s = (sgn_s - sum_lines z_u beta_su sgn_u)/2
  T ig[MQ_MAXSLOT];
  V = T(0.0); G = T(1.0); Rp = M(1.0);
  const int off_at = g.off_at, off_aq = g.off_aq, off_bt = g.off_bt;
  for (int s = 0; s < ns; s++) {
    const uint32_t es = g.slot[s].eps;
    T w[MQ_MAXL];
#pragma unroll
    for (int j = 0; j < MQ_MAXL; j++) { T a = T(0.0);
#pragma unroll
      for (int i = 0; i < MQ_MAXL; i++) if (es >> i & 1u) a = a + Inv[i][j];
      w[j] = a; }
    T x = T(0.0), q = T(0.0);
    for (int u = 0; u < ns; u++) {
      const uint32_t eu = g.slot[u].eps;
      T bsu = T(0.0);
#pragma unroll
      for (int j = 0; j < MQ_MAXL; j++) if (eu >> j & 1u) bsu = bsu + w[j];
      if (g.slot[u].kind == MQ_SLOT_LINE) {
        const T zb = bsu * T(z[g.slot[u].zline]);
        x = x + zb; if (g.slot[u].sgn < 0) q = q - zb; else q = q + zb;
      }
      if (u > s && wr) acc.st(off_bt + s * ns - s * (s + 1) / 2 + (u - s - 1), bsu);   // raw beta, scaled below
    }
    const bool line = g.slot[s].kind == MQ_SLOT_LINE;
    const T gs = T(2.0) - x;
    const T igs = line ? T(1.0) / gs : T(1.0);
    ig[s] = igs;
    const T rs = x * igs;
    if (wr) acc.st(s, rs);                                              // r_t = x_t / g_t   (lines)
    if (off_at >= 0 && wr) acc.st(off_at + s, T(1.0) - x);              // A_t
    const T sg = T((double)g.slot[s].sgn);
    if (off_aq >= 0 && wr) acc.st(off_aq + s, (sg - q) * igs * T(0.5));   // A'_t / g_t
    if (line) {
      V = V + x * T(z[g.slot[s].zline]); G = G * gs;
      const M xd = mq_mag(x);
      amin = mq_mmin(amin, mq_absd(M(1.0) - xd)); xmin = mq_mmin(xmin, M(2.0) - xd);   // |A_t| (scalar factors of insertion pieces) ; g_t divides every operand of slot t
      Rp = Rp * mq_mmax1(mq_absd(rs));                                  // bounds prod |r_t|^sigma over any subset of the lines
    }
  }
  if (wr)
  for (int s = 0; s < ns; s++)
    for (int u = s + 1; u < ns; u++) {
      const int at = off_bt + s * ns - s * (s + 1) / 2 + (u - s - 1);
      acc.st(at, acc.ld(at) * ig[s] * ig[u]);
    }
}

template <class T> __device__ __forceinline__ void graded_mul(T *acc, const T *b, int nb) {   // acc <- acc (*) b, truncated at NGRADE
  T r[MQ_NGRADE];
#pragma unroll
  for (int c = 0; c < MQ_NGRADE; c++) { T s = T(0.0);
#pragma unroll
    for (int i = 0; i < MQ_NGRADE; i++) if (i <= c && c - i < nb) s = s + acc[i] * b[c - i];
    r[c] = s; }
#pragma unroll
  for (int c = 0; c < MQ_NGRADE; c++) acc[c] = r[c];
}

// ------------------------------------------------------------------ a4-a6: integrand at one point
// S: shared-memory scalar scratch of this thread (S[index*stride]); nodeval / nodeU / nodeV: per-thread local arrays.
// For T = double a second, sign-free copy of the whole computation is carried along at family granularity
// (|family value| summed, |child value| multiplied): abs_out = sum over terms and grades of that bound. It measures
// every cancellation between families, pieces and terms (O8) at the cost of one add per family.
//
// Lane split (LANES = true; binary64 and double-double kernels): MQ_WL lanes of a warp share one sample point. All of
// them compute the point's scalars (only lane role sub = 0 writes S), then each evaluates ITS member of every stream
// entry (MQ_WL same-shape families side by side, device_layout.h) from the common S[index][point]; the partial graded
// sums are added across the lane roles with warp shuffles once per table, so every lane ends with the same totals.
// This multiplies the warps per SM at constant shared memory per point (occupancy is capped by S), with no
// duplicated family work. LANES = false (quad-double): one lane per point evaluates the members one after the other.
// Warp split: W warps share one group of points. Warp gw = 0 of the group owns the points (scalars, node
// values, terms); the entries of every table are dealt round-robin to the W warps, which all read the same
// S[index][point] in shared memory; their partial graded sums are added through the exchange area xT/xA.
// CTA-collective: contains __syncthreads; every thread of the CTA must call it.
template <class T> __device__ __forceinline__ T mq_shfl_xor(T v, int m);
template <> __device__ __forceinline__ double mq_shfl_xor<double>(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }
template <> __device__ __forceinline__ pt2 mq_shfl_xor<pt2>(pt2 v, int m) { pt2 r; r.v[0] = __shfl_xor_sync(0xffffffffu, v.v[0], m); r.v[1] = __shfl_xor_sync(0xffffffffu, v.v[1], m); return r; }
template <> __device__ __forceinline__ pt4 mq_shfl_xor<pt4>(pt4 v, int m) {
  pt4 r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.v[i] = __shfl_xor_sync(0xffffffffu, v.v[i], m);
  return r;
}
template <> __device__ __forceinline__ dd mq_shfl_xor<dd>(dd v, int m) { return dd(__shfl_xor_sync(0xffffffffu, v.hi, m), __shfl_xor_sync(0xffffffffu, v.lo, m)); }

template <class T, int W, bool LANES, bool SPREAD = false>
__device__ __noinline__ void eval_integrand(const DiagView &v, StreamReader &rd_io, const typename MagOf<T>::type *z, const double *zl, unsigned char *S, int stride, T *xT, typename MagOf<T>::type *xA, int gw, int sub,
                                            T &f_out, T &abs_out, typename MagOf<T>::type &amin_out, typename MagOf<T>::type &xmin_out) {
  static_assert(W == 1, "the warp split (W warps per point group) was measured slower and is gone");
  constexpr bool TRACK = true;
  using M = typename MagOf<T>::type;                   // magnitudes (round-off bounds, pivot ratios): one per sample point of the lane
  // DIST: the MQ_WL lanes of a point group carry MQ_WL points; lane role `sub` computes the scalars of point `sub` in plain
  // binary64 from zl (its coordinates) and writes that component of S; U, V, G, Rp are gathered with shuffles. Otherwise all
  // lanes compute all points of the group from z (role 0 writes).
  constexpr int NPT = PtsOf<T>::n;
  constexpr bool DIST = LANES && !SPREAD && NPT > 1 && NPT == MQ_WL;
  StreamReader rd = rd_io;                             // work on a register copy (the caller's object lives in local memory across this call)
  const DevHeader &h = *v.h;
  // node values: per lane. DIST: lane role k assembles the nodes and terms of point k in plain binary64 (TT = MM = double), so
  // the four roles share that work too and the per-thread arrays are binary64; otherwise the owner lane does all points
  using TT = typename std::conditional<DIST, double, T>::type;
  using MM = typename std::conditional<DIST, double, M>::type;
  TT nodeval[MQ_MAXNODEVAL];
  MM nodeabs[TRACK ? MQ_MAXNODEVAL : 1];
  TT nodeU[MQ_MAXNODE], nodeV[MQ_MAXNODE];
  M amin(1.0), xmin(1.0);
  double amin_l = 1.0, xmin_l = 1.0;                   // DIST: of this lane's point
  const bool owner = gw == 0 && sub == 0 && (!SPREAD || threadIdx.x == 0);   // the lane whose f_out is used
  const uint32_t s_S = smem_u32(S), sstride = (uint32_t)(stride * sizeof(T));
  rd.begin(v.blob + h.off_stream, (int)h.stream_chunks);
  for (int gi = 0; gi < h.ngeom; gi++) {
    const DevGeom &g = v.geom[gi];
    MQ_DASSERT(g.scal_len <= h.max_scal_len && g.nslot <= MQ_MAXSLOT && g.nch <= MQ_MAXL && g.nS <= 4 && g.nchild <= MQ_MAXCHILD);
    T U = T(1.0), V = T(0.0), G = T(1.0); M Rp(1.0);
    if constexpr (LANES) __syncwarp();                 // every lane role has finished reading S of the previous piece
    if constexpr (SPREAD) __syncthreads();             // (entry-parallel) nobody still reads S of the previous piece
    double Ul = 1.0, Vl = 0.0, Gl = 1.0, Rl = 1.0;              // DIST: U, V, G, Rp of this lane's point
    if constexpr (DIST) piece_scalars<double>(g, zl, SComp<NPT>(S, stride, sub), true, Ul, Vl, Gl, Rl, amin_l, xmin_l);
    else piece_scalars<T>(g, z, SWhole<T>{S, stride}, SPREAD ? threadIdx.x == 0 : sub == 0, U, V, G, Rp, amin, xmin);
    if constexpr (SPREAD) __syncthreads();              // S of this piece is complete before any warp gathers from it
    else if constexpr (LANES) __syncwarp();
    const int npat = 1 << g.nS;
    for (int ti = g.first_table; ti < g.first_table + g.ntable; ti++) {
      const DevTable &tb = v.tab[ti];
      MQ_DASSERT(ti < h.ntable && tb.nout >= 1 && tb.nout <= 2 && npat <= MQ_MAXPAT && tb.geom == gi);
      T N[2][MQ_MAXPAT][MQ_NGRADE];
      M Na[TRACK ? 2 : 1][TRACK ? MQ_MAXPAT : 1][MQ_NGRADE];
      for (int o = 0; o < tb.nout; o++) for (int p = 0; p < npat; p++)
#pragma unroll
          for (int c = 0; c < MQ_NGRADE; c++) { N[o][p][c] = T(0.0); if constexpr (TRACK) Na[o][p][c] = M(0.0); }
      // entries of this table from the staged stream; a run of families with the same (output, pattern, grade)
      // accumulates in registers and is flushed when the key changes
      if constexpr (SPREAD) {
        // entry-parallel: the whole CTA works on ONE point; every thread walks the staged stream (headers only), takes the
        // entries with index = its thread id (mod CTA size) and evaluates them from global memory once a full round is dealt
        const uint64_t *pend = nullptr; uint64_t pend_h = 0;
        auto flush_round = [&]() {
          if (pend) {
#pragma unroll 1
            for (int m = 0; m < MQ_WL; m++) {
              int kk; double am;
              const T val = family_spread<T>(pend, pend_h, m, reinterpret_cast<const T *>(S), stride, kk, am);
              N[kk >> 7][(kk >> 3) & 15][kk & 7] = N[kk >> 7][(kk >> 3) & 15][kk & 7] + val;
              if constexpr (TRACK) Na[kk >> 7][(kk >> 3) & 15][kk & 7] += M(am);
            }
            pend = nullptr;
          }
        };
        unsigned unit = 0;
        for (int left = tb.nfam; left > 0;) {
          if (rd.pos == MQ_CHUNK_WORDS) rd.advance();
          const uint64_t hd = lds_u64(rd.addr());
          const int idxw = (int)(hd >> 16 & 0xFFFF);
          if ((int)(hd & 7) == MQ_PAD_MARK) { rd.pos += 1 + idxw; continue; }
          if (unit % blockDim.x == threadIdx.x) { pend = rd.gsrc + (size_t)rd.chunk * MQ_CHUNK_WORDS + rd.pos; pend_h = hd; }
          rd.pos += MQ_WL * (1 + idxw) + (int)(hd >> 32 & 0xFFFF); left--; unit++;
          if (unit % blockDim.x == 0) flush_round();
        }
        flush_round();
        // CTA-wide sum of the partial graded sums: warp butterflies, then the warp totals through xT / xA; every thread ends
        // with the same totals
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
        const int ne = tb.nout * npat * MQ_NGRADE;
        for (int e = 0; e < ne; e++) {
          const int o = e / (npat * MQ_NGRADE), p = (e / MQ_NGRADE) % npat, c = e % MQ_NGRADE;
          T t = N[o][p][c]; M ta = Na[o][p][c];
          for (int m = 1; m < 32; m <<= 1) { t = t + mq_shfl_xor<T>(t, m); ta += mq_shfl_xor<M>(ta, m); }
          if (lane == 0) { xT[wid * ne + e] = t; xA[wid * ne + e] = ta; }
        }
        __syncthreads();
        for (int e = 0; e < ne; e++) {
          const int o = e / (npat * MQ_NGRADE), p = (e / MQ_NGRADE) % npat, c = e % MQ_NGRADE;
          T t = xT[e]; M ta = xA[e];
          for (int w = 1; w < nw; w++) { t = t + xT[w * ne + e]; ta += xA[w * ne + e]; }
          N[o][p][c] = t; Na[o][p][c] = ta;
        }
        __syncthreads();
      } else {
        static_assert(SPREAD || LANES, "one lane per point without the lane split is not supported any more");
        RunAcc<T> ra; ra.key = -1; ra.racc = T(0.0); ra.racca = M(0.0);
        for (int left = tb.nfam; left > 0;) {
          if (rd.pos == MQ_CHUNK_WORDS) rd.advance();
          const uint64_t hd = lds_u64(rd.addr());
          if ((int)(hd & 7) == MQ_PAD_MARK) { rd.pos += 1 + (int)(hd >> 16 & 0xFFFF); continue; }
          const int run = (int)(hd >> 48);
          run_dispatch<T>((int)(hd & 7) * 8 + (int)(hd >> 3 & 7), rd, run, sub, s_S, sstride, N, Na, ra);
          left -= run;
        }
        if (ra.key >= 0) { N[ra.key >> 7][(ra.key >> 3) & 15][ra.key & 7] = ra.racc; Na[ra.key >> 7][(ra.key >> 3) & 15][ra.key & 7] = ra.racca; }
      }
      if constexpr (LANES && MQ_WL > 1) {              // add the partial sums of the lane roles: afterwards every lane holds the totals
        for (int o = 0; o < tb.nout; o++) for (int p = 0; p < npat; p++)
#pragma unroll
          for (int c = 0; c < MQ_NGRADE; c++) {
#pragma unroll
            for (int m = 32 / MQ_WL; m < 32; m <<= 1) {
              N[o][p][c] = N[o][p][c] + mq_shfl_xor<T>(N[o][p][c], m);
              if constexpr (TRACK) Na[o][p][c] += mq_shfl_xor<M>(Na[o][p][c], m);
            }
          }
      }
      if constexpr (!SPREAD && !DIST) {                // the families' magnitudes leave out prod max(1,|r_inner|) <= Rp (DIST: applied at the assembly)
        for (int o = 0; o < tb.nout; o++) for (int p = 0; p < npat; p++)
#pragma unroll
          for (int c = 0; c < MQ_NGRADE; c++) Na[o][p][c] = Na[o][p][c] * Rp;
      }
      if (tb.nout == 1 && (tb.op == MQ_OP_U || tb.op == MQ_OP_LMU)) {   // these tables hold 12*coefficient (coef_gen.hpp)
        const T i12 = T(1.0) / T(12.0);
        for (int p = 0; p < npat; p++)
#pragma unroll
          for (int c = 0; c < MQ_NGRADE; c++) { N[0][p][c] = N[0][p][c] * i12; if constexpr (TRACK) Na[0][p][c] = Na[0][p][c] * M(1.0 / 12.0); }
      }
      // nodes that use this table: combine with the children's graded values. DIST: every lane role does it for its own point
      // (component `sub` of the totals, binary64); otherwise only the owner lane of a point (the other roles hold the same totals)
      auto nval = [&](const T &x) -> TT { if constexpr (DIST) return mq_comp(x, sub); else return x; };
      auto naval = [&](const M &x) -> MM { if constexpr (DIST) return mq_comp(x, sub) * Rl; else return x; };
      TT Uq, Vq, Gq;
      if constexpr (DIST) { Uq = Ul; Vq = Vl; Gq = Gl; } else { Uq = U; Vq = V; Gq = G; }
      if (DIST || owner)
      for (int ni = tb.first_node; ni < tb.first_node + tb.nnode; ni++) {
        const DevNode &nd = v.node[ni];
        MQ_DASSERT(ni < MQ_MAXNODE && ni < h.nnode && nd.ngr <= MQ_NGRADE && nd.nout <= tb.nout && nd.val_off >= 0 && nd.val_off + nd.nout * nd.ngr <= MQ_MAXNODEVAL);
        for (int k = 0; k < nd.nchild; k++) MQ_DASSERT(nd.child[k] >= 0 && nd.child[k] < ni);      // children are assembled before their parent
        TT Up = Uq, Vs = Vq;
        for (int k = 0; k < nd.nchild; k++) { Up = Up * nodeU[nd.child[k]]; Vs = Vs + nodeV[nd.child[k]]; }
        nodeU[ni] = Up; nodeV[ni] = Vs;
        for (int o = 0; o < nd.nout; o++) {
          TT tot[MQ_NGRADE]; MM tota[MQ_NGRADE];
#pragma unroll
          for (int c = 0; c < MQ_NGRADE; c++) { tot[c] = TT(0.0); tota[c] = MM(0.0); }
          for (int p = 0; p < npat; p++) {
            TT acc[MQ_NGRADE]; MM acca[MQ_NGRADE];
#pragma unroll
            for (int c = 0; c < MQ_NGRADE; c++) { acc[c] = nval(N[o][p][c]) * Gq; if constexpr (TRACK) acca[c] = naval(Na[o][p][c]) * mq_mag(Gq); }
            for (int k = 0; k < nd.nchild; k++) {
              const DevNode &ch = v.node[nd.child[k]];
              const int pb = g.child_patbit[k];
              const int which = (pb >= 0 && (p >> pb & 1)) ? 1 : 0;      // S-child: a (0) or b (1); V-child: its single value
              graded_mul<TT>(acc, &nodeval[ch.val_off + which * ch.ngr], ch.ngr);
              if constexpr (TRACK) graded_mul<MM>(acca, &nodeabs[ch.val_off + which * ch.ngr], ch.ngr);
            }
#pragma unroll
            for (int c = 0; c < MQ_NGRADE; c++) { tot[c] = tot[c] + acc[c]; if constexpr (TRACK) tota[c] += acca[c]; }
          }
          for (int c = 0; c < nd.ngr; c++) { nodeval[nd.val_off + o * nd.ngr + c] = tot[c]; if constexpr (TRACK) nodeabs[nd.val_off + o * nd.ngr + c] = tota[c]; }
        }
      }
    }
  }
  // a6: terms.  f = sum sign * sum_{c<L} (L-c-1)! N_c / (Uprod^2 Vsum^(L-c))
  const int L = h.L;
  TT f = TT(0.0), asum = TT(0.0);
  if (DIST || owner)
  for (int t = 0; t < h.nterm; t++) {
    const DevTerm tm = v.term[t];
    MQ_DASSERT(tm.root >= 0 && tm.root < h.nnode && tm.root < MQ_MAXNODE);
    const DevNode &nd = v.node[tm.root];
    const TT U2 = nodeU[tm.root] * nodeU[tm.root], Vs = nodeV[tm.root];
    TT Vp = TT(1.0);
    double fact = 1.0;
    for (int c = L - 1; c >= 0; c--) {
      Vp = Vp * Vs;
      if (L - c - 1 > 0) fact *= (double)(L - c - 1);
      const TT scale = TT(fact * (double)tm.sign) / (U2 * Vp);
      const TT contrib = (c < nd.ngr ? nodeval[nd.val_off + c] : TT(0.0)) * scale;
      f = f + contrib;
      if constexpr (TRACK) asum = asum + TT(c < nd.ngr ? nodeabs[nd.val_off + c] * mq_absd(mq_mag(scale)) : MM(0.0));
      else asum = asum + mq_abs(contrib);
    }
  }
  // DIST: every lane returns the values of ITS point (broadcast into all components of the outputs)
  if constexpr (DIST) { f_out = T(f); abs_out = T(asum); amin_out = M(amin_l); xmin_out = M(xmin_l); rd_io = rd; return; }
  if constexpr (!DIST) { f_out = f; abs_out = asum; amin_out = amin; xmin_out = xmin; }
  rd_io = rd;
}

}  // namespace mqk
