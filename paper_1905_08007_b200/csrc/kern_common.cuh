// kern_common.cuh — pieces shared by the kernel translation units (binary64, double-double, quad-double): thread roles,
// reductions, the precision decision, the batched path's item lookup.
// Product code (libmcqed.so).
#pragma once
#include "diagram.hpp"
#include "mcqed_kernels.cuh"

namespace mqk {

struct KahanPair {   // compensated running sum (hi, lo)
  double hi, lo;
  __device__ __forceinline__ void add(double x) { dd s = dd_two_sum(hi, x); hi = s.hi; lo = __dadd_rn(lo, s.lo); }
  __device__ __forceinline__ void merge(double ohi, double olo) { dd s = dd_two_sum(hi, ohi); hi = s.hi; lo = __dadd_rn(lo, __dadd_rn(s.lo, olo)); }
};

// a7: block reduction of two compensated sums (warp shuffles, then shared memory); thread 0 writes partial[block][0..3]
// dst[0..3] = (sum hi, sum lo, sumsq hi, sumsq lo) of the CTA; callers in a loop must pass a __syncthreads between calls
__device__ __forceinline__ void block_reduce_to(KahanPair a, KahanPair b, double *dst) {
  __shared__ double red[32][4];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    double ah = __shfl_down_sync(0xffffffffu, a.hi, off), al = __shfl_down_sync(0xffffffffu, a.lo, off);
    double bh = __shfl_down_sync(0xffffffffu, b.hi, off), bl = __shfl_down_sync(0xffffffffu, b.lo, off);
    a.merge(ah, al); b.merge(bh, bl);
  }
  if (lane == 0) { red[warp][0] = a.hi; red[warp][1] = a.lo; red[warp][2] = b.hi; red[warp][3] = b.lo; }
  __syncthreads();
  if (threadIdx.x == 0) {
    KahanPair sa{0.0, 0.0}, sb{0.0, 0.0};
    for (int w = 0; w < nw; w++) { sa.merge(red[w][0], red[w][1]); sb.merge(red[w][2], red[w][3]); }
    dst[0] = sa.hi; dst[1] = sa.lo; dst[2] = sb.hi; dst[3] = sb.lo;
  }
}
__device__ __forceinline__ void block_reduce_store(KahanPair a, KahanPair b, double *partial) { block_reduce_to(a, b, partial + (size_t)blockIdx.x * 4); }

// Opt every evaluating kernel in to the device's maximum dynamic shared memory once: the attribute is per function, not
// per launch, and diagrams of different size share the kernels (a smaller diagram prepared later must not lower it).
template <class K> inline cudaError_t allow_max_smem(K kernel) {
  cudaFuncAttributes fa; cudaError_t e;
  if ((e = cudaFuncGetAttributes(&fa, kernel)) != cudaSuccess) return e;
  int dev = 0, optin = 0;
  cudaGetDevice(&dev);
  if ((e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
}

// ---- batched path (mc_batch_*): one persistent launch per precision tier serves every diagram of a batch ----
// A work item is one CTA-load of points of ONE diagram (the evaluator is CTA-collective and its table reads are
// CTA-uniform). CTAs take items from a global queue head, so diagrams of different cost balance themselves and the
// only tail is the last item of the whole batch. Every item writes its own compensated partial sums; the final
// reduction adds them in item order, so the result does not depend on which CTA ran which item.
// (BatchDiag / BatchView: diagram.hpp)
// item -> diagram for the passes whose item counts are known only on the device
__device__ __forceinline__ int batch_find(const uint32_t *start, int nd, uint32_t item) {
  int lo = 0, hi = nd;             // start[lo] <= item < start[hi]
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (start[mid] <= item) lo = mid; else hi = mid; }
  return lo;
}

// sample range of diagram d in this call: uniform (first, n) or the per-diagram arrays of mc_batch_integrate_counts
__device__ __forceinline__ uint64_t batch_first(const BatchView &bv, int d, uint64_t first) { return bv.v_first ? bv.v_first[d] : first; }
__device__ __forceinline__ uint64_t batch_n(const BatchView &bv, int d, uint64_t n) { return bv.v_n ? (uint64_t)bv.v_n[d] : n; }

__device__ __forceinline__ bool bad_point(const double *z, int M, double p) {   // DESIGN.md A15
  bool bad = !(p > 0.0) || !isfinite(p);
  for (int i = 0; i < M; i++) bad |= !(z[i] >= 0x1p-600);
  return bad;
}
template <int N> __device__ __forceinline__ bool bad_point(const ptn<N> *z, int k, int M, double p) {   // the same for point k of a lane that carries N
  bool bad = !(p > 0.0) || !isfinite(p);
  for (int i = 0; i < M; i++) bad |= !(mq_comp(z[i], k) >= 0x1p-600);
  return bad;
}
__device__ __forceinline__ bool bad_point(const double *z, int, int M, double p) { return bad_point(z, M, p); }

// draws the PtsOf<T>::n sample points of this lane: indices first + min(i0 + k, n - 1), k = 0, 1 (surplus slots redo the last
// point and are discarded by the caller); z[line] holds the coordinates of both, p[k] the densities
template <class T, bool WANT_ORDER>
__device__ __forceinline__ void draw_points(const DiagView &v, uint64_t first, uint64_t i0, uint64_t n, uint64_t seed, typename MagOf<T>::type *z, double *p, int32_t *order_out) {
  constexpr int NP = PtsOf<T>::n;
  if constexpr (NP == 1) p[0] = draw_point<WANT_ORDER>(v, first + (i0 < n ? i0 : n - 1), seed, z, order_out);
  else {
    const int M = v.h->M;
#pragma unroll 1
    for (int k = 0; k < NP; k++) {
      double zz[MQ_MAXM];
      p[k] = draw_point<WANT_ORDER>(v, first + (i0 + k < n ? i0 + k : n - 1), seed, zz, WANT_ORDER ? order_out + k * MQ_MAXM : nullptr);
      for (int j = 0; j < M; j++) mq_setc(z[j], k, zz[j]);
    }
  }
}

// Precision decision of one tier (O8). a = sum of |monomial| bounds carried by the evaluator (sum|c| of every
// coefficient block x |pairing weight| x |scalar factors|, through the whole tree), amin = min |A_t| over the electron lines
// of every piece, xmin = min over pieces of (pivot / diagonal of the loop-matrix elimination, g_t = 1 + A_t): the quantities
// every operand is divided by. unit = 32 (binary64) / 64 (double-double) ulp of the tier's arithmetic.
//   0: accepted, relative round-off bound met (a <= cond_max |f| min(1, amin, xmin) and min(amin, xmin) >= inner_min): with
//      cond_max = 2.8e4 = 1e-10 / unit in tier 1 this is unit * a / min(1, amin, xmin) <= 1e-10 |f|
//   2: precision loss detected, but the absolute round-off bound on the WEIGHT w = f/p is below w_abs_tol: the
//      Monte Carlo sums need absolute, not relative, accuracy of w (PAPER.md:91 controls the round-off error of the result)
//   1: handed to the next tier
#define MQ_UNIT_F64 (32.0 * 0x1p-53)
#define MQ_UNIT_DD (64.0 * 0x1p-103)
__device__ __forceinline__ int tier_decision(bool hard, double f, double a, double amin, double xmin, double p, double cond_max, double inner_min, double unit, double w_abs_tol) {
  if (hard || !isfinite(f) || !isfinite(a)) return 1;
  // relative: the error model is unit * a / min(1, xmin, amin) (every operand of a slot is divided by g_t and the pivots, the scalar
  // factors of insertion pieces are the A_t), so the divisor belongs INSIDE the bound; inner_min stays as a floor on it
  const double inner = fmin(amin, xmin);
  if (a <= cond_max * fabs(f) * fmin(1.0, inner) && inner >= inner_min) return 0;
  if (unit * a <= w_abs_tol * p * fmin(1.0, xmin)) return 2;
  return 1;
}

// Thread roles (mcqed_kernels.cuh "lane split" / "warp split"): WLX lanes of a warp share one sample point (WLX = MQ_WL in
// the binary64 and double-double kernels, 1 in quad-double) and W warps share one group of 32 / WLX points, so a CTA of
// `threads` threads holds P = threads / (W * WLX) points; warp w works for point group w / W in role gw = w % W, lane l
// for point l % (32 / WLX) of the group in role sub = l / (32 / WLX) (a quarter warp reads consecutive points: no
// shared-memory bank conflicts). Dynamic shared memory of every evaluating kernel:
//   [ S: scal_len x P x elem | xT: (W-1) x NGRADE x P x elem | xA: (W-1) x NGRADE x P x 8 | pad to 128 | 2 stream chunks | 2 mbarriers | slack ]
__host__ __device__ inline size_t smem_head_bytes(int scal_len, int threads, size_t elem, int W, int WLX) {
  const size_t P = (size_t)threads / (W * WLX);
  size_t s = (size_t)scal_len * P * elem + (size_t)(W - 1) * MQ_NGRADE * P * (elem + 8);
  return (s + 127) & ~(size_t)127;
}
__host__ __device__ inline size_t smem_bytes(int scal_len, int threads, size_t elem, int W, int WLX) {
  return smem_head_bytes(scal_len, threads, elem, W, WLX) + 2 * MQ_CHUNK_WORDS * 8 + 16 + 64;   // + slack: the header prefetch may read 8*MQ_WL + 24 bytes past a chunk
}
template <class T, int W, int WLX> struct Roles {
  int gw, sub, slot, P;     // role of this warp in its group, role of this lane for its point, point slot of this lane in the CTA, points per CTA
  unsigned char *S; T *xT; typename MagOf<T>::type *xA;   // S: this lane's slot base of the scalar scratch (SAcc<T>, mcqed_kernels.cuh)
  __device__ __forceinline__ Roles(unsigned char *smem, int scal_len) {
    constexpr int PPW = 32 / WLX;
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    gw = w % W; sub = l / PPW; P = blockDim.x / (W * WLX); slot = (w / W) * PPW + l % PPW;
    S = smem + (size_t)slot * SAcc<T>::slot_bytes;
    xT = reinterpret_cast<T *>(smem) + (size_t)scal_len * P + slot;
    xA = reinterpret_cast<typename MagOf<T>::type *>(smem + ((size_t)scal_len * P + (size_t)(W - 1) * MQ_NGRADE * P) * sizeof(T)) + slot;
  }
};
template <int W, int WLX> __device__ __forceinline__ void setup_reader(StreamReader &rd, unsigned char *smem, int scal_len, size_t elem) {
  const size_t s = smem_head_bytes(scal_len, blockDim.x, elem, W, WLX);
  rd.init(reinterpret_cast<uint64_t *>(smem + s), reinterpret_cast<uint64_t *>(smem + s + 2 * MQ_CHUNK_WORDS * 8));
#if MQ_DEVICE_ASSERTS
  rd.dbg_scal_len = scal_len;
#endif
}


}  // namespace mqk
