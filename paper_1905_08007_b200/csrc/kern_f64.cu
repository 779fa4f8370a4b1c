// kern_f64.cu — binary64 kernels of the hot path (a1-a7) and their launchers. sm_100a.
// Product code (libmcqed.so); shares nothing with oracle/.
#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>
#include <type_traits>

#include "kern_common.cuh"

namespace mqk {

// value type of the binary64 tier: pt2 = two sample points per lane (pt2_arith.cuh), double = one
using FT = std::conditional<NP_F64 == 4, pt4, std::conditional<NP_F64 == 2, pt2, double>::type>::type;
using FM = MagOf<FT>::type;
constexpr int NP = PtsOf<FT>::n;
// DISTK: the MQ_WL lanes of a point group carry NP = MQ_WL points; lane role k draws point k, computes its scalars and assembles
// its nodes and terms in plain binary64, and FINALISES it (precision decision, weight, sums): outside the family evaluation the
// kernel is "one point per lane" with no redundant work across the lane roles. Otherwise lane role 0 (the owner) finalises
// all NP points of its group.
constexpr bool DISTK = NP > 1 && NP == MQ_WL;
constexpr int NF = DISTK ? 1 : NP;                     // points finalised by one lane

// the points this lane finalises after the evaluation: sample index (relative), density, hard flag, value, magnitude, amin, xmin
struct LanePts {
  uint64_t idx[NF]; double p[NF], f[NF], a[NF], amin[NF], xmin[NF]; bool bad[NF], live[NF];
};
// draws the lane's point(s) (a1-a3) and runs the evaluator (a4-a6). CTA-collective.
template <bool WANT_ORDER, int W, class RO>
__device__ __forceinline__ void eval_group(const DiagView &v, StreamReader &rd, const RO &ro, uint64_t first, uint64_t i0, uint64_t n, uint64_t seed,
                                           const double *z_in, double *zl, int32_t *ord, FM *z, LanePts &lp) {
  const int M = v.h->M;
  if constexpr (DISTK) {
    const uint64_t im = i0 + (uint64_t)ro.sub, ic = im < n ? im : n - 1;          // surplus slots redo the last point
    if (z_in) { for (int j = 0; j < MQ_MAXM; j++) zl[j] = j < M ? z_in[ic * M + j] : 0.0; lp.p[0] = 1.0; lp.bad[0] = false; }
    else { lp.p[0] = draw_point<WANT_ORDER>(v, first + ic, seed, zl, ord); lp.bad[0] = bad_point(zl, M, lp.p[0]); }
    lp.idx[0] = im; lp.live[0] = im < n;
  } else {
    if (z_in) {
      for (int k = 0; k < NP; k++) { const uint64_t i = i0 + k < n ? i0 + k : n - 1; for (int j = 0; j < MQ_MAXM; j++) mq_setc(z[j], k, j < M ? z_in[i * M + j] : 0.0); lp.p[k] = 1.0; }
    } else draw_points<FT, WANT_ORDER>(v, first, i0, n, seed, z, lp.p, ord);
#pragma unroll
    for (int k = 0; k < NP; k++) { lp.idx[k] = i0 + k; lp.live[k] = i0 + k < n && ro.sub == 0; lp.bad[k] = z_in ? false : bad_point(z, k, M, lp.p[k]); }
  }
  FT f, a; FM amin, xmin;
  eval_integrand<FT, W, true>(v, rd, z, zl, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
#pragma unroll
  for (int k = 0; k < NF; k++) { lp.f[k] = mq_comp(f, k); lp.a[k] = mq_comp(a, k); lp.amin[k] = mq_comp(amin, k); lp.xmin[k] = mq_comp(xmin, k); }
}

// a1-a7 in binary64. Flagged points are appended to flag_list (sample index) and not accumulated here.
__global__ void __launch_bounds__(TPB_F64, MQ_MINB_F64) k_integrate_f64(const uint64_t *__restrict__ blob, uint64_t first, uint64_t n, uint64_t seed,
                                                           MqPrec pr, double *partial,
                                                           unsigned long long *flag_list, unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const Roles<FT, W_F64, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_F64, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(FT));
  KahanPair s1{0.0, 0.0}, s2{0.0, 0.0};
  // the evaluator is CTA-collective (it stages the table stream through shared memory): every thread of the CTA runs the same
  // number of iterations; slots past the end re-evaluate the last point and discard it
  const uint64_t per = (uint64_t)ro.P * NP;
  for (uint64_t base = (uint64_t)blockIdx.x * per; base < n; base += (uint64_t)gridDim.x * per) {
    const uint64_t i0 = base + (uint64_t)ro.slot * NP;
    FM z[DISTK ? 1 : MQ_MAXM]; double zl[DISTK ? MQ_MAXM : 1]; LanePts lp;
    eval_group<false, W_F64>(v, rd, ro, first, i0, n, seed, nullptr, zl, nullptr, z, lp);
#pragma unroll
    for (int k = 0; k < NF; k++) {
      if (!lp.live[k]) continue;
      const bool flag = tier_decision(lp.bad[k], lp.f[k], lp.a[k], lp.amin[k], lp.xmin[k], lp.p[k], pr.cond_max, pr.amin_min, MQ_UNIT_F64, pr.w_abs_tol) == 1;
      if (flag) { unsigned long long slot = atomicAdd(&counters[0], 1ull); MQ_DASSERT(slot < n); flag_list[slot] = first + lp.idx[k]; }
      else { const double w = lp.f[k] / lp.p[k]; s1.add(w); s2.add(w * w); }
    }
  }
  block_reduce_store(s1, s2, partial);
}

// deterministic final reduction of the per-block partials of both passes; out += result
__global__ void k_finish(const double *partial, int nb1, int nb2, int nb3, unsigned long long *counters,
                         double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  KahanPair a{0.0, 0.0}, b{0.0, 0.0};
  for (int i = 0; i < nb1; i++) { a.merge(partial[i * 4], partial[i * 4 + 1]); b.merge(partial[i * 4 + 2], partial[i * 4 + 3]); }
  const double *p2 = partial + (size_t)MAXGRID * 4;
  for (int i = 0; i < nb2; i++) { a.merge(p2[i * 4], p2[i * 4 + 1]); b.merge(p2[i * 4 + 2], p2[i * 4 + 3]); }
  const double *p3 = partial + (size_t)2 * MAXGRID * 4;
  for (int i = 0; i < nb3; i++) { a.merge(p3[i * 4], p3[i * 4 + 1]); b.merge(p3[i * 4 + 2], p3[i * 4 + 3]); }
  if (out_sum) *out_sum += a.hi + a.lo;
  if (out_sumsq) *out_sumsq += b.hi + b.lo;
  if (out_nflag) *out_nflag += counters[0];
  if (out_ndrop) *out_ndrop += counters[1];
  counters[0] = 0; counters[1] = 0; counters[2] = 0;
}
__global__ void k_reset_counters(unsigned long long *counters) { counters[0] = 0; counters[1] = 0; counters[2] = 0; }

// parity hook: per-point outputs (binary64 pass); flagged points are listed for the dd pass
__global__ void __launch_bounds__(TPB_EVAL) k_eval_points(const uint64_t *__restrict__ blob, uint64_t first, uint64_t n, uint64_t seed,
                                                          MqPrec pr,
                                                          double *z_out, int32_t *order_out, double *p_out, double *f_out, double *f64_out,
                                                          double *cond_out, uint8_t *flag_out, unsigned long long *flag_list, unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const Roles<FT, W_F64, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  const int M = v.h->M;
  StreamReader rd; setup_reader<W_F64, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(FT));
  const uint64_t per = (uint64_t)ro.P * NP;
  for (uint64_t base = (uint64_t)blockIdx.x * per; base < n; base += (uint64_t)gridDim.x * per) {
    const uint64_t i0 = base + (uint64_t)ro.slot * NP;
    FM z[DISTK ? 1 : MQ_MAXM]; double zl[DISTK ? MQ_MAXM : 1]; int32_t ord[NF * MQ_MAXM]; LanePts lp;
    eval_group<true, W_F64>(v, rd, ro, first, i0, n, seed, nullptr, zl, ord, z, lp);
    for (int k = 0; k < NF; k++) {
      if (!lp.live[k]) continue;
      const uint64_t i = lp.idx[k];
      const int dec = tier_decision(lp.bad[k], lp.f[k], lp.a[k], lp.amin[k], lp.xmin[k], lp.p[k], pr.cond_max, pr.amin_min, MQ_UNIT_F64, pr.w_abs_tol);
      const bool flag = dec == 1;
      if (z_out) for (int j = 0; j < M; j++) z_out[i * M + j] = DISTK ? zl[j] : mq_comp(z[DISTK ? 0 : j], k);
      if (order_out) for (int j = 0; j < M; j++) order_out[i * M + j] = ord[k * MQ_MAXM + j];
      if (p_out) p_out[i] = lp.p[k];
      if (f_out) f_out[i] = lp.f[k];
      if (f64_out) f64_out[i] = lp.f[k];
      if (cond_out) cond_out[i] = lp.a[k] / fabs(lp.f[k]);
      if (flag_out) flag_out[i] = (uint8_t)dec;      // 0 accepted (relative), 1 re-evaluated in double-double, 2 accepted by the absolute bound on w
      if (flag && flag_list) { unsigned long long slot = atomicAdd(&counters[0], 1ull); flag_list[slot] = i; }
    }
  }
}

__global__ void __launch_bounds__(TPB_EVAL) k_eval_z_f64(const uint64_t *__restrict__ blob, uint64_t n, const double *__restrict__ z_in,
                                                         double *f64_out, double *cond_out, double *aux_out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const Roles<FT, W_F64, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_F64, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(FT));
  const uint64_t per = (uint64_t)ro.P * NP;
  for (uint64_t base = (uint64_t)blockIdx.x * per; base < n; base += (uint64_t)gridDim.x * per) {
    const uint64_t i0 = base + (uint64_t)ro.slot * NP;
    FM z[DISTK ? 1 : MQ_MAXM]; double zl[DISTK ? MQ_MAXM : 1]; LanePts lp;
    eval_group<false, W_F64>(v, rd, ro, 0, i0, n, 0, z_in, zl, nullptr, z, lp);
    for (int k = 0; k < NF; k++) {
      if (!lp.live[k]) continue;
      const uint64_t i = lp.idx[k];
      if (f64_out) f64_out[i] = lp.f[k];
      if (cond_out) cond_out[i] = lp.a[k] / fabs(lp.f[k]);
      if (aux_out) { aux_out[2 * i] = lp.amin[k]; aux_out[2 * i + 1] = lp.xmin[k]; }
    }
  }
}

// ------------------------------------------------------------------ batched path, binary64 tier (a1-a7 for every diagram of a batch)
// Persistent CTAs; item = PTS_F64 consecutive sample indices of one diagram, taken from queue[0].
// Flagged points are compacted inside the item in thread order (ballot + prefix): deterministic lists.
__global__ void __launch_bounds__(TPB_F64, MQ_MINB_F64) k_batch_f64(BatchView bv, uint64_t first_u, uint64_t n_u, uint64_t seed, int scal_len, int no_dd) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ unsigned s_item, s_wcnt[TPB_F64 / 32];
  const Roles<FT, 1, MQ_WL> ro(smem_raw, scal_len);
  StreamReader rd; setup_reader<1, MQ_WL>(rd, smem_raw, scal_len, sizeof(FT));
  const uint32_t total = bv.f64_start ? bv.f64_start[bv.nd] : (uint32_t)bv.nd * bv.ipd;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) s_item = (unsigned)atomicAdd(&bv.queue[0], 1ull);
    __syncthreads();
    const uint32_t item = s_item;
    if (item >= total) break;
    const int d = bv.f64_start ? batch_find(bv.f64_start, bv.nd, item) : (int)(item / bv.ipd);
    const uint32_t b = bv.f64_start ? item - bv.f64_start[d] : item % bv.ipd;
    const uint64_t first = batch_first(bv, d, first_u), n = batch_n(bv, d, n_u);
    MQ_DASSERT(d >= 0 && d < bv.nd && (uint64_t)(b + 1) * PTS_F64 <= (uint64_t)bv.cap);       // the item's slice of the per-diagram lists
    const DiagView v = make_view(bv.dg[d].blob);
    MQ_DASSERT(v.h->max_scal_len <= scal_len && v.h->wl == MQ_WL);
    MqPrec pr = bv.dg[d].pr;
    if (no_dd) { pr.cond_max = 1e300; pr.amin_min = -1.0; }
    const uint64_t i0 = (uint64_t)b * PTS_F64 + (uint64_t)ro.slot * NP;
    FM z[DISTK ? 1 : MQ_MAXM]; double zl[DISTK ? MQ_MAXM : 1]; LanePts lp;
    eval_group<false, 1>(v, rd, ro, first, i0, n, seed, nullptr, zl, nullptr, z, lp);
    // flagged points of the item, compacted in (warp, lane, point) order: a deterministic list
    bool flag[NF]; unsigned bal[NF]; unsigned mine = 0, wsum = 0;
#pragma unroll
    for (int k = 0; k < NF; k++) {
      flag[k] = lp.live[k] && tier_decision(lp.bad[k], lp.f[k], lp.a[k], lp.amin[k], lp.xmin[k], lp.p[k], pr.cond_max, pr.amin_min, MQ_UNIT_F64, pr.w_abs_tol) == 1;
      bal[k] = __ballot_sync(0xffffffffu, flag[k]);
      mine += __popc(bal[k] & ((1u << lane) - 1u)); wsum += __popc(bal[k]);
    }
    if (lane == 0) s_wcnt[warp] = wsum;
    __syncthreads();
    unsigned before = 0, all = 0;
#pragma unroll
    for (int w = 0; w < TPB_F64 / 32; w++) { if (w < warp) before += s_wcnt[w]; all += s_wcnt[w]; }
    KahanPair s1{0.0, 0.0}, s2{0.0, 0.0};
    unsigned pos = before + mine;
#pragma unroll
    for (int k = 0; k < NF; k++) {
      if (flag[k]) { MQ_DASSERT(pos < (unsigned)PTS_F64); bv.flag_raw[(size_t)d * bv.cap + (size_t)b * PTS_F64 + pos++] = (uint32_t)lp.idx[k]; }
      else if (lp.live[k]) { const double w = lp.f[k] / lp.p[k]; s1.add(w); s2.add(w * w); }
    }
    if (threadIdx.x == 0) bv.item_cnt[(size_t)d * (bv.cap / PTS_F64) + b] = all;
    block_reduce_to(s1, s2, bv.part_f64 + (size_t)item * 4);
  }
}

// one CTA per diagram: concatenates the item-local flagged lists in item order (ascending sample index)
__global__ void __launch_bounds__(128) k_batch_compact(BatchView bv) {
  __shared__ unsigned sc[128];
  __shared__ unsigned s_base;
  const int d = blockIdx.x, t = threadIdx.x;
  const uint32_t *cnt = bv.item_cnt + (size_t)d * (bv.cap / PTS_F64);
  const uint32_t *raw = bv.flag_raw + (size_t)d * bv.cap;
  uint32_t *out = bv.flag_list + (size_t)d * bv.cap;
  if (t == 0) s_base = 0;
  __syncthreads();
  const uint32_t ipd = bv.f64_start ? bv.f64_start[d + 1] - bv.f64_start[d] : bv.ipd;
  for (uint32_t b0 = 0; b0 < ipd; b0 += 128) {
    const uint32_t b = b0 + t;
    const unsigned c = b < ipd ? cnt[b] : 0u;
    sc[t] = c;
    __syncthreads();
    for (int off = 1; off < 128; off <<= 1) {        // inclusive scan
      const unsigned x = t >= off ? sc[t - off] : 0u;
      __syncthreads();
      sc[t] += x;
      __syncthreads();
    }
    const unsigned o = s_base + sc[t] - c;
    MQ_DASSERT(c <= (unsigned)PTS_F64 && (size_t)o + c <= (size_t)bv.cap);
    for (unsigned k = 0; k < c; k++) out[o + k] = raw[(size_t)b * PTS_F64 + k];
    __syncthreads();
    if (t == 127) s_base += sc[127];
    __syncthreads();
  }
  if (t == 0) bv.nflag[d] = s_base;
}
// item ranges of the next tier: start[d] = sum_{d'<d} ceil(count[d'] / per); resets that tier's queue head
__global__ void k_batch_ranges(const unsigned long long *count, unsigned long long limit, int nd, unsigned per, uint32_t *start, unsigned long long *queue_head) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  uint32_t acc = 0;
  for (int d = 0; d < nd; d++) { start[d] = acc; const unsigned long long c = count[d] < limit ? count[d] : limit; acc += (uint32_t)((c + per - 1) / per); }
  start[nd] = acc;
  *queue_head = 0ull;
}
// one thread per diagram: adds the per-item partial sums of the three tiers in item order; out += result
__global__ void k_batch_finish(BatchView bv, int tiers, double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop) {
  const int d = blockIdx.x * blockDim.x + threadIdx.x;
  if (d == 0) bv.queue[0] = 0ull;
  if (d >= bv.nd) return;
  KahanPair a{0.0, 0.0}, b{0.0, 0.0};
  const uint32_t ipd = bv.f64_start ? bv.f64_start[d + 1] - bv.f64_start[d] : bv.ipd;
  const double *p = bv.part_f64 + (size_t)(bv.f64_start ? bv.f64_start[d] : d * bv.ipd) * 4;
  for (uint32_t i = 0; i < ipd; i++) { a.merge(p[i * 4], p[i * 4 + 1]); b.merge(p[i * 4 + 2], p[i * 4 + 3]); }
  unsigned long long ndrop = bv.ndrop[d];
  if (tiers > 1)
    for (uint32_t i = bv.dd_start[d]; i < bv.dd_start[d + 1]; i++) { const double *q = bv.part_dd + (size_t)i * 4; a.merge(q[0], q[1]); b.merge(q[2], q[3]); }
  if (tiers > 2)
    for (uint32_t i = bv.qd_start[d]; i < bv.qd_start[d + 1]; i++) { const double *q = bv.part_qd + (size_t)i * 4; a.merge(q[0], q[1]); b.merge(q[2], q[3]); }
  else if (tiers == 2) ndrop += bv.nlost[d] < bv.lostcap ? bv.nlost[d] : bv.lostcap;   // quad-double pass skipped: its points count as dropped
  if (out_sum) out_sum[d] += a.hi + a.lo;
  if (out_sumsq) out_sumsq[d] += b.hi + b.lo;
  if (out_nflag) out_nflag[d] += bv.nflag[d];
  if (out_ndrop) out_ndrop[d] += ndrop;
  bv.nflag[d] = 0; bv.nlost[d] = 0; bv.ndrop[d] = 0;
}

// FP64 FMA peak: 8 independent chains per thread
__global__ void k_fp64_peak(int iters, double *sink) {
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3, a4 = a0 + 4e-3, a5 = a0 + 5e-3, a6 = a0 + 6e-3, a7 = a0 + 7e-3;
  const double m = 0.999999999, c = 1e-9;
  for (int i = 0; i < iters; i++) {
#pragma unroll
    for (int k = 0; k < 16; k++) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  if (a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7 == 12345.678) sink[0] = a0;
}

}  // namespace mqk

using namespace mqk;

int mq_config_f64(mc_diagram *d) {
  d->smem_f64 = smem_bytes(d->max_scal_len, TPB_F64, sizeof(FT), W_F64, MQ_WL);
  d->smem_eval = smem_bytes(d->max_scal_len, TPB_EVAL, sizeof(FT), W_F64, MQ_WL);
  cudaError_t e;
  if ((e = allow_max_smem(k_integrate_f64)) != cudaSuccess) return (int)e;
  if ((e = allow_max_smem(k_eval_points)) != cudaSuccess) return (int)e;
  if ((e = allow_max_smem(k_eval_z_f64)) != cudaSuccess) return (int)e;
  int nsm = 0, occ = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_integrate_f64, TPB_F64, d->smem_f64)) != cudaSuccess) return (int)e;
  if (occ < 1) return (int)cudaErrorLaunchOutOfResources;
  d->grid_f64 = std::min(MAXGRID, nsm * occ);
  return 0;
}
void mq_launch_integrate_f64(const mc_diagram *d, int grid, uint64_t first, uint64_t n, uint64_t seed, MqPrec pr, mq_stream st) {
  k_integrate_f64<<<grid, TPB_F64, d->smem_f64, (cudaStream_t)st>>>(d->d_blob, first, n, seed, pr, d->ws.partial, d->ws.flag_list, d->ws.counters);
}
void mq_launch_finish(const mc_diagram *d, int nb1, int nb2, int nb3, double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop, mq_stream st) {
  k_finish<<<1, 32, 0, (cudaStream_t)st>>>(d->ws.partial, nb1, nb2, nb3, d->ws.counters, out_sum, out_sumsq, out_nflag, out_ndrop);
}
void mq_launch_reset(const mc_diagram *d, mq_stream st) { k_reset_counters<<<1, 1, 0, (cudaStream_t)st>>>(d->ws.counters); }
void mq_launch_eval_points(const mc_diagram *d, int grid, uint64_t first, uint64_t n, uint64_t seed, MqPrec pr,
                           double *z_out, int32_t *order_out, double *p_out, double *f_out, double *f64_out, double *cond_out,
                           uint8_t *flag_out, bool list_flagged, mq_stream st) {
  k_eval_points<<<grid, TPB_EVAL, d->smem_eval, (cudaStream_t)st>>>(d->d_blob, first, n, seed, pr, z_out, order_out, p_out, f_out, f64_out,
                                                                  cond_out, flag_out, list_flagged ? d->ws.flag_list : nullptr, d->ws.counters);
}
void mq_launch_eval_z_f64(const mc_diagram *d, int grid, uint64_t n, const double *z_in, double *f64_out, double *cond_out, double *aux_out, mq_stream st) {
  k_eval_z_f64<<<grid, TPB_EVAL, d->smem_eval, (cudaStream_t)st>>>(d->d_blob, n, z_in, f64_out, cond_out, aux_out);
}
int mq_fp64_peak(int iters, mq_stream stream, double *flops, double *ms) {
  cudaStream_t st = (cudaStream_t)stream;
  int nsm = 0, dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  double *sink = nullptr;
  cudaError_t e;
  if ((e = cudaMalloc(&sink, 8)) != cudaSuccess) return (int)e;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = nsm * 2, tpb = 1024;
  k_fp64_peak<<<blocks, tpb, 0, st>>>(iters / 8 + 1, sink);   // warm-up
  cudaEventRecord(e0, st);
  k_fp64_peak<<<blocks, tpb, 0, st>>>(iters, sink);
  cudaEventRecord(e1, st);
  e = cudaEventSynchronize(e1);
  float t = 0; cudaEventElapsedTime(&t, e0, e1);
  if (ms) *ms = t;
  if (flops) *flops = 2.0 * 8.0 * 16.0 * (double)iters * (double)blocks * tpb / (t * 1e-3);
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
  return (int)e;
}

// ---- mc_integrate_static: the binary64 tier with its scratch in a file-scope device array (no allocation at call time) ----
// Layout of g_static_scratch: [ counters: 4 x u64 | partial: MAXGRID x 4 doubles | flag_list: MC_STATIC_MAX_SAMPLES x u64 ].
// Every GPU that loads the library holds the array until the process exits; every call shares it (calls that overlap on
// one GPU race). In host code the array's NAME is only a host-side stand-in: the device address comes from
// cudaGetSymbolAddress, resolved once per device with that device current.
namespace {
constexpr size_t STATIC_OFF_PARTIAL = 256;                                                      // after the counters
constexpr size_t STATIC_OFF_FLAGS = STATIC_OFF_PARTIAL + sizeof(double) * 4 * (size_t)mqk::MAXGRID;
constexpr size_t STATIC_BYTES = STATIC_OFF_FLAGS + sizeof(unsigned long long) * (size_t)MC_STATIC_MAX_SAMPLES;
static_assert(STATIC_OFF_FLAGS % 256 == 0, "flag list stays 256-byte aligned");
constexpr int STATIC_MAXDEV = 64;
void *g_static_ptr[STATIC_MAXDEV];                  // device address of g_static_scratch per device ordinal, nullptr = not resolved yet
std::mutex g_static_mu;
}  // namespace
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_BYTES];

int mq_static_integrate_f64(const mc_diagram *d, uint64_t first, uint64_t n, uint64_t seed, mqk::MqPrec pr,
                            double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop, mq_stream stream) {
  int dev = -1;
  cudaError_t e;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return (int)e;
  if (dev < 0 || dev >= STATIC_MAXDEV) return (int)cudaErrorInvalidDevice;
  unsigned char *base;
  {
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
      void *p = nullptr;
      if ((e = cudaGetSymbolAddress(&p, g_static_scratch)) != cudaSuccess) return (int)e;
      g_static_ptr[dev] = p;
    }
    base = static_cast<unsigned char *>(g_static_ptr[dev]);
  }
  unsigned long long *counters = reinterpret_cast<unsigned long long *>(base);
  double *partial = reinterpret_cast<double *>(base + STATIC_OFF_PARTIAL);
  unsigned long long *flag_list = reinterpret_cast<unsigned long long *>(base + STATIC_OFF_FLAGS);
  cudaStream_t st = (cudaStream_t)stream;
  const int grid = (int)std::min<uint64_t>((uint64_t)d->grid_f64, (n + PTS_F64 - 1) / PTS_F64);
  k_reset_counters<<<1, 1, 0, st>>>(counters);      // the array keeps the last call's contents: the counters must start at zero
  k_integrate_f64<<<grid, TPB_F64, d->smem_f64, st>>>(d->d_blob, first, n, seed, pr, partial, flag_list, counters);
  k_finish<<<1, 32, 0, st>>>(partial, grid, 0, 0, counters, out_sum, out_sumsq, out_nflag, out_ndrop);
  return (int)cudaGetLastError();
}

// ---- batched path launchers ----
int mq_batch_config_f64(size_t smem, int *grid) {
  cudaError_t e;
  if ((e = allow_max_smem(k_batch_f64)) != cudaSuccess) return (int)e;
  int nsm = 0, occ = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_batch_f64, TPB_F64, smem)) != cudaSuccess) return (int)e;
  if (occ < 1) return (int)cudaErrorLaunchOutOfResources;
  *grid = nsm * occ;
  return 0;
}
size_t mq_batch_smem_f64(int scal_len) { return smem_bytes(scal_len, TPB_F64, sizeof(FT), 1, MQ_WL); }
void mq_launch_batch_f64(const BatchView &bv, int grid, size_t smem, uint64_t first, uint64_t n, uint64_t seed, int scal_len, int no_dd, mq_stream st) {
  k_batch_f64<<<grid, TPB_F64, smem, (cudaStream_t)st>>>(bv, first, n, seed, scal_len, no_dd);
}
void mq_launch_batch_compact(const BatchView &bv, mq_stream st) { k_batch_compact<<<bv.nd, 128, 0, (cudaStream_t)st>>>(bv); }
void mq_launch_batch_ranges(const BatchView &bv, int tier, mq_stream st) {
  if (tier == 1) k_batch_ranges<<<1, 1, 0, (cudaStream_t)st>>>(bv.nflag, ~0ull, bv.nd, (unsigned)PTS_DD, bv.dd_start, bv.queue + 1);
  else k_batch_ranges<<<1, 1, 0, (cudaStream_t)st>>>(bv.nlost, (unsigned long long)bv.lostcap, bv.nd, 1u, bv.qd_start, bv.queue + 2);   // quad-double items are single points
}
void mq_launch_batch_finish(const BatchView &bv, int tiers, double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop, mq_stream st) {
  k_batch_finish<<<(bv.nd + 127) / 128, 128, 0, (cudaStream_t)st>>>(bv, tiers, out_sum, out_sumsq, out_nflag, out_ndrop);
}
