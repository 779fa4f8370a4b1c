// kern_qd.cu — third precision tier: quad-double re-evaluation of the points whose cancellation exceeds what
// double-double resolves (O8; "arithmetic with different precisions"). sm_100a.
// Product code (libmcqed.so); shares nothing with oracle/. Speed is irrelevant here (per-mille of the points):
// the evaluator is instantiated with the loop-based family code (family_generic), 32 threads per CTA.
#include <cuda_runtime.h>

#include <algorithm>

#include "qd_arith.cuh"
#include "kern_common.cuh"

namespace mqk {

template <> __device__ __forceinline__ qd mq_shfl_xor<qd>(qd v, int m) {
  return qd(__shfl_xor_sync(0xffffffffu, v.x[0], m), __shfl_xor_sync(0xffffffffu, v.x[1], m), __shfl_xor_sync(0xffffffffu, v.x[2], m), __shfl_xor_sync(0xffffffffu, v.x[3], m));
}
template <> __device__ __forceinline__ qd lds_T<qd>(uint32_t a) {
  const double2 lo = lds_f64x2(a), hi = lds_f64x2(a + 16);
  return qd(lo.x, lo.y, hi.x, hi.y);
}

// Few points reach this tier (per-mille of the flagged ones), so the parallelism must come from inside a point: W_QD warps
// share one group of 32 points and split its families (mcqed_kernels.cuh "warp split").
constexpr int W_QD = 8, PTS_QD = 32 / MQ_WL, TPB_QD = W_QD * 32;   // per CTA: one group of 32 / MQ_WL points, MQ_WL lanes per point, W_QD warps

// points listed in lost_list (sample indices) by the double-double pass
__global__ void __launch_bounds__(TPB_QD) k_integrate_qd(const uint64_t *__restrict__ blob, uint64_t seed, double *partial,
                                                         const unsigned long long *lost_list, unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const Roles<qd, W_QD, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_QD, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(qd));
  const unsigned long long cnt = counters[2] < LOSTCAP ? counters[2] : LOSTCAP;
  KahanPair s1{0.0, 0.0}, s2{0.0, 0.0};
  for (unsigned long long base = (unsigned long long)blockIdx.x * ro.P; base < cnt; base += (unsigned long long)gridDim.x * ro.P) {
    const unsigned long long i = base + ro.slot; const bool live = i < cnt && ro.gw == 0 && ro.sub == 0;
    double z[MQ_MAXM]; double p = 1.0;
    if (ro.gw == 0) p = draw_point<false>(v, lost_list[i < cnt ? i : cnt - 1], seed, z, nullptr);
    qd f, a; double amin, xmin;
    eval_integrand<qd, W_QD, true>(v, rd, z, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    if (!live) continue;
    const double fd = mq_to_double(f);
    if (bad_point(z, v.h->M, p) || !isfinite(fd)) atomicAdd(&counters[1], 1ull);     // dropped: w = 0
    else { const double w = fd / p; s1.add(w); s2.add(w * w); }
  }
  block_reduce_store(s1, s2, partial);
}

// batched path, quad-double tier: persistent CTAs; item = 32 entries of one diagram's lost list
__global__ void __launch_bounds__(TPB_QD) k_batch_qd(BatchView bv, uint64_t first, uint64_t seed, int scal_len) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ unsigned s_item; __shared__ int s_d;
  const Roles<qd, W_QD, MQ_WL> ro(smem_raw, scal_len);
  StreamReader rd; setup_reader<W_QD, MQ_WL>(rd, smem_raw, scal_len, sizeof(qd));
  const uint32_t total = bv.qd_start[bv.nd];
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) { s_item = (unsigned)atomicAdd(&bv.queue[2], 1ull); s_d = s_item < total ? batch_find(bv.qd_start, bv.nd, s_item) : 0; }
    __syncthreads();
    const uint32_t item = s_item;
    if (item >= total) break;
    const int d = s_d;
    const DiagView v = make_view(bv.dg[d].blob);
    const unsigned long long cnt = bv.nlost[d] < bv.lostcap ? bv.nlost[d] : bv.lostcap;
    const unsigned long long i = (unsigned long long)(item - bv.qd_start[d]) * PTS_QD + ro.slot; const bool live = i < cnt && ro.gw == 0 && ro.sub == 0;
    const uint32_t rel = bv.lost_list[(size_t)d * bv.lostcap + (i < cnt ? i : cnt - 1)];
    double z[MQ_MAXM]; double p = 1.0;
    if (ro.gw == 0) p = draw_point<false>(v, first + rel, seed, z, nullptr);
    qd f, a; double amin, xmin;
    eval_integrand<qd, W_QD, true>(v, rd, z, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    KahanPair s1{0.0, 0.0}, s2{0.0, 0.0};
    if (live) {
      const double fd = mq_to_double(f);
      if (bad_point(z, v.h->M, p) || !isfinite(fd)) atomicAdd(&bv.ndrop[d], 1ull);
      else { const double w = fd / p; s1.add(w); s2.add(w * w); }
    }
    block_reduce_to(s1, s2, bv.part_qd + (size_t)item * 4);
  }
}

// parity hooks: per-point values of the lost points (relative indices), and the integrand at given z
__global__ void __launch_bounds__(TPB_QD) k_eval_points_qd(const uint64_t *__restrict__ blob, uint64_t first, uint64_t seed, double *f_out,
                                                           const unsigned long long *lost_list, const unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const Roles<qd, W_QD, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_QD, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(qd));
  const unsigned long long cnt = counters[2] < LOSTCAP ? counters[2] : LOSTCAP;
  for (unsigned long long base = (unsigned long long)blockIdx.x * ro.P; base < cnt; base += (unsigned long long)gridDim.x * ro.P) {
    const unsigned long long i = base + ro.slot; const bool live = i < cnt && ro.gw == 0 && ro.sub == 0;
    double z[MQ_MAXM];
    const unsigned long long rel = lost_list[i < cnt ? i : cnt - 1];
    if (ro.gw == 0) draw_point<false>(v, first + rel, seed, z, nullptr);
    qd f, a; double amin, xmin;
    eval_integrand<qd, W_QD, true>(v, rd, z, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    if (live) f_out[rel] = mq_to_double(f);
  }
}
__global__ void __launch_bounds__(TPB_QD) k_eval_z_qd(const uint64_t *__restrict__ blob, uint64_t n, const double *__restrict__ z_in, double *fqd_out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const int M = v.h->M;
  const Roles<qd, W_QD, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_QD, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(qd));
  for (uint64_t base = (uint64_t)blockIdx.x * ro.P; base < n; base += (uint64_t)gridDim.x * ro.P) {
    const bool live = base + ro.slot < n && ro.gw == 0 && ro.sub == 0;
    const uint64_t i = base + ro.slot < n ? base + ro.slot : n - 1;
    double z[MQ_MAXM];
    for (int k = 0; k < MQ_MAXM; k++) z[k] = k < M ? z_in[i * M + k] : 0.0;
    qd f, a; double amin, xmin;
    eval_integrand<qd, W_QD, true>(v, rd, z, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    if (live) fqd_out[i] = mq_to_double(f);
  }
}

}  // namespace mqk

using namespace mqk;

int mq_config_qd(mc_diagram *d) {
  d->smem_qd = smem_bytes(d->max_scal_len, TPB_QD, sizeof(qd), W_QD, MQ_WL);
  cudaError_t e;
  if ((e = allow_max_smem(k_integrate_qd)) != cudaSuccess) return (int)e;
  if ((e = allow_max_smem(k_eval_points_qd)) != cudaSuccess) return (int)e;
  if ((e = allow_max_smem(k_eval_z_qd)) != cudaSuccess) return (int)e;
  int nsm = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  int occ = 1;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_integrate_qd, TPB_QD, d->smem_qd)) != cudaSuccess) return (int)e;
  if (occ < 1) return (int)cudaErrorLaunchOutOfResources;
  d->grid_qd = nsm * occ;
  return 0;
}
void mq_launch_integrate_qd(const mc_diagram *d, uint64_t seed, mq_stream st) {
  k_integrate_qd<<<d->grid_qd, TPB_QD, d->smem_qd, (cudaStream_t)st>>>(d->d_blob, seed, d->ws.partial + (size_t)2 * MAXGRID * 4, d->ws.lost_list, d->ws.counters);
}
void mq_launch_eval_points_qd(const mc_diagram *d, uint64_t first, uint64_t seed, double *f_out, mq_stream st) {
  k_eval_points_qd<<<d->grid_qd, TPB_QD, d->smem_qd, (cudaStream_t)st>>>(d->d_blob, first, seed, f_out, d->ws.lost_list, d->ws.counters);
}
void mq_launch_eval_z_qd(const mc_diagram *d, uint64_t n, const double *z_in, double *fqd_out, mq_stream st) {
  const int g = (int)std::min<uint64_t>((uint64_t)MAXGRID, (n + PTS_QD - 1) / PTS_QD);
  k_eval_z_qd<<<g, TPB_QD, d->smem_qd, (cudaStream_t)st>>>(d->d_blob, n, z_in, fqd_out);
}

// ---- batched path launchers ----
int mq_batch_config_qd(size_t smem, int *grid) {
  cudaError_t e;
  if ((e = allow_max_smem(k_batch_qd)) != cudaSuccess) return (int)e;
  int nsm = 0, occ = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_batch_qd, TPB_QD, smem)) != cudaSuccess) return (int)e;
  if (occ < 1) return (int)cudaErrorLaunchOutOfResources;
  *grid = nsm * occ;
  return 0;
}
size_t mq_batch_smem_qd(int scal_len) { return smem_bytes(scal_len, TPB_QD, sizeof(qd), W_QD, MQ_WL); }
void mq_launch_batch_qd(const BatchView &bv, int grid, size_t smem, uint64_t first, uint64_t seed, int scal_len, mq_stream st) {
  k_batch_qd<<<grid, TPB_QD, smem, (cudaStream_t)st>>>(bv, first, seed, scal_len);
}
