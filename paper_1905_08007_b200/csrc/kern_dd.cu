// kern_dd.cu — double-double kernels: the precision fallback (a8) and their launchers. sm_100a.
// Product code (libmcqed.so); shares nothing with oracle/.
#include <cuda_runtime.h>

#include <algorithm>

#include "kern_common.cuh"

namespace mqk {

// beyond double-double (O8): pair arithmetic carries ~2^-103 relative to the operands, so a point whose
// condition number (or pivot / current loss) exceeds dd_cond_max (default 1e26: ~5 digits left) goes on to quad-double,
// unless the absolute round-off bound on its weight is already below w_abs_tol (tier_decision, kern_common.cuh)

// register budget of the double-double kernels: left to ptxas by default (it settles at 168 registers = 3 CTAs of 128 threads per SM);
// MCQED_DEFS=-DMQ_MINB_DD=n forces n resident CTAs per SM (tuning builds)
#ifdef MQ_MINB_DD
#define MQ_DD_BOUNDS __launch_bounds__(TPB_DD, MQ_MINB_DD)
#else
#define MQ_DD_BOUNDS __launch_bounds__(TPB_DD)
#endif

// a8: double-double re-evaluation of the flagged points (dense lanes: one list entry per thread)
__global__ void MQ_DD_BOUNDS k_integrate_dd(const uint64_t *__restrict__ blob, uint64_t seed, MqPrec pr, double *partial,
                                                         const unsigned long long *flag_list, unsigned long long *lost_list, unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const Roles<dd, W_DD, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_DD, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(dd));
  const unsigned long long cnt = counters[0];
  KahanPair s1{0.0, 0.0}, s2{0.0, 0.0};
  for (unsigned long long base = (unsigned long long)blockIdx.x * ro.P; base < cnt; base += (unsigned long long)gridDim.x * ro.P) {
    const unsigned long long i = base + ro.slot; const bool live = i < cnt && ro.gw == 0 && ro.sub == 0;
    double z[MQ_MAXM]; double p = 1.0;
    if (ro.gw == 0) p = draw_point<false>(v, flag_list[i < cnt ? i : cnt - 1], seed, z, nullptr);
    dd f, a; double amin, xmin;
    eval_integrand<dd, W_DD, true>(v, rd, z, nullptr, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    if (!live) continue;
    const double fd = mq_to_double(f);
    const bool lost = tier_decision(false, fd, mq_to_double(a), amin, xmin, p, pr.dd_cond_max, 1.0 / pr.dd_cond_max, MQ_UNIT_DD, pr.w_abs_tol) == 1;
    if (bad_point(z, v.h->M, p)) atomicAdd(&counters[1], 1ull);                  // dropped: w = 0
    else if (lost) {                                          // third tier: quad-double
      const unsigned long long slot = atomicAdd(&counters[2], 1ull);
      if (slot < LOSTCAP) lost_list[slot] = flag_list[i]; else { atomicAdd(&counters[1], 1ull); }
    }
    else { const double w = fd / p; s1.add(w); s2.add(w * w); }
  }
  block_reduce_store(s1, s2, partial);
}

// batched path, double-double tier: persistent CTAs; item = PTS_DD consecutive entries of one diagram's flagged list
__global__ void MQ_DD_BOUNDS k_batch_dd(BatchView bv, uint64_t first, uint64_t seed, int scal_len) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ unsigned s_item; __shared__ int s_d;
  const Roles<dd, W_DD, MQ_WL> ro(smem_raw, scal_len);
  StreamReader rd; setup_reader<W_DD, MQ_WL>(rd, smem_raw, scal_len, sizeof(dd));
  const uint32_t total = bv.dd_start[bv.nd];
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) { s_item = (unsigned)atomicAdd(&bv.queue[1], 1ull); s_d = s_item < total ? batch_find(bv.dd_start, bv.nd, s_item) : 0; }
    __syncthreads();
    const uint32_t item = s_item;
    if (item >= total) break;
    const int d = s_d;
    const DiagView v = make_view(bv.dg[d].blob);
    const MqPrec pr = bv.dg[d].pr;
    const unsigned long long cnt = bv.nflag[d];
    const unsigned long long i = (unsigned long long)(item - bv.dd_start[d]) * PTS_DD + ro.slot; const bool live = i < cnt && ro.sub == 0 && ro.gw == 0;
    const uint32_t rel = bv.flag_list[(size_t)d * bv.cap + (i < cnt ? i : cnt - 1)];
    double z[MQ_MAXM];
    const double p = draw_point<false>(v, batch_first(bv, d, first) + rel, seed, z, nullptr);
    dd f, a; double amin, xmin;
    eval_integrand<dd, W_DD, true>(v, rd, z, nullptr, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    KahanPair s1{0.0, 0.0}, s2{0.0, 0.0};
    if (live) {
      const double fd = mq_to_double(f);
      const bool lost = tier_decision(false, fd, mq_to_double(a), amin, xmin, p, pr.dd_cond_max, 1.0 / pr.dd_cond_max, MQ_UNIT_DD, pr.w_abs_tol) == 1;     // same rule as k_integrate_dd
      if (bad_point(z, v.h->M, p)) atomicAdd(&bv.ndrop[d], 1ull);
      else if (lost) {
        const unsigned long long slot = atomicAdd(&bv.nlost[d], 1ull);
        if (slot < bv.lostcap) bv.lost_list[(size_t)d * bv.lostcap + slot] = rel; else atomicAdd(&bv.ndrop[d], 1ull);
      }
      else { const double w = fd / p; s1.add(w); s2.add(w * w); }
    }
    block_reduce_to(s1, s2, bv.part_dd + (size_t)item * 4);
  }
}

__global__ void MQ_DD_BOUNDS k_eval_points_dd(const uint64_t *__restrict__ blob, uint64_t first, uint64_t seed, MqPrec pr, double *f_out,
                                                           const unsigned long long *flag_list, unsigned long long *lost_list, unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const Roles<dd, W_DD, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_DD, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(dd));
  const unsigned long long cnt = counters[0];
  for (unsigned long long base = (unsigned long long)blockIdx.x * ro.P; base < cnt; base += (unsigned long long)gridDim.x * ro.P) {
    const unsigned long long i = base + ro.slot; const bool live = i < cnt && ro.gw == 0 && ro.sub == 0;
    double z[MQ_MAXM]; double p = 1.0;
    const unsigned long long rel = flag_list[i < cnt ? i : cnt - 1];
    if (ro.gw == 0) p = draw_point<false>(v, first + rel, seed, z, nullptr);
    dd f, a; double amin, xmin;
    eval_integrand<dd, W_DD, true>(v, rd, z, nullptr, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    if (live) {
      const double fd = mq_to_double(f);
      f_out[rel] = fd;
      if (tier_decision(false, fd, mq_to_double(a), amin, xmin, p, pr.dd_cond_max, 1.0 / pr.dd_cond_max, MQ_UNIT_DD, pr.w_abs_tol) == 1) {
        const unsigned long long slot = atomicAdd(&counters[2], 1ull);
        if (slot < LOSTCAP) lost_list[slot] = rel;
      }
    }
  }
}

__global__ void MQ_DD_BOUNDS k_eval_z_dd(const uint64_t *__restrict__ blob, uint64_t n, const double *__restrict__ z_in, double *fdd_out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const int M = v.h->M;
  const Roles<dd, W_DD, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<W_DD, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(dd));
  for (uint64_t base = (uint64_t)blockIdx.x * ro.P; base < n; base += (uint64_t)gridDim.x * ro.P) {
    const bool live = base + ro.slot < n && ro.gw == 0 && ro.sub == 0;
    const uint64_t i = base + ro.slot < n ? base + ro.slot : n - 1;
    double z[MQ_MAXM];
    for (int k = 0; k < MQ_MAXM; k++) z[k] = k < M ? z_in[i * M + k] : 0.0;
    dd f, a; double amin, xmin;
    eval_integrand<dd, W_DD, true>(v, rd, z, nullptr, ro.S, ro.P, ro.xT, ro.xA, ro.gw, ro.sub, f, a, amin, xmin);
    if (live) fdd_out[i] = mq_to_double(f);
  }
}

}  // namespace mqk

using namespace mqk;

int mq_config_dd(mc_diagram *d) {
  d->smem_dd = smem_bytes(d->max_scal_len, TPB_DD, sizeof(dd), W_DD, MQ_WL);
  cudaError_t e;
  if ((e = allow_max_smem(k_integrate_dd)) != cudaSuccess) return (int)e;
  if ((e = allow_max_smem(k_eval_points_dd)) != cudaSuccess) return (int)e;
  if ((e = allow_max_smem(k_eval_z_dd)) != cudaSuccess) return (int)e;
  int nsm = 0, occ = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_integrate_dd, TPB_DD, d->smem_dd)) != cudaSuccess) return (int)e;
  if (occ < 1) return (int)cudaErrorLaunchOutOfResources;
  d->grid_dd = std::min(MAXGRID, nsm * occ);
  return 0;
}
void mq_launch_integrate_dd(const mc_diagram *d, uint64_t seed, mq_stream st) {
  k_integrate_dd<<<d->grid_dd, TPB_DD, d->smem_dd, (cudaStream_t)st>>>(d->d_blob, seed, d->prec(false), d->ws.partial + (size_t)MAXGRID * 4, d->ws.flag_list, d->ws.lost_list, d->ws.counters);
}
void mq_launch_eval_points_dd(const mc_diagram *d, uint64_t first, uint64_t seed, double *f_out, mq_stream st) {
  k_eval_points_dd<<<d->grid_dd, TPB_DD, d->smem_dd, (cudaStream_t)st>>>(d->d_blob, first, seed, d->prec(false), f_out, d->ws.flag_list, d->ws.lost_list, d->ws.counters);
}
void mq_launch_eval_z_dd(const mc_diagram *d, int grid, uint64_t n, const double *z_in, double *fdd_out, mq_stream st) {
  k_eval_z_dd<<<grid, TPB_DD, d->smem_dd, (cudaStream_t)st>>>(d->d_blob, n, z_in, fdd_out);
}

// ---- batched path launchers ----
int mq_batch_config_dd(size_t smem, int *grid) {
  cudaError_t e;
  if ((e = allow_max_smem(k_batch_dd)) != cudaSuccess) return (int)e;
  int nsm = 0, occ = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_batch_dd, TPB_DD, smem)) != cudaSuccess) return (int)e;
  if (occ < 1) return (int)cudaErrorLaunchOutOfResources;
  *grid = nsm * occ;
  return 0;
}
size_t mq_batch_smem_dd(int scal_len) { return smem_bytes(scal_len, TPB_DD, sizeof(dd), W_DD, MQ_WL); }
void mq_launch_batch_dd(const BatchView &bv, int grid, size_t smem, uint64_t first, uint64_t seed, int scal_len, mq_stream st) {
  k_batch_dd<<<grid, TPB_DD, smem, (cudaStream_t)st>>>(bv, first, seed, scal_len);
}
