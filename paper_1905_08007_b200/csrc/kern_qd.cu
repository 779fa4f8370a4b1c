// kern_qd.cu — third precision tier: quad-double re-evaluation of the points whose cancellation exceeds what
// double-double resolves (O8; "arithmetic with different precisions"). sm_100a.
// Product code (libmcqed.so); shares nothing with oracle/. Loop-based family code (family_spread), one point per CTA.
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

// Few points reach this tier (some 1e-5 of all), so the parallelism must come from inside a point: a CTA of TPB_QD threads
// works on ONE point at a time and deals the stream entries of every table to its threads (mcqed_kernels.cuh
// "entry-parallel"); the partial graded sums are added across the CTA once per table.
// Dynamic shared memory: [ S: scal_len x qd | xT: NW x NE x qd | xA: NW x NE x 8 | pad to 128 | 2 stream chunks | 2 mbarriers | slack ]
constexpr int TPB_QD = 256, QD_NW = TPB_QD / 32, QD_NE = 2 * MQ_MAXPAT * MQ_NGRADE;
__host__ __device__ inline size_t qd_head_bytes(int scal_len) {
  return (((size_t)scal_len * sizeof(qd) + (size_t)QD_NW * QD_NE * (sizeof(qd) + 8)) + 127) & ~(size_t)127;
}
inline size_t qd_smem_bytes(int scal_len) { return qd_head_bytes(scal_len) + 2 * MQ_CHUNK_WORDS * 8 + 16 + 64; }
struct QdRoles {
  qd *S, *xT; double *xA;
  __device__ __forceinline__ QdRoles(unsigned char *smem, int scal_len) {
    S = reinterpret_cast<qd *>(smem); xT = S + scal_len; xA = reinterpret_cast<double *>(xT + QD_NW * QD_NE);
  }
};
__device__ __forceinline__ void qd_setup_reader(StreamReader &rd, unsigned char *smem, int scal_len) {
  const size_t s = qd_head_bytes(scal_len);
  rd.init(reinterpret_cast<uint64_t *>(smem + s), reinterpret_cast<uint64_t *>(smem + s + 2 * MQ_CHUNK_WORDS * 8));
}
// the integrand of one point in quad-double, computed by the whole CTA; the value is valid in thread 0
__device__ __forceinline__ double qd_point(const DiagView &v, StreamReader &rd, const QdRoles &ro, const double *z) {
  qd f, a; double amin, xmin;
  eval_integrand<qd, 1, false, true>(v, rd, z, nullptr, reinterpret_cast<unsigned char *>(ro.S), 1, ro.xT, ro.xA, 0, 0, f, a, amin, xmin);
  return mq_to_double(f);
}

// points listed in lost_list (sample indices) by the double-double pass
__global__ void __launch_bounds__(TPB_QD) k_integrate_qd(const uint64_t *__restrict__ blob, uint64_t seed, double *partial,
                                                         const unsigned long long *lost_list, unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const QdRoles ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; qd_setup_reader(rd, smem_raw, v.h->max_scal_len);
  const unsigned long long cnt = counters[2] < LOSTCAP ? counters[2] : LOSTCAP;
  KahanPair s1{0.0, 0.0}, s2{0.0, 0.0};
  for (unsigned long long i = blockIdx.x; i < cnt; i += gridDim.x) {
    double z[MQ_MAXM];
    const double p = draw_point<false>(v, lost_list[i], seed, z, nullptr);
    const double fd = qd_point(v, rd, ro, z);
    if (threadIdx.x == 0) {
      if (bad_point(z, v.h->M, p) || !isfinite(fd)) atomicAdd(&counters[1], 1ull);     // dropped: w = 0
      else { const double w = fd / p; s1.add(w); s2.add(w * w); }
    }
  }
  if (threadIdx.x == 0) { double *d = partial + (size_t)blockIdx.x * 4; d[0] = s1.hi; d[1] = s1.lo; d[2] = s2.hi; d[3] = s2.lo; }
}

// batched path, quad-double tier: persistent CTAs; item = one entry of one diagram's lost list
__global__ void __launch_bounds__(TPB_QD) k_batch_qd(BatchView bv, uint64_t first, uint64_t seed, int scal_len) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ unsigned s_item; __shared__ int s_d;
  const QdRoles ro(smem_raw, scal_len);
  StreamReader rd; qd_setup_reader(rd, smem_raw, scal_len);
  const uint32_t total = bv.qd_start[bv.nd];
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) { s_item = (unsigned)atomicAdd(&bv.queue[2], 1ull); s_d = s_item < total ? batch_find(bv.qd_start, bv.nd, s_item) : 0; }
    __syncthreads();
    const uint32_t item = s_item;
    if (item >= total) break;
    const int d = s_d;
    const DiagView v = make_view(bv.dg[d].blob);
    const uint32_t rel = bv.lost_list[(size_t)d * bv.lostcap + (item - bv.qd_start[d])];
    double z[MQ_MAXM];
    const double p = draw_point<false>(v, batch_first(bv, d, first) + rel, seed, z, nullptr);
    const double fd = qd_point(v, rd, ro, z);
    if (threadIdx.x == 0) {
      double *dst = bv.part_qd + (size_t)item * 4;
      dst[0] = dst[1] = dst[2] = dst[3] = 0.0;
      if (bad_point(z, v.h->M, p) || !isfinite(fd)) atomicAdd(&bv.ndrop[d], 1ull);
      else { const double w = fd / p; dst[0] = w; dst[2] = w * w; }
    }
  }
}

// parity hooks: per-point values of the lost points (relative indices), and the integrand at given z
__global__ void __launch_bounds__(TPB_QD) k_eval_points_qd(const uint64_t *__restrict__ blob, uint64_t first, uint64_t seed, double *f_out,
                                                           const unsigned long long *lost_list, const unsigned long long *counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const QdRoles ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; qd_setup_reader(rd, smem_raw, v.h->max_scal_len);
  const unsigned long long cnt = counters[2] < LOSTCAP ? counters[2] : LOSTCAP;
  for (unsigned long long i = blockIdx.x; i < cnt; i += gridDim.x) {
    double z[MQ_MAXM];
    const unsigned long long rel = lost_list[i];
    draw_point<false>(v, first + rel, seed, z, nullptr);
    const double fd = qd_point(v, rd, ro, z);
    if (threadIdx.x == 0) f_out[rel] = fd;
  }
}
__global__ void __launch_bounds__(TPB_QD) k_eval_z_qd(const uint64_t *__restrict__ blob, uint64_t n, const double *__restrict__ z_in, double *fqd_out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const int M = v.h->M;
  const QdRoles ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; qd_setup_reader(rd, smem_raw, v.h->max_scal_len);
  for (uint64_t i = blockIdx.x; i < n; i += gridDim.x) {
    double z[MQ_MAXM];
    for (int k = 0; k < MQ_MAXM; k++) z[k] = k < M ? z_in[i * M + k] : 0.0;
    const double fd = qd_point(v, rd, ro, z);
    if (threadIdx.x == 0) fqd_out[i] = fd;
  }
}

}  // namespace mqk

using namespace mqk;

int mq_config_qd(mc_diagram *d) {
  d->smem_qd = qd_smem_bytes(d->max_scal_len);
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
  const int g = (int)std::min<uint64_t>((uint64_t)MAXGRID, n);
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
size_t mq_batch_smem_qd(int scal_len) { return qd_smem_bytes(scal_len); }
void mq_launch_batch_qd(const BatchView &bv, int grid, size_t smem, uint64_t first, uint64_t seed, int scal_len, mq_stream st) {
  k_batch_qd<<<grid, TPB_QD, smem, (cudaStream_t)st>>>(bv, first, seed, scal_len);
}
