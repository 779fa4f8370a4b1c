// kern_iv.cu — interval tier: the integrand at given points in binary64 INTERVAL arithmetic with directed rounding
// ("interval arithmetic"; iv_arith.cuh). A parity / validation hook (mc_eval_z_interval): the enclosure it returns
// contains the true value of the integrand at the given coordinates, whatever the cancellation. sm_100a.
// Product code (libmcqed.so); shares nothing with oracle/.
#include <cuda_runtime.h>

#include <algorithm>

#include "iv_arith.cuh"
#include "kern_common.cuh"

namespace mqk {

template <> __device__ __forceinline__ iv mq_shfl_xor<iv>(iv v, int m) { return iv(__shfl_xor_sync(0xffffffffu, v.lo, m), __shfl_xor_sync(0xffffffffu, v.hi, m)); }
template <> __device__ __forceinline__ iv lds_T<iv>(uint32_t a) { const double2 v = lds_f64x2(a); return iv(v.x, v.y); }

constexpr int TPB_IV = 128;

// one point per lane group (MQ_WL lane roles share it and split the families of every stream entry, as in the double-double tier)
__global__ void __launch_bounds__(TPB_IV) k_eval_z_iv(const uint64_t *__restrict__ blob, uint64_t n, const double *__restrict__ z_in, double *lo_out, double *hi_out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DiagView v = make_view(blob);
  const int M = v.h->M;
  const Roles<iv, 1, MQ_WL> ro(smem_raw, v.h->max_scal_len);
  StreamReader rd; setup_reader<1, MQ_WL>(rd, smem_raw, v.h->max_scal_len, sizeof(iv));
  for (uint64_t base = (uint64_t)blockIdx.x * ro.P; base < n; base += (uint64_t)gridDim.x * ro.P) {
    const bool live = base + ro.slot < n && ro.sub == 0;
    const uint64_t i = base + ro.slot < n ? base + ro.slot : n - 1;          // surplus slots redo the last point
    double z[MQ_MAXM];
    for (int k = 0; k < MQ_MAXM; k++) z[k] = k < M ? z_in[i * M + k] : 0.0;
    iv f, a; double amin, xmin;
    eval_integrand<iv, 1, true>(v, rd, z, nullptr, ro.S, ro.P, ro.xT, ro.xA, 0, ro.sub, f, a, amin, xmin);
    if (live) {
      const bool ok = f.lo <= f.hi;                                         // false for NaN: a division by an interval containing 0
      lo_out[i] = ok ? f.lo : -__longlong_as_double(0x7ff0000000000000ll);
      hi_out[i] = ok ? f.hi : __longlong_as_double(0x7ff0000000000000ll);
    }
  }
}

}  // namespace mqk

using namespace mqk;

int mq_launch_eval_z_iv(const mc_diagram *d, uint64_t n, const double *z_in, double *lo_out, double *hi_out, mq_stream st) {
  const size_t smem = smem_bytes(d->max_scal_len, TPB_IV, sizeof(iv), 1, MQ_WL);
  cudaError_t e;
  if ((e = allow_max_smem(k_eval_z_iv)) != cudaSuccess) return (int)e;
  const int P = TPB_IV / MQ_WL;
  const int grid = (int)std::min<uint64_t>(MAXGRID, (n + P - 1) / P);
  k_eval_z_iv<<<grid, TPB_IV, smem, (cudaStream_t)st>>>(d->d_blob, n, z_in, lo_out, hi_out);
  return (int)cudaGetLastError();
}
