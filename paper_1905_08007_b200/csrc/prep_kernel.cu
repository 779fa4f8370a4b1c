// prep_kernel.cu — prepare-time accelerator: counts the spinor paths of the gamma strings on the GPU.
// Product code (libmcqed.so); shares nothing with oracle/. Same walk as mq::detail::Walker (coef_gen.hpp):
// for fixed Lorentz indices a basis spinor follows one path through the string (every factor is a
// generalised permutation matrix or a block projector), so a coefficient is a signed path count.
// One CTA per unit; the first up to three summed indices are spread over 64 threads, the rest is an
// explicit-stack depth-first walk; counts are accumulated with shared-memory integer atomics.
#include <cuda_runtime.h>

#include "device_layout.h"

namespace {

__constant__ int8_t c_dst[4][4] = {{0, 1, 2, 3}, {3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}};
__constant__ int8_t c_ph[4][4] = {{0, 0, 2, 2}, {2, 2, 0, 0}, {3, 1, 1, 3}, {2, 0, 0, 2}};

__global__ void __launch_bounds__(64) k_count_paths(const MqCountUnit *__restrict__ units, int32_t *__restrict__ counts) {
  extern __shared__ int32_t acc[];
  __shared__ MqCountUnit u;
  if (threadIdx.x < sizeof(MqCountUnit) / 4) reinterpret_cast<uint32_t *>(&u)[threadIdx.x] = reinterpret_cast<const uint32_t *>(&units[blockIdx.x])[threadIdx.x];
  __syncthreads();
  const int nsig2 = 2 * (int)u.nsig;
  for (int i = threadIdx.x; i < nsig2; i += blockDim.x) acc[i] = 0;
  __syncthreads();
  const int d = u.npairs < 3 ? u.npairs : 3;          // indices fixed by the thread id
  if ((int)threadIdx.x < (1 << (2 * d))) {
    int8_t rho[16];
    int st_pos[12], st_s[12], st_ph[12], st_r[12]; uint32_t st_sig[12];
    int level = 0, pos = 0, s = u.start, ph = 0; uint32_t sig = 0;
    const int n = u.n, start = u.start;
    for (;;) {
      bool leaf = true;
      while (pos < n) {
        const MqWElem e = u.el[pos];
        if (e.type == MQ_W_OPEN) { leaf = false; break; }
        if (e.type == MQ_W_FIX) { ph += c_ph[e.arg][s]; s = c_dst[e.arg][s]; }
        else if (e.type == MQ_W_G0) { ph += (s >= 2) ? 2 : 0; }
        else if (e.type == MQ_W_BIN) { sig |= (uint32_t)(s >= 2) << e.arg; }
        else { const int r = rho[e.arg]; ph += c_ph[r][s] + (r ? 2 : 0); s = c_dst[r][s]; }
        pos++;
      }
      if (!leaf) {                                     // an index opens here
        const MqWElem e = u.el[pos];
        int r;
        if (level < d) r = (threadIdx.x >> (2 * level)) & 3;
        else { st_pos[level] = pos; st_s[level] = s; st_ph[level] = ph; st_sig[level] = sig; st_r[level] = 0; r = 0; }
        rho[e.arg] = (int8_t)r; ph += c_ph[r][s]; s = c_dst[r][s]; pos++; level++;
        continue;
      }
      if (s == start) atomicAdd(&acc[2 * sig + (ph & 1)], (ph & 2) ? -1 : 1);
      // backtrack to the deepest index that still has values left
      bool more = false;
      while (level > d) {
        level--;
        const int r = ++st_r[level];
        if (r < 4) {
          pos = st_pos[level]; s = st_s[level]; ph = st_ph[level]; sig = st_sig[level];
          const MqWElem e = u.el[pos];
          rho[e.arg] = (int8_t)r; ph += c_ph[r][s]; s = c_dst[r][s]; pos++; level++;
          more = true; break;
        }
      }
      if (!more) break;
    }
  }
  __syncthreads();
  int32_t *out = counts + u.off;
  for (int i = threadIdx.x; i < nsig2; i += blockDim.x) out[i] = acc[i];
}

}  // namespace

// returns 0 on success (cudaError_t otherwise); counts must hold nints int32
int mq_count_units_gpu(const MqCountUnit *units, size_t nunits, int32_t *counts, size_t nints) {
  if (nunits == 0) return 0;
  MqCountUnit *d_units = nullptr; int32_t *d_counts = nullptr;
  cudaError_t e;
  if ((e = cudaMalloc(&d_units, nunits * sizeof(MqCountUnit))) != cudaSuccess) return (int)e;
  if ((e = cudaMalloc(&d_counts, nints * sizeof(int32_t))) != cudaSuccess) { cudaFree(d_units); return (int)e; }
  e = cudaMemcpy(d_units, units, nunits * sizeof(MqCountUnit), cudaMemcpyHostToDevice);
  uint32_t maxsig = 1;
  for (size_t i = 0; i < nunits; i++) if (units[i].nsig > maxsig) maxsig = units[i].nsig;
  const size_t smem = 2 * (size_t)maxsig * sizeof(int32_t);
  if (e == cudaSuccess && smem > 48 * 1024) e = cudaFuncSetAttribute(k_count_paths, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) {
    k_count_paths<<<(unsigned)nunits, 64, smem>>>(d_units, d_counts);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(counts, d_counts, nints * sizeof(int32_t), cudaMemcpyDeviceToHost);
  cudaFree(d_units); cudaFree(d_counts);
  return (int)e;
}
