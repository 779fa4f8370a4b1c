// microbench_lds_dfma.cu — stand-alone micro-benchmark behind the design rules of DESIGN.md §5 (not part of libmcqed.so):
//   (1) DFMA latency and the independent chains a scheduler needs to saturate the FP64 pipe,
//   (2) shared-memory load throughput per SM for broadcast and lane-distinct patterns, alone and next to N DFMA per load.
// Build and run on a B200:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/mb paper_1905_08007_b200/csrc/microbench_lds_dfma.cu && /tmp/mb
#include <cstdio>
#include <cuda_runtime.h>

__device__ __forceinline__ double2 lds128(unsigned a) { double2 v; asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a)); return v; }
__device__ __forceinline__ double lds64(unsigned a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }

template <int NCH> __global__ void k_chain(int iters, double *out, long long *cyc) {
  double a[8];
  for (int i = 0; i < 8; i++) a[i] = 1.0 + threadIdx.x * 1e-9 + i;
  const double m = 0.999999, c = 1e-9;
  const long long t0 = clock64();
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < 16; u++)
#pragma unroll
      for (int j = 0; j < NCH; j++) a[j] = fma(a[j], m, c);
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
  double s = 0;
  for (int j = 0; j < 8; j++) s += a[j];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
// groups = distinct addresses per warp (32 = every lane its own); WIDE: LDS.128 else LDS.64; NFMA = DFMA per load
template <int WIDE, int NFMA> __global__ void k_lds(int iters, int groups, int stride_bytes, double *out, long long *cyc) {
  extern __shared__ double sm[];
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sm[i] = 1.0 + i * 1e-9;
  __syncthreads();
  const int lane = threadIdx.x & 31, g = groups >= 32 ? lane : lane / (32 / groups);
  const unsigned base = (unsigned)__cvta_generic_to_shared(sm) + g * stride_bytes;
  double a[8] = {1.0, 1.1, 1.2, 1.3, 1.4, 1.5, 1.6, 1.7}, acc = 0;
  const long long t0 = clock64();
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < 16; u++) {
      double c;
      if (WIDE) { const double2 v = lds128(base + u * 512 + ((it & 3) << 4)); c = v.x; acc += v.y; }
      else c = lds64(base + u * 512 + ((it & 3) << 3));
#pragma unroll
      for (int j = 0; j < NFMA; j++) a[j] = fma(a[j], c, 0.5);
      if (NFMA == 0) acc += c;
    }
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
  double s = acc;
  for (int j = 0; j < 8; j++) s += a[j];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
static double mean_cycles(long long *cyc) { long long h[148]; cudaMemcpy(h, cyc, sizeof h, cudaMemcpyDeviceToHost); double c = 0; for (int i = 0; i < 148; i++) c += h[i]; return c / 148; }
template <int NCH> void run_chain(int tpb, double *out, long long *cyc) {
  const int iters = 4000;
  k_chain<NCH><<<148, tpb>>>(10, out, cyc); k_chain<NCH><<<148, tpb>>>(iters, out, cyc);
  const double c = mean_cycles(cyc), n = (double)iters * 16 * NCH;
  printf("DFMA  warps/scheduler=%d independent chains/warp=%d: %.2f cycles per DFMA per warp; %.3f warp-DFMA/cycle/SM\n", tpb / 128, NCH, c / n, n * (tpb / 32) / c);
}
template <int WIDE, int NFMA> void run_lds(const char *name, int groups, int stride, double *out, long long *cyc) {
  const int iters = 2000, tpb = 512;
  k_lds<WIDE, NFMA><<<148, tpb, 40000>>>(10, groups, stride, out, cyc); k_lds<WIDE, NFMA><<<148, tpb, 40000>>>(iters, groups, stride, out, cyc);
  const double c = mean_cycles(cyc), loads = (double)iters * 16 * (tpb / 32);
  printf("%-34s distinct addresses/warp=%2d: %.2f cycles per warp-load per SM; %.2f warp-DFMA/cycle/SM\n", name, groups, c / loads, loads * NFMA / c);
}
int main() {
  double *out; long long *cyc; cudaMalloc(&out, 148 * 1024 * 8); cudaMalloc(&cyc, 148 * 8);
  run_chain<1>(128, out, cyc); run_chain<2>(128, out, cyc); run_chain<4>(128, out, cyc); run_chain<8>(128, out, cyc);
  run_chain<1>(256, out, cyc); run_chain<2>(256, out, cyc); run_chain<1>(512, out, cyc); run_chain<1>(1024, out, cyc);
  run_lds<1, 0>("LDS.128 alone", 1, 16, out, cyc); run_lds<1, 0>("LDS.128 alone", 4, 16, out, cyc); run_lds<1, 0>("LDS.128 alone", 32, 16, out, cyc);
  run_lds<0, 0>("LDS.64 alone", 1, 8, out, cyc); run_lds<0, 0>("LDS.64 alone", 4, 8, out, cyc); run_lds<0, 0>("LDS.64 alone", 32, 8, out, cyc);
  run_lds<0, 1>("LDS.64 + 1 DFMA (1 point/lane)", 1, 8, out, cyc); run_lds<0, 2>("LDS.64 + 2 DFMA (2 points/lane)", 1, 8, out, cyc);
  run_lds<0, 4>("LDS.64 + 4 DFMA (4 points/lane)", 1, 8, out, cyc); run_lds<0, 8>("LDS.64 + 8 DFMA", 1, 8, out, cyc);
  run_lds<1, 2>("LDS.128 + 2 DFMA (1 point/lane)", 4, 16, out, cyc); run_lds<1, 4>("LDS.128 + 4 DFMA (2 points/lane)", 4, 16, out, cyc);
  run_lds<1, 8>("LDS.128 + 8 DFMA (4 points/lane)", 4, 16, out, cyc);
  return 0;
}
