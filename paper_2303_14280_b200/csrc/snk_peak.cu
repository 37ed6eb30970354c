// snk_peak.cu -- measured FP64 roofs of the GPU the library runs on: MEASURED_PEAKS.json has no
// FP64 entry, so the denominators of the a4/a5/a6 roofline fractions are measured here: a register-resident DFMA loop
// (vector FP64 pipe) and a DMMA.884 loop (fp64 mma.sync), both with enough independent chains to cover the pipe latency.
#include "snk_kernels.h"

namespace snk {
namespace {
constexpr int kChains = 8, kIters = 4096;

__global__ void __launch_bounds__(256) k_peak_dfma(double* out, double a, double b) {
  double v[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) v[i] = a + threadIdx.x * 1e-9 + i;
  for (int it = 0; it < kIters; ++it) {
#pragma unroll
    for (int i = 0; i < kChains; ++i) v[i] = fma(v[i], b, a);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += v[i];
  if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) k_peak_dmma(double* out, double a, double b) {
  double c[kChains][2];
#pragma unroll
  for (int i = 0; i < kChains; ++i) { c[i][0] = a + i; c[i][1] = b - i; }
  const double fa = a + (threadIdx.x & 31) * 1e-9, fb = b;
  for (int it = 0; it < kIters; ++it) {
#pragma unroll
    for (int i = 0; i < kChains; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(fa), "d"(fb));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += c[i][0] + c[i][1];
  if (s == 123.456) out[0] = s;
}
}  // namespace

cudaError_t run_fp64_peak(double* dfma_tflops, double* dmma_tflops, int reps) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* d = nullptr;
  if ((e = cudaMalloc(&d, 8)) != cudaSuccess) return e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = sms * 8, block = 256;
  double best[2] = {0, 0};
  for (int which = 0; which < 2; ++which)
    for (int r = 0; r < reps + 1; ++r) {
      cudaEventRecord(e0);
      if (which == 0) k_peak_dfma<<<grid, block>>>(d, 1.0, 0.999999);
      else k_peak_dmma<<<grid, block>>>(d, 1.0, 0.999999);
      cudaEventRecord(e1);
      if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
      float ms = 0;
      cudaEventElapsedTime(&ms, e0, e1);
      const double flops = which == 0 ? (double)grid * block * kIters * kChains * 2.0
                                      : (double)grid * (block / 32) * kIters * kChains * 512.0;
      if (r > 0) best[which] = fmax(best[which], flops / (ms * 1e-3) * 1e-12);
    }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d);
  if (e != cudaSuccess) return e;
  *dfma_tflops = best[0]; *dmma_tflops = best[1];
  return cudaGetLastError();
}
}  // namespace snk
