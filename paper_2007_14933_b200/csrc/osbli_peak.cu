// osbli_peak.cu -- DFMA micro-benchmark: the measured fp64-pipe peak this box sustains, used as the
// denominator of the "alu" roofline in bench.py (MEASURED_PEAKS.json carries no fp64 figure).
// 8 independent dependent-FMA chains per thread, 1024 threads per SM-resident block, no memory traffic.
#include "osbli_kernels.h"

namespace osbli {

__global__ void __launch_bounds__(1024)
dfma_peak_kernel(double *out, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-9, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0;
  double x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 123.456) out[0] = s;      // never true; keeps the chains alive
}

// Runs the kernel `reps` times on `st` between two events; returns TFLOP/s (2 flop per DFMA) of the best run.
cudaError_t measure_fp64_peak(double *d_scratch, cudaStream_t st, double *tflops) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  const int iters = 4096, blocks = sms * 2, threads = 1024;
  cudaEvent_t t0, t1;
  if ((e = cudaEventCreate(&t0)) != cudaSuccess) return e;
  if ((e = cudaEventCreate(&t1)) != cudaSuccess) return e;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(t0, st);
    dfma_peak_kernel<<<blocks, threads, 0, st>>>(d_scratch, iters, 0.999999, 1e-7);
    cudaEventRecord(t1, st);
    if ((e = cudaEventSynchronize(t1)) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, t0, t1);
    const double flop = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads;
    if (rep > 0 && ms > 0.f) best = fmax(best, flop / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(t0);
  cudaEventDestroy(t1);
  if (e == cudaSuccess) e = cudaGetLastError();
  *tflops = best;
  return e;
}

}  // namespace osbli
