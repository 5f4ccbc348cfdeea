// k_microbench.cu -- the fp64 FMA peak of this device, measured ("per-kernel fp64 pipe
// utilisation vs a DFMA micro-benchmark peak"; MEASURED_PEAKS.json has no fp64 figure).
#include <cuda_runtime.h>

#include "../../include/erf_b200.h"

namespace erfb {

// 8 independent DFMA chains per thread, ITER * 8 FMAs each; the result is stored so nothing is optimised away
__global__ void __launch_bounds__(256) k_dfma(double *out, double a, double b, int iters) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
#pragma unroll 1
  for (int n = 0; n < iters; n++) {
#pragma unroll
    for (int m = 0; m < 8; m++) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

}  // namespace erfb

extern "C" int erf_measure_fp64_peak(double *tflops, void *stream) {
  if (!tflops) return ERF_EINVAL;
  *tflops = 0.0;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    return ERF_ECUDA;
  }
  const int blocks = sms * 8, threads = 256, iters = 4096;
  double *buf = nullptr;
  if (cudaMalloc(&buf, (size_t)blocks * threads * sizeof(double)) != cudaSuccess) {
    cudaGetLastError();
    return ERF_ENOMEM;
  }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; rep++) {  // first repetition warms up
    cudaEventRecord(e0, st);
    erfb::k_dfma<<<blocks, threads, 0, st>>>(buf, 0.999999, 1e-6, iters);
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(buf);
  if (cudaGetLastError() != cudaSuccess) return ERF_ECUDA;
  const double flops = 2.0 * 64.0 * iters * (double)blocks * threads;  // 64 FMAs per loop pass, 2 flop each
  *tflops = flops / (best * 1e-3) / 1e12;
  return ERF_OK;
}
