// wt_measure_fp32_fma: the FP32 FMA rate of the device, measured ("MEASURED_PEAKS.json has no fp32
// figure -- measure one").  A helper for bench.py's roofline object, not part of the hot path.
#include <cuda_runtime.h>

#include <algorithm>

#include "geometry.h"

namespace {
// 8 independent FMA chains per thread, `iters` x 8 x 4 dependent steps each
__global__ void __launch_bounds__(256) k_fma_peak(float* out, int iters, float a, float b) {
  float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
      x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
    }
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}
}  // namespace

// Enqueues the measurement on `cuda_stream` and WAITS for it (the only call of the library that synchronises: it is a
// measurement, not part of the path).  scratch_dev: >= 148 * 8 * 256 * 4 bytes.  *tflops = 2 flops per FMA.
extern "C" int wt_measure_fp32_fma(void* scratch_dev, size_t scratch_bytes, void* cuda_stream, double* tflops) {
  if (!scratch_dev || !cuda_stream || !tflops) { wt_set_error("wt_measure_fp32_fma: null argument"); return WT_EINVAL; }
  int dev = 0, n_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    wt_set_error("wt_measure_fp32_fma: no device"); return WT_ECUDA;
  }
  const int blocks = n_sm * 8, threads = 256, iters = 4096;
  if (scratch_bytes < (size_t)blocks * threads * sizeof(float)) { wt_set_error("wt_measure_fp32_fma: scratch too small"); return WT_ENOMEM; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0, st);
    k_fma_peak<<<blocks, threads, 0, st>>>((float*)scratch_dev, iters, 0.999f, 0.001f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { wt_set_error("wt_measure_fp32_fma: kernel failed"); return WT_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flops = 2.0 * 32.0 * iters * (double)blocks * threads;
    if (ms > 0.f) best = std::max(best, flops / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  g_wt_launches += 5;
  *tflops = best;
  wt_set_error("");
  return WT_OK;
}
