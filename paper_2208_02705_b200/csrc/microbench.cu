// r360 -- measurement helper: the FP32 FMA rate of this GPU, the roofline of the fp32 MLP path (bound "alu").
// "not in MEASURED_PEAKS.json -- measure with an FMA microbenchmark on the box and use that".
#include "scene.h"

namespace {

// 16 independent FMA chains per thread (enough to cover the 4-cycle FMA latency with 2 resident blocks of 1024 threads per SM)
__global__ void __launch_bounds__(1024, 2) k_fma_peak(float* out, int iters, float a, float b) {
  float x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  if (s == 123.456f) out[0] = s;          // never true: keeps the chains alive
}

}  // namespace

extern "C" r360_status r360_measure_fp32_fma(double* tflops_out, double* sm_mhz_out) {
  if (!tflops_out) return R360_ERR_INVALID_ARG;
  int dev = 0, n_sms = 0, khz = 0;
  R360_CUDA(cudaGetDevice(&dev));
  R360_CUDA(cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev));
  R360_CUDA(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  float* d = nullptr;
  R360_CUDA(cudaMalloc(&d, 4));
  cudaEvent_t e0, e1;
  R360_CUDA(cudaEventCreate(&e0));
  R360_CUDA(cudaEventCreate(&e1));
  const int iters = 4096, blocks = n_sms * 2 * 4;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0, 0);
    k_fma_peak<<<blocks, 1024>>>(d, iters, 0.999f, 1e-3f);
    cudaEventRecord(e1, 0);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaFree(d); return r360_cuda_fail(e, "k_fma_peak"); }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = 2.0 * 16.0 * (double)iters * 1024.0 * (double)blocks;
    const double tf = flop / ((double)ms * 1e-3) / 1e12;
    if (rep > 0 && tf > best) best = tf;     // first launch is the warm-up
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  *tflops_out = best;
  if (sm_mhz_out) *sm_mhz_out = (double)khz / 1e3;
  return R360_OK;
}
