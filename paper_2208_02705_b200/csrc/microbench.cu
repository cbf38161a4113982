// r360 -- measurement helper for bench.py, NOT part of the product ABI: built into its own library
// (libr360_bench.so, build.py), so that libr360.so exports the method and nothing else.
// The FP32 FMA rate of this GPU, the roofline of the fp32 MLP path (bound "alu").  SURVEY.md 8(d): "not in
// MEASURED_PEAKS.json -- measure with an FMA microbenchmark on the box and use that".
#include <cuda_runtime.h>

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

#define BENCH_CUDA(call)                       \
  do {                                         \
    cudaError_t e_ = (call);                   \
    if (e_ != cudaSuccess) return (int)e_;     \
  } while (0)

// TFLOP/s (2 FLOP per FMA; best of five launches of a register-only FMA kernel that fills every SM) and the nominal
// SM clock of the current device.  Returns 0, -1 for a null argument, or the cudaError_t of a failed call.
extern "C" int r360bench_fp32_fma(double* tflops_out, double* sm_mhz_out) {
  if (!tflops_out) return -1;
  int dev = 0, n_sms = 0, khz = 0;
  BENCH_CUDA(cudaGetDevice(&dev));
  BENCH_CUDA(cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev));
  BENCH_CUDA(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  float* d = nullptr;
  BENCH_CUDA(cudaMalloc(&d, 4));
  cudaEvent_t e0, e1;
  BENCH_CUDA(cudaEventCreate(&e0));
  BENCH_CUDA(cudaEventCreate(&e1));
  const int iters = 4096, blocks = n_sms * 2 * 4;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0, 0);
    k_fma_peak<<<blocks, 1024>>>(d, iters, 0.999f, 1e-3f);
    cudaEventRecord(e1, 0);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaFree(d); return (int)e; }
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
  return 0;
}
