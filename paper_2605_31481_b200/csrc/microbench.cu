// bard_measure_fp32_peak: the plain-FP32 (non-tensor) FMA throughput of the device, measured -- the denominator of the
// "alu" roofline ("the builder must ... measure an FMA-only microbenchmark on the box, and use
// the measured figure").  Eight independent FFMA chains per thread, 1024 threads per CTA, two CTAs per SM, 4096 x 8 FMAs
// per chain step; CUDA events around the second of two launches.  Utility only: no operator depends on it.
#include <cuda_runtime.h>

#include <string>

#include "bard_internal.h"

namespace bard {
namespace {
__global__ void __launch_bounds__(1024) ffma_kernel(float* out, float a, float b, int iters) {
  float x0 = threadIdx.x * 1e-3f, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
      x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
    }
  }
  const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;      // never true: keeps the chains alive
}
}  // namespace
}  // namespace bard

extern "C" bard_status bard_measure_fp32_peak(int cuda_device, double* tflops) {
  if (!tflops || cuda_device < 0) { bard::set_error("bard_measure_fp32_peak: bad arguments"); return BARD_ERR_INVALID_ARG; }
  bard::DeviceGuard guard(cuda_device);
  int sms = 0;
  cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device);
  float* out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  const int grid = sms * 2, block = 1024, iters = 4096;
  if (e == cudaSuccess) e = cudaMalloc(&out, sizeof(float) * (size_t)grid * block);
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  double best = 0.0;
  for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {
    cudaEventRecord(e0, 0);
    bard::ffma_kernel<<<grid, block>>>(out, 0.999f, 1e-3f, iters);
    cudaEventRecord(e1, 0);
    e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    const double flop = 2.0 * 64.0 * iters * (double)grid * block;
    if (e == cudaSuccess && rep > 0 && ms > 0.f) best = std::max(best, flop / (ms * 1e-3) / 1e12);
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (out) cudaFree(out);
  if (e != cudaSuccess) { bard::set_error(std::string("bard_measure_fp32_peak: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
  *tflops = best;
  return BARD_OK;
}
