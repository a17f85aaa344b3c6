// The batch-first (AoS) adaptor of SURVEY.md section 8(f)4: the paper's workspace is (B, n, ...) batch-first
// (PAPER.md:103); the library's kernels are SoA, batch fastest (every warp access a full 128-byte line).  Callers with
// (B, n) tensors are served by a tiled transpose on the way in and on the way out, through a caller-owned workspace:
// [rows][cols] -> [cols][rows], 32 x 32 tiles through shared memory, 128-byte lines on both sides, one launch per array.
// (Addressing AoS from inside the operator kernels -- one element per thread and line -- was measured 20x slower on
// the write-dominated operators: humanoid FK at B = 65 536 280 us against 13.5 us SoA + 25 us of transposes.)
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <string>

#include "bard_internal.h"

namespace bard {
extern std::atomic<int64_t> g_launches;
namespace {

template <class T>
__global__ void __launch_bounds__(256) transpose_kernel(const T* __restrict__ src, T* __restrict__ dst, uint32_t rows, uint32_t cols) {
  __shared__ T tile[32][33];
  const uint32_t c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
  const uint32_t tx = threadIdx.x, ty = threadIdx.y;
#pragma unroll
  for (int k = 0; k < 32; k += 8) {
    const uint32_t r = r0 + ty + k, c = c0 + tx;
    if (r < rows && c < cols) tile[ty + k][tx] = src[(size_t)r * cols + c];
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 32; k += 8) {
    const uint32_t c = c0 + ty + k, r = r0 + tx;
    if (r < rows && c < cols) dst[(size_t)c * rows + r] = tile[tx][ty + k];
  }
}

}  // namespace

bard_status launch_transpose(const void* src, void* dst, int64_t rows, int64_t cols, int elem, void* stream) {
  if (rows <= 0 || cols <= 0) return BARD_OK;
  const dim3 block(32, 8), grid((unsigned)((cols + 31) / 32), (unsigned)((rows + 31) / 32));
  if (grid.y > 65535u) {                                      // AoS inputs put the batch on grid.y: 65535 x 32 environments
    set_error("bard_*_v: batch too large for the AoS adaptor (B <= 2 097 120)");
    return BARD_ERR_UNSUPPORTED;
  }
  if (elem == 8) transpose_kernel<double><<<grid, block, 0, (cudaStream_t)stream>>>((const double*)src, (double*)dst, (uint32_t)rows, (uint32_t)cols);
  else transpose_kernel<float><<<grid, block, 0, (cudaStream_t)stream>>>((const float*)src, (float*)dst, (uint32_t)rows, (uint32_t)cols);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_error(std::string("bard_*_v: transpose: ") + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
  g_launches.fetch_add(1);
  return BARD_OK;
}

}  // namespace bard
