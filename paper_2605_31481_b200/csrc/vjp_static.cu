// bard_rnea_vjp_params_static: bard_rnea_vjp_params for callers that cannot allocate device memory -- code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The operation is the one of vjp.cu (SURVEY.md
// section 8(f)3): the same two kernels, the same deterministic reduction; only the scratch
// (the per-CTA partial sums, [CTAs][nb * 10] floats) is not the caller's: it is the file-scope device array below.
//
// * Size: BARD_VJP_STATIC_SCRATCH_FLOATS floats = 1 MiB, held by every GPU that loads the library until the process
//   exits.  A call whose bard_rnea_vjp_workspace_floats(model, B) exceeds it is refused (BARD_ERR_UNSUPPORTED); on a
//   148-SM part that is a model of more than 44 bodies at a batch of more than ~18 600 environments.
// * In host code the array's NAME is a host-side stand-in, not a device address.  The device address is looked up once
//   per device, with that device current, by cudaGetSymbolAddress -- in this file, because the array is static -- and
//   that pointer is what the kernels get.
// * Every call on a device shares the array.  Nothing in it has to start at zero: rnea_vjp_kernel writes every partial
//   the reduction kernel then reads (all nb * 10 entries of every CTA of ITS grid), so the contents a previous call left
//   behind are never read.  Two calls that overlap on the GPU (different streams without an ordering between them, or
//   two host threads on different streams) RACE on it; calls on one stream are ordered and safe.
// * The call allocates nothing: no cudaMalloc / cudaFree, no allocating library routine.  The first call on a device
//   resolves the symbol (with lazy module loading that may load the module): make it once outside stream capture.
#include <cuda_runtime.h>

#include <mutex>
#include <string>

#include "bard_internal.h"

namespace bard {
namespace {

static __device__ __align__(256) float g_vjp_scratch[BARD_VJP_STATIC_SCRATCH_FLOATS];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
float* g_ptr[kMaxDevices] = {};     // device address of g_vjp_scratch on every device that asked for it

// The current device must be `device`.
bard_status scratch_address(int device, float** ptr) {
  if (device < 0 || device >= kMaxDevices) { set_error("bard_rnea_vjp_params_static: device ordinal out of range"); return BARD_ERR_UNSUPPORTED; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_ptr[device]) {
    float* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_vjp_scratch);
    if (e != cudaSuccess || !p) {
      set_error(std::string("bard_rnea_vjp_params_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
      cudaGetLastError();
      return BARD_ERR_CUDA;
    }
    g_ptr[device] = p;
  }
  *ptr = g_ptr[device];
  return BARD_OK;
}

}  // namespace

bard_status launch_rnea_vjp_static(const Model& M, int64_t B, const float* q, const float* qd, const float* qdd, const float* dtau,
                                   float* dparams, void* stream) {
  const size_t need = rnea_vjp_workspace_floats(M, B);
  if (need > (size_t)BARD_VJP_STATIC_SCRATCH_FLOATS) {
    set_error("bard_rnea_vjp_params_static: this model and batch need " + std::to_string(need) + " floats of scratch, the static array holds " +
              std::to_string((size_t)BARD_VJP_STATIC_SCRATCH_FLOATS) + ": use bard_rnea_vjp_params with a caller-owned workspace");
    return BARD_ERR_UNSUPPORTED;
  }
  float* ws = nullptr;
  const bard_status s = scratch_address(M.device, &ws);
  if (s != BARD_OK) return s;
  return launch_rnea_vjp(M, B, q, qd, qdd, dtau, dparams, ws, stream);
}

}  // namespace bard
