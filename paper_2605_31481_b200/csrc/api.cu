// C ABI (include/bard.h): argument checks, table export, dispatch to the kernel launchers.
#include <cuda_runtime.h>

#include <atomic>
#include <cctype>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "bard_internal.h"

// bard_step's fork-join: three side streams and the events that order them against the caller's stream.
// Created once with the model, so that bard_step itself allocates nothing.
struct StepFork {
  cudaStream_t side[3] = {nullptr, nullptr, nullptr};
  cudaEvent_t fork = nullptr, join[3] = {nullptr, nullptr, nullptr};
  std::mutex mu;              // one fork-join is enqueued at a time (the events are re-recorded by every call)
  bool ok = false;
};

struct bard_model {
  bard::Model m;
  StepFork fj;
};

namespace bard {
static thread_local std::string g_err;
std::atomic<int64_t> g_launches{0};
void set_error(const std::string& s) { g_err = s; }
bool& launching_side_by_side() { static thread_local bool v = false; return v; }

DeviceGuard::DeviceGuard(int device) {
  if (device < 0 || cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return; }
  if (prev != device) switched = cudaSetDevice(device) == cudaSuccess;
}
DeviceGuard::~DeviceGuard() {
  if (switched) cudaSetDevice(prev);
}

// option name -> field; the environment default of option "x" is BARD_X
bool option_ref(Options& o, const char* key, int64_t** ref) {
  if (!key) return false;
#define BARD_OPT_REF(name, dflt) if (std::strcmp(key, #name) == 0) { *ref = &o.name; return true; }
  BARD_OPTIONS(BARD_OPT_REF)
#undef BARD_OPT_REF
  return false;
}
void options_from_env(Options& o) {
  auto env = [](const char* name, int64_t& dst) {
    std::string e = "BARD_";
    for (const char* c = name; *c; ++c) e += (char)std::toupper((unsigned char)*c);
    if (const char* v = std::getenv(e.c_str())) dst = std::atoll(v);
  };
#define BARD_OPT_ENV(name, dflt) env(#name, o.name);
  BARD_OPTIONS(BARD_OPT_ENV)
#undef BARD_OPT_ENV
}
bard_status build_model(const bard_model_desc* d, int device, Model& M);
bard_status set_frames(Model& M, int32_t nframes, const int32_t* body, const double* offset);
}  // namespace bard

using bard::set_error;

extern "C" {

bard_status bard_model_create(const bard_model_desc* desc, int cuda_device, bard_model** out) {
  if (!out) { set_error("bard_model_create: out is NULL"); return BARD_ERR_INVALID_ARG; }
  bard_model* bm = new (std::nothrow) bard_model();
  if (!bm) { set_error("bard_model_create: host allocation failed"); return BARD_ERR_ALLOC; }
  bard_status s = bard::build_model(desc, cuda_device, bm->m);
  if (s != BARD_OK) { delete bm; return s; }
  if (bm->m.d_blob) {         // device model: the fork-join plumbing of bard_step (not fatal if it cannot be created)
    int prev = 0;
    cudaGetDevice(&prev);
    cudaSetDevice(bm->m.device);
    StepFork& f = bm->fj;
    bool ok = cudaEventCreateWithFlags(&f.fork, cudaEventDisableTiming) == cudaSuccess;
    for (int k = 0; k < 3 && ok; ++k)
      ok = cudaStreamCreateWithFlags(&f.side[k], cudaStreamNonBlocking) == cudaSuccess &&
           cudaEventCreateWithFlags(&f.join[k], cudaEventDisableTiming) == cudaSuccess;
    f.ok = ok;
    if (!ok) cudaGetLastError();
    cudaSetDevice(prev);
  }
  *out = bm;
  return BARD_OK;
}

void bard_model_destroy(bard_model* bm) {
  if (!bm) return;
  if (bm->m.d_blob) {
    int prev = 0;
    cudaGetDevice(&prev);
    cudaSetDevice(bm->m.device);
    cudaFree(bm->m.d_blob);
    if (bm->m.d_jblob) cudaFree(bm->m.d_jblob);
    for (int k = 0; k < 3; ++k) {
      if (bm->fj.side[k]) cudaStreamDestroy(bm->fj.side[k]);
      if (bm->fj.join[k]) cudaEventDestroy(bm->fj.join[k]);
    }
    if (bm->fj.fork) cudaEventDestroy(bm->fj.fork);
    cudaSetDevice(prev);
  }
  bard::free_specialized(bm->m.spec);
  delete bm;
}

bard_status bard_model_dims(const bard_model* bm, int32_t* nb, int32_t* nq, int32_t* nv, int32_t* nlevels) {
  if (!bm) { set_error("bard_model_dims: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (nb) *nb = bm->m.nb;
  if (nq) *nq = bm->m.nq;
  if (nv) *nv = bm->m.nv;
  if (nlevels) *nlevels = bm->m.nlevels;
  return BARD_OK;
}

bard_status bard_model_get_table(const bard_model* bm, int table_id, void* host_dst, size_t cap, size_t* need) {
  if (!bm) { set_error("bard_model_get_table: model is NULL"); return BARD_ERR_INVALID_ARG; }
  const bard::Model& m = bm->m;
  const void* src = nullptr;
  size_t bytes = 0;
  auto vec32 = [&](const std::vector<int32_t>& v) { src = v.data(); bytes = v.size() * sizeof(int32_t); };
  switch (table_id) {
    case BARD_TAB_LEVEL_PTR: vec32(m.level_ptr); break;
    case BARD_TAB_LEVEL_BODY: vec32(m.level_body); break;
    case BARD_TAB_BODY_LEVEL: vec32(m.body_level); break;
    case BARD_TAB_PARENT_SLOT: vec32(m.parent_slot); break;
    case BARD_TAB_Q_OFF: vec32(m.q_off); break;
    case BARD_TAB_V_OFF: vec32(m.v_off); break;
    case BARD_TAB_DOF_BODY: vec32(m.dof_body); break;
    case BARD_TAB_ANC_MASK: src = m.anc_mask.data(); bytes = m.anc_mask.size() * sizeof(uint64_t); break;
    case BARD_TAB_RODRIGUES: src = m.rodrigues.data(); bytes = m.rodrigues.size() * sizeof(float); break;
    default: set_error("bard_model_get_table: unknown table id"); return BARD_ERR_INVALID_ARG;
  }
  if (need) *need = bytes;
  if (cap < bytes || (!host_dst && bytes)) {
    set_error("bard_model_get_table: destination too small");
    return BARD_ERR_INVALID_ARG;
  }
  if (bytes) std::memcpy(host_dst, src, bytes);
  return BARD_OK;
}

bard_status bard_model_set_frames(bard_model* bm, int32_t nframes, const int32_t* body, const double* offset) {
  if (!bm) { set_error("bard_model_set_frames: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (bm->m.d_blob) {
    // The J tables are rewritten in place and the generated Jacobian / step kernels are unloaded: nothing that reads
    // them may still be in flight -- on the caller's streams, on non-blocking streams, or on bard_step's own side
    // streams.  set_frames is a rare, build-time call: wait for the whole device.
    bard::DeviceGuard guard(bm->m.device);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { set_error(std::string("bard_model_set_frames: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
  }
  bard::drop_specialized_jacobian(bm->m);
  return bard::set_frames(bm->m, nframes, body, offset);
}

// Which form of bard_step is faster for THIS model on THIS device at small batches, measured: the forked step and the one-
// / two-launch step at B = 4096 and 16 384 on scratch buffers (zeros; unit quaternions), eight plain calls each on a stream
// of its own between CUDA events -- plain calls on purpose: a caller that does not replay CUDA graphs pays the fork-join's
// sixteen API calls (15-20 us).  The faster form decides where the fork regime ends (specialize.cu: step_fork_max_b): 3072
// if the one- / two-launch form wins already at 4096, 8192 if it wins at 16 384, 128 x SMs otherwise.  Under stream capture
// the host cost does not exist and forking pays a little longer: where the plain-call answer is below 8192 the captured
// one is 8192 (graph replay on the four robots: spined quadruped at 4096 / 8192 forked 10.8 / 10.8 us, fused 13.1 / 13.1; at
// 12 288 13.1 / 13.3; chain-7 6.2-6.9 / 6.9).  That second answer is a rule, not a measurement, because measuring it means
// building a CUDA graph here, and a process that has launched one ran the humanoid's 65 536-environment step 3 % slower
// afterwards (96.7 against 93.6 us, reproducibly).  Best effort: any failure leaves the static rule in charge.
static void calibrate_step(bard_model* bm) {
  bard::Model& m = bm->m;
  m.fork_max_cal[0] = m.fork_max_cal[1] = -1;
  if (!m.d_blob || m.nv == 0 || m.nframes == 0 || m.opt.step_calibrate == 0 || m.opt.step_fork_max_b >= 0 || !bm->fj.ok) return;
  const int64_t sizes[2] = {4096, 16384}, Bmax = sizes[1];
  const size_t n_in = (size_t)(m.nq + 2 * m.nv) * Bmax;
  const size_t n_out = ((size_t)12 * m.nb + (size_t)6 * m.nframes * m.nv + (size_t)m.nv + (size_t)m.nv * m.nv) * Bmax;
  bard::DeviceGuard guard(m.device);
  float* buf = nullptr;
  cudaStream_t st = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  const int64_t keep_mode = m.opt.step_mode;
  float t[2][2] = {};                                // [batch][forked / not]
  bool ok = cudaMalloc(&buf, sizeof(float) * (n_in + n_out)) == cudaSuccess &&
            cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) == cudaSuccess && cudaEventCreate(&e0) == cudaSuccess &&
            cudaEventCreate(&e1) == cudaSuccess && cudaMemsetAsync(buf, 0, sizeof(float) * n_in, st) == cudaSuccess;
  for (int sz = 0; sz < 2 && ok; ++sz) {
    const int64_t B = sizes[sz];
    float *q = buf, *qd = buf + (size_t)m.nq * B, *qdd = qd + (size_t)m.nv * B, *pose = buf + n_in, *J = pose + (size_t)12 * m.nb * B,
          *tau = J + (size_t)6 * m.nframes * m.nv * B, *Mo = tau + (size_t)m.nv * B;
    const std::vector<float> ones((size_t)B, 1.0f);
    ok = cudaMemsetAsync(buf, 0, sizeof(float) * n_in, st) == cudaSuccess;
    for (int i = 0; i < m.nb && ok; ++i)           // unit quaternions
      if (m.jtype[i] == BARD_JOINT_FREE)
        ok = cudaMemcpyAsync(q + (size_t)(m.q_off[i] + 6) * B, ones.data(), sizeof(float) * B, cudaMemcpyHostToDevice, st) == cudaSuccess &&
             cudaStreamSynchronize(st) == cudaSuccess;
    for (int form = 0; form < 2 && ok; ++form) {
      m.opt.step_mode = form == 0 ? 1 : -1;         // forked / whatever follows the fork regime
      m.fork_max_cal[0] = m.fork_max_cal[1] = form == 0 ? -1 : 0;
      for (int k = 0; k < 11 && ok; ++k) {          // plain calls
        if (k == 3) ok = cudaEventRecord(e0, st) == cudaSuccess;
        ok = ok && bard_step(bm, B, q, qd, qdd, pose, J, tau, Mo, st) == BARD_OK;
      }
      ok = ok && cudaEventRecord(e1, st) == cudaSuccess && cudaStreamSynchronize(st) == cudaSuccess && cudaEventElapsedTime(&t[sz][form], e0, e1) == cudaSuccess;
    }
  }
  m.opt.step_mode = keep_mode;
  m.fork_max_cal[0] = !ok ? -1 : t[0][1] < t[0][0] ? 96 * 32 : t[1][1] < t[1][0] ? 8192 : 128 * (int64_t)m.sm_count;
  m.fork_max_cal[1] = !ok ? -1 : std::max<int64_t>(m.fork_max_cal[0], 8192);
  if (!ok) cudaGetLastError();
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (st) cudaStreamDestroy(st);
  if (buf) cudaFree(buf);
}

bard_status bard_model_specialize(bard_model* bm, uint32_t ops) {
  if (!bm) { set_error("bard_model_specialize: model is NULL"); return BARD_ERR_INVALID_ARG; }
  const bard_status s = bard::specialize(bm->m, ops);
  if (s == BARD_OK && (ops & BARD_OP_FUSED)) calibrate_step(bm);
  return s;
}

bard_status bard_model_set_option(bard_model* bm, const char* key, int64_t value) {
  if (!bm) { set_error("bard_model_set_option: model is NULL"); return BARD_ERR_INVALID_ARG; }
  int64_t* ref = nullptr;
  if (!bard::option_ref(bm->m.opt, key, &ref)) { set_error(std::string("bard_model_set_option: unknown option: ") + (key ? key : "(null)")); return BARD_ERR_INVALID_ARG; }
  *ref = value;
  return BARD_OK;
}

bard_status bard_model_get_option(const bard_model* bm, const char* key, int64_t* value) {
  if (!bm || !value) { set_error("bard_model_get_option: NULL argument"); return BARD_ERR_INVALID_ARG; }
  if (key && std::strcmp(key, "step_fork_regime") == 0) { *value = bard::step_fork_max_b(bm->m, false); return BARD_OK; }   // read-only: the rule's current answer
  if (key && std::strcmp(key, "step_fork_regime_captured") == 0) { *value = bard::step_fork_max_b(bm->m, true); return BARD_OK; }
  int64_t* ref = nullptr;
  if (!bard::option_ref(const_cast<bard_model*>(bm)->m.opt, key, &ref)) { set_error(std::string("bard_model_get_option: unknown option: ") + (key ? key : "(null)")); return BARD_ERR_INVALID_ARG; }
  *value = *ref;
  return BARD_OK;
}

bard_status bard_model_specialized_source(const bard_model* bm, uint32_t op, char* host_dst, size_t cap, size_t* need) {
  if (!bm) { set_error("bard_model_specialized_source: model is NULL"); return BARD_ERR_INVALID_ARG; }
  const std::string* src = bard::specialized_source(bm->m, op);
  if (!src) { set_error("bard_model_specialized_source: operator not specialised"); return BARD_ERR_INVALID_ARG; }
  if (need) *need = src->size() + 1;
  if (cap < src->size() + 1 || !host_dst) { set_error("bard_model_specialized_source: destination too small"); return BARD_ERR_INVALID_ARG; }
  std::memcpy(host_dst, src->c_str(), src->size() + 1);
  return BARD_OK;
}

static bard_status check_call(const char* fn, const bard_model* bm, int64_t B, const void* a, const void* b,
                              const void* c, const void* d) {
  if (!bm) { set_error(std::string(fn) + ": model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (!bm->m.d_blob) { set_error(std::string(fn) + ": host-only model (created with cuda_device < 0)"); return BARD_ERR_INVALID_ARG; }
  if (B < 0) { set_error(std::string(fn) + ": negative batch size"); return BARD_ERR_INVALID_ARG; }
  if (B > 0 && (!a || !b || !c || !d)) { set_error(std::string(fn) + ": NULL device pointer"); return BARD_ERR_INVALID_ARG; }
  // 4 B must fit 32 bits (row-stride arithmetic in the kernels)
  if (B > ((int64_t)1 << 29)) { set_error(std::string(fn) + ": B too large"); return BARD_ERR_UNSUPPORTED; }
  return BARD_OK;
}

bard_status bard_fk(const bard_model* bm, int64_t B, const float* q, float* pose, bard_stream stream) {
  bard_status s = check_call("bard_fk", bm, B, bm && bm->m.nq == 0 ? (const void*)pose : q, pose, pose, pose);
  if (s != BARD_OK || B == 0) return s;
  bard::DeviceGuard guard(bm->m.device);
  if (bard::launch_specialized(bm->m, BARD_OP_FK, B, q, nullptr, nullptr, pose, nullptr, nullptr, nullptr, stream, s)) return s;
  return bard::launch_fk(bm->m, B, q, pose, stream);
}

bard_status bard_jacobian(const bard_model* bm, int64_t B, const float* q, float* J, bard_stream stream) {
  if (!bm) { set_error("bard_jacobian: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (bm->m.nframes == 0 || bm->m.nv == 0) return check_call("bard_jacobian", bm, B, bm, bm, bm, bm);  // empty output
  bard_status s = check_call("bard_jacobian", bm, B, bm->m.nq == 0 ? (const void*)J : q, J, J, J);
  if (s != BARD_OK || B == 0) return s;
  bard::DeviceGuard guard(bm->m.device);
  if (bard::launch_specialized(bm->m, BARD_OP_JACOBIAN, B, q, nullptr, nullptr, nullptr, J, nullptr, nullptr, stream, s)) return s;
  return bard::launch_jacobian(bm->m, B, q, J, stream);
}

bard_status bard_rnea(const bard_model* bm, int64_t B, const float* q, const float* qd, const float* qdd, float* tau,
                      bard_stream stream) {
  if (bm && bm->m.nv == 0) return check_call("bard_rnea", bm, B, bm, bm, bm, bm);  // nothing to write
  bard_status s = check_call("bard_rnea", bm, B, q, qd, qdd, tau);
  if (s != BARD_OK || B == 0) return s;
  bard::DeviceGuard guard(bm->m.device);
  if (bard::launch_specialized(bm->m, BARD_OP_RNEA, B, q, qd, qdd, nullptr, nullptr, tau, nullptr, stream, s)) return s;
  return bard::launch_rnea(bm->m, B, q, qd, qdd, tau, stream);
}

bard_status bard_crba(const bard_model* bm, int64_t B, const float* q, float* M, bard_stream stream) {
  if (bm && bm->m.nv == 0) return check_call("bard_crba", bm, B, bm, bm, bm, bm);
  bard_status s = check_call("bard_crba", bm, B, q, M, M, M);
  if (s != BARD_OK || B == 0) return s;
  bard::DeviceGuard guard(bm->m.device);
  if (bard::launch_specialized(bm->m, BARD_OP_CRBA, B, q, nullptr, nullptr, nullptr, nullptr, nullptr, M, stream, s)) return s;
  return bard::launch_crba(bm->m, B, q, M, stream);
}

bard_status bard_kinematics(const bard_model* bm, int64_t B, const float* q, float* pose, float* J, float* M, bard_stream stream) {
  if (!bm) { set_error("bard_kinematics: model is NULL"); return BARD_ERR_INVALID_ARG; }
  bard::DeviceGuard guard(bm->m.device);
  if (bm->m.nv > 0 && bm->m.nframes > 0) {
    bard_status s = check_call("bard_kinematics", bm, B, bm->m.nq ? (const void*)q : (const void*)pose, pose, J, M);
    if (s != BARD_OK || B == 0) return s;
    if (bard::launch_kin(bm->m, B, q, pose, J, M, stream, s)) return s;     // one walk, one launch
  }
  bard_status s = bard_fk(bm, B, q, pose, stream);
  if (s == BARD_OK) s = bard_jacobian(bm, B, q, J, stream);
  if (s == BARD_OK) s = bard_crba(bm, B, q, M, stream);
  return s;
}

bard_status bard_step(const bard_model* bm, int64_t B, const float* q, const float* qd, const float* qdd, float* pose, float* J,
                      float* tau, float* M, bard_stream stream) {
  if (!bm) { set_error("bard_step: model is NULL"); return BARD_ERR_INVALID_ARG; }
  bard::DeviceGuard guard(bm->m.device);
  // Which form the step takes (measured on the BASELINE robots under CUDA-graph replay):
  //  * small batches (B <= step_fork_max_b(model): 3072, 128 x SMs or 256 x SMs, see specialize.cu): one operator's grid does not
  //    fill the machine (B = 4096: 128 tiles on 148 SMs) and the four operators are independent given (q, qd, qdd), so
  //    they are FORKED over three side streams and joined: the step costs about its longest operator, each operator
  //    running its own best small-batch kernel (a fused straight-line kernel is one long dependent instruction stream
  //    there: quadruped at 4096: 25.9 us fused, 7.4 us for its longest operator; humanoid at 32 768: 50 us forked, 77 us
  //    in sequence);
  //  * above: ONE launch where the model has a one-launch kernel that pays at this batch (fused / side by side), or TWO
  //    (kinematics-fused kernel + RNEA on a side stream: humanoid at 65 536: 94.8 us against 103.8 us as four launches),
  //    else the four operators in sequence on the caller's stream.
  // step_mode forces a form (tests, experiments).
  const int64_t mode = bm->m.opt.step_mode;
  cudaStreamCaptureStatus capture = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing((cudaStream_t)stream, &capture) != cudaSuccess) { cudaGetLastError(); capture = cudaStreamCaptureStatusNone; }
  const int64_t fork_max_b = bard::step_fork_max_b(bm->m, capture == cudaStreamCaptureStatusActive);
  StepFork& f = const_cast<bard_model*>(bm)->fj;
  const bool want_fork = mode == 1 || (mode < 0 && B <= fork_max_b);
  if (bm->m.nv > 0 && bm->m.nframes > 0 && (mode == 2 || (mode < 0 && !want_fork))) {
    // a one-launch kernel needs all four outputs to exist
    bard_status s = check_call("bard_step", bm, B, q, qd, qdd, tau);
    if (s == BARD_OK) s = check_call("bard_step", bm, B, pose, J, M, M);
    if (s != BARD_OK || B == 0) return s;
    if (bard::launch_specialized(bm->m, BARD_OP_STEP, B, q, qd, qdd, pose, J, tau, M, stream, s)) return s;
    // no full fused kernel for this robot / batch: kinematics-fused kernel + RNEA.  RNEA goes to a side stream when the
    // fork plumbing exists (it is ALU-bound, the kinematics kernel HBM-bound: they overlap), else after it on `stream`.
    if ((mode < 0 || mode == 2) && bard::kin_available(bm->m, B)) {
      const bool side = f.ok && bm->m.opt.step_kin_fork != 0;
      cudaStream_t user = (cudaStream_t)stream;
      std::unique_lock<std::mutex> lock(f.mu, std::defer_lock);
      bool forked = false;
      if (side) {
        lock.lock();
        forked = cudaEventRecord(f.fork, user) == cudaSuccess && cudaStreamWaitEvent(f.side[1], f.fork, 0) == cudaSuccess;
        if (!forked) cudaGetLastError();
      }
      bard_status sr = BARD_OK;
      bard::launching_side_by_side() = forked;
      if (forked) sr = bard_rnea(bm, B, q, qd, qdd, tau, f.side[1]);      // first: it is short and fills the machine's ALUs early
      const bool kin_ok = bard::launch_kin(bm->m, B, q, pose, J, M, stream, s);
      bard::launching_side_by_side() = false;
      if (kin_ok) {
        if (!forked) sr = bard_rnea(bm, B, q, qd, qdd, tau, stream);
        else if (cudaEventRecord(f.join[1], f.side[1]) != cudaSuccess || cudaStreamWaitEvent(user, f.join[1], 0) != cudaSuccess) {
          set_error(std::string("bard_step: fork-join: ") + cudaGetErrorString(cudaGetLastError()));
          return BARD_ERR_CUDA;
        }
        return s != BARD_OK ? s : sr;
      }
      if (forked) {                                             // no kinematics kernel after all: join and run the rest in sequence
        if (cudaEventRecord(f.join[1], f.side[1]) != cudaSuccess || cudaStreamWaitEvent(user, f.join[1], 0) != cudaSuccess) {
          set_error(std::string("bard_step: fork-join: ") + cudaGetErrorString(cudaGetLastError()));
          return BARD_ERR_CUDA;
        }
        lock.unlock();
        bard_status t = bard_fk(bm, B, q, pose, stream);
        if (t == BARD_OK) t = bard_jacobian(bm, B, q, J, stream);
        if (t == BARD_OK) t = bard_crba(bm, B, q, M, stream);
        return t != BARD_OK ? t : sr;
      }
    }
  }
  if (f.ok && B > 0 && want_fork && bm->m.nv > 0) {
    // Works under stream capture (the side streams join the capture).  One fork-join is enqueued at a time: the events
    // are re-recorded by every call (a wait captures the event's state at the time of the call, so that is safe).
    std::lock_guard<std::mutex> lock(f.mu);
    cudaStream_t user = (cudaStream_t)stream;
    bool ok = cudaEventRecord(f.fork, user) == cudaSuccess;
    for (int k = 0; k < 3 && ok; ++k) ok = cudaStreamWaitEvent(f.side[k], f.fork, 0) == cudaSuccess;
    if (ok) {
      bard::launching_side_by_side() = true;                    // the four grids are meant to share the SMs
      bard_status s = bard_crba(bm, B, q, M, stream);           // the longest operator stays on the caller's stream
      bard_status s1 = bard_jacobian(bm, B, q, J, f.side[0]);
      bard_status s2 = bard_rnea(bm, B, q, qd, qdd, tau, f.side[1]);
      bard_status s3 = bard_fk(bm, B, q, pose, f.side[2]);
      bard::launching_side_by_side() = false;
      for (int k = 0; k < 3; ++k)                               // always join, whatever the launches returned
        if (cudaEventRecord(f.join[k], f.side[k]) != cudaSuccess || cudaStreamWaitEvent(user, f.join[k], 0) != cudaSuccess) ok = false;
      if (!ok) { set_error(std::string("bard_step: fork-join: ") + cudaGetErrorString(cudaGetLastError())); return BARD_ERR_CUDA; }
      return s != BARD_OK ? s : s1 != BARD_OK ? s1 : s2 != BARD_OK ? s2 : s3;
    }
    cudaGetLastError();                                         // could not fork: fall through to the plain sequence
  }
  bard_status s = bard_fk(bm, B, q, pose, stream);
  if (s == BARD_OK) s = bard_jacobian(bm, B, q, J, stream);
  if (s == BARD_OK) s = bard_rnea(bm, B, q, qd, qdd, tau, stream);
  if (s == BARD_OK) s = bard_crba(bm, B, q, M, stream);
  return s;
}

bard_status bard_euler_step(const bard_model* bm, int64_t B, float dt, float* q, float* qd, const float* qdd, bard_stream stream) {
  if (!bm) { set_error("bard_euler_step: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (bm->m.nq == 0) return check_call("bard_euler_step", bm, B, bm, bm, bm, bm);   // nothing to integrate
  bard_status s = check_call("bard_euler_step", bm, B, q, bm->m.nv ? (const void*)qd : q, bm->m.nv ? (const void*)qdd : q, q);
  if (s != BARD_OK || B == 0) return s;
  bard::DeviceGuard guard(bm->m.device);
  return bard::launch_euler(bm->m, B, dt, q, qd, qdd, q, qd, stream);
}

bard_status bard_euler_step_to(const bard_model* bm, int64_t B, float dt, const float* q, const float* qd, const float* qdd, float* q_out,
                               float* qd_out, bard_stream stream) {
  if (!bm) { set_error("bard_euler_step_to: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (bm->m.nq == 0) return check_call("bard_euler_step_to", bm, B, bm, bm, bm, bm);
  bard_status s = check_call("bard_euler_step_to", bm, B, q, bm->m.nv ? (const void*)qd : q, bm->m.nv ? (const void*)qdd : q, q_out);
  if (s == BARD_OK && B > 0 && bm->m.nv && !qd_out) { set_error("bard_euler_step_to: NULL device pointer"); s = BARD_ERR_INVALID_ARG; }
  if (s != BARD_OK || B == 0) return s;
  bard::DeviceGuard guard(bm->m.device);
  return bard::launch_euler(bm->m, B, dt, q, qd, qdd, q_out, qd_out, stream);
}

size_t bard_aba_workspace_floats(const bard_model* bm, int64_t B) {
  if (!bm || B <= 0) return 0;
  return bard::aba_is_specialized(bm->m) ? (size_t)10 * (size_t)bm->m.nv * (size_t)B : bard::aba_generic_workspace_floats(bm->m, B);
}

bard_status bard_aba(const bard_model* bm, int64_t B, const float* q, const float* qd, const float* tau, float* qdd, float* workspace,
                     bard_stream stream) {
  if (bm && bm->m.nv == 0) return check_call("bard_aba", bm, B, bm, bm, bm, bm);  // nothing to write
  bard_status s = check_call("bard_aba", bm, B, q, qd, tau, qdd);
  if (s == BARD_OK && B > 0 && !workspace) { set_error("bard_aba: workspace is NULL"); s = BARD_ERR_INVALID_ARG; }
  if (s != BARD_OK || B == 0) return s;
  bard::DeviceGuard guard(bm->m.device);
  return bard::launch_aba(bm->m, B, q, qd, tau, qdd, workspace, stream);
}

bard_status bard_model_specialize_variant(bard_model* bm, uint32_t ops, int dtype, int layout) {
  if (!bm) { set_error("bard_model_specialize_variant: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (dtype < 0 || dtype > 1 || layout < 0 || layout > 1) { set_error("bard_model_specialize_variant: unknown dtype / layout"); return BARD_ERR_INVALID_ARG; }
  if (ops & ~(uint32_t)BARD_OP_STEP) { set_error("bard_model_specialize_variant: only BARD_OP_FK / JACOBIAN / RNEA / CRBA have variants"); return BARD_ERR_INVALID_ARG; }
  // the layout needs no code of its own (transposes around the SoA kernels); fp32 variants are the plain kernels
  return dtype == BARD_F64 ? bard::specialize_f64(bm->m, ops) : bard::specialize(bm->m, ops);
}

bard_status bard_model_variant_source(const bard_model* bm, uint32_t op, int dtype, int layout, char* host_dst, size_t cap, size_t* need) {
  if (!bm) { set_error("bard_model_variant_source: model is NULL"); return BARD_ERR_INVALID_ARG; }
  (void)layout;
  const std::string* src = dtype == BARD_F64 ? bard::f64_source(bm->m, op) : bard::specialized_source(bm->m, op);
  if (!src) { set_error("bard_model_variant_source: operator variant not specialised"); return BARD_ERR_INVALID_ARG; }
  if (need) *need = src->size() + 1;
  if (cap < src->size() + 1 || !host_dst) { set_error("bard_model_variant_source: destination too small"); return BARD_ERR_INVALID_ARG; }
  std::memcpy(host_dst, src->c_str(), src->size() + 1);
  return BARD_OK;
}

static int64_t out_rows(const bard::Model& m, uint32_t op) {
  return op == BARD_OP_FK ? 12 * (int64_t)m.nb : op == BARD_OP_JACOBIAN ? 6 * (int64_t)m.nframes * m.nv : op == BARD_OP_RNEA ? m.nv : (int64_t)m.nv * m.nv;
}

size_t bard_variant_workspace_bytes(const bard_model* bm, uint32_t op, int dtype, int layout, int64_t B) {
  if (!bm || B <= 0 || layout != BARD_LAYOUT_AOS) return 0;
  const bard::Model& m = bm->m;
  const int64_t in_rows = m.nq + (op == BARD_OP_RNEA ? 2 * (int64_t)m.nv : 0);
  return (size_t)(in_rows + out_rows(m, op)) * (size_t)B * (dtype == BARD_F64 ? 8 : 4) + 64;
}

// the _v calls: dtype / layout variants of the four operators.  (F32, SoA) is the plain call.
static bard_status variant_call(const char* fn, const bard_model* bm, uint32_t op, int dtype, int layout, int64_t B, const void* q,
                                const void* qd, const void* qdd, void* out, void* workspace, bard_stream stream) {
  if (!bm) { set_error(std::string(fn) + ": model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (dtype < 0 || dtype > 1 || layout < 0 || layout > 1) { set_error(std::string(fn) + ": unknown dtype / layout"); return BARD_ERR_INVALID_ARG; }
  const bard::Model& m = bm->m;
  const bool empty = (op != BARD_OP_FK && m.nv == 0) || (op == BARD_OP_JACOBIAN && m.nframes == 0);
  const void* dummy = bm;
  bard_status s = check_call(fn, bm, B, (m.nq == 0 || empty) ? dummy : q, (op == BARD_OP_RNEA && !empty) ? qd : dummy,
                             (op == BARD_OP_RNEA && !empty) ? qdd : dummy, empty ? dummy : (const void*)out);
  if (s != BARD_OK || B == 0 || empty) return s;
  bard::DeviceGuard guard(m.device);
  const int es = dtype == BARD_F64 ? 8 : 4;
  const void *sq = q, *sqd = qd, *sqdd = qdd;
  void* sout = out;
  if (layout == BARD_LAYOUT_AOS) {
    // (B, n) -> [n][B] into the workspace, the SoA operator, [rows][B] -> (B, rows) into the caller's output
    if (!workspace) { set_error(std::string(fn) + ": the AoS layout needs a workspace of bard_variant_workspace_bytes()"); return BARD_ERR_INVALID_ARG; }
    char* w = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(workspace) + 15) & ~(uintptr_t)15);
    auto take = [&](int64_t rows) { void* p = w; w += (size_t)rows * (size_t)B * es; return p; };
    if (m.nq > 0) { void* p = take(m.nq); s = bard::launch_transpose(q, p, B, m.nq, es, stream); sq = p; }
    if (op == BARD_OP_RNEA) {
      void* p = take(m.nv);
      if (s == BARD_OK) s = bard::launch_transpose(qd, p, B, m.nv, es, stream);
      sqd = p;
      p = take(m.nv);
      if (s == BARD_OK) s = bard::launch_transpose(qdd, p, B, m.nv, es, stream);
      sqdd = p;
    }
    if (s != BARD_OK) return s;
    sout = take(out_rows(m, op));
  }
  if (dtype == BARD_F64) {
    s = bard::launch_f64(m, op, B, sq, sqd, sqdd, op == BARD_OP_FK ? sout : nullptr, op == BARD_OP_JACOBIAN ? sout : nullptr,
                         op == BARD_OP_RNEA ? sout : nullptr, op == BARD_OP_CRBA ? sout : nullptr, stream);
  } else {
    s = op == BARD_OP_FK ? bard_fk(bm, B, (const float*)sq, (float*)sout, stream)
        : op == BARD_OP_JACOBIAN ? bard_jacobian(bm, B, (const float*)sq, (float*)sout, stream)
        : op == BARD_OP_RNEA ? bard_rnea(bm, B, (const float*)sq, (const float*)sqd, (const float*)sqdd, (float*)sout, stream)
                             : bard_crba(bm, B, (const float*)sq, (float*)sout, stream);
  }
  if (s == BARD_OK && layout == BARD_LAYOUT_AOS) s = bard::launch_transpose(sout, out, out_rows(m, op), B, es, stream);
  return s;
}

bard_status bard_fk_v(const bard_model* bm, int dtype, int layout, int64_t B, const void* q, void* pose, void* workspace, bard_stream stream) {
  return variant_call("bard_fk_v", bm, BARD_OP_FK, dtype, layout, B, q, nullptr, nullptr, pose, workspace, stream);
}
bard_status bard_jacobian_v(const bard_model* bm, int dtype, int layout, int64_t B, const void* q, void* J, void* workspace, bard_stream stream) {
  return variant_call("bard_jacobian_v", bm, BARD_OP_JACOBIAN, dtype, layout, B, q, nullptr, nullptr, J, workspace, stream);
}
bard_status bard_rnea_v(const bard_model* bm, int dtype, int layout, int64_t B, const void* q, const void* qd, const void* qdd, void* tau,
                        void* workspace, bard_stream stream) {
  return variant_call("bard_rnea_v", bm, BARD_OP_RNEA, dtype, layout, B, q, qd, qdd, tau, workspace, stream);
}
bard_status bard_crba_v(const bard_model* bm, int dtype, int layout, int64_t B, const void* q, void* M, void* workspace, bard_stream stream) {
  return variant_call("bard_crba_v", bm, BARD_OP_CRBA, dtype, layout, B, q, nullptr, nullptr, M, workspace, stream);
}

size_t bard_rnea_vjp_workspace_floats(const bard_model* bm, int64_t B) {
  return (bm && B > 0) ? bard::rnea_vjp_workspace_floats(bm->m, B) : 0;
}

bard_status bard_rnea_vjp_params(const bard_model* bm, int64_t B, const float* q, const float* qd, const float* qdd, const float* dtau,
                                 float* dparams, float* workspace, bard_stream stream) {
  if (!bm) { set_error("bard_rnea_vjp_params: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (!dparams) { set_error("bard_rnea_vjp_params: dparams is NULL"); return BARD_ERR_INVALID_ARG; }
  bard_status s = check_call("bard_rnea_vjp_params", bm, B, bm->m.nq ? (const void*)q : dparams, bm->m.nv ? (const void*)qd : dparams,
                             bm->m.nv ? (const void*)qdd : dparams, bm->m.nv ? (const void*)dtau : dparams);
  if (s == BARD_OK && B > 0 && !workspace) { set_error("bard_rnea_vjp_params: workspace is NULL"); s = BARD_ERR_INVALID_ARG; }
  if (s != BARD_OK) return s;
  bard::DeviceGuard guard(bm->m.device);
  if (B == 0) {                                             // the sum over no environments
    cudaError_t e = cudaMemsetAsync(dparams, 0, sizeof(float) * 10 * (size_t)bm->m.nb, (cudaStream_t)stream);
    if (e != cudaSuccess) { set_error(std::string("bard_rnea_vjp_params: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
    return BARD_OK;
  }
  return bard::launch_rnea_vjp(bm->m, B, q, qd, qdd, dtau, dparams, workspace, stream);
}

bard_status bard_rnea_vjp_params_static(const bard_model* bm, int64_t B, const float* q, const float* qd, const float* qdd, const float* dtau,
                                        float* dparams, bard_stream stream) {
  if (!bm) { set_error("bard_rnea_vjp_params_static: model is NULL"); return BARD_ERR_INVALID_ARG; }
  if (!dparams) { set_error("bard_rnea_vjp_params_static: dparams is NULL"); return BARD_ERR_INVALID_ARG; }
  bard_status s = check_call("bard_rnea_vjp_params_static", bm, B, bm->m.nq ? (const void*)q : dparams, bm->m.nv ? (const void*)qd : dparams,
                             bm->m.nv ? (const void*)qdd : dparams, bm->m.nv ? (const void*)dtau : dparams);
  if (s != BARD_OK) return s;
  bard::DeviceGuard guard(bm->m.device);
  if (B == 0) {                                             // the sum over no environments
    cudaError_t e = cudaMemsetAsync(dparams, 0, sizeof(float) * 10 * (size_t)bm->m.nb, (cudaStream_t)stream);
    if (e != cudaSuccess) { set_error(std::string("bard_rnea_vjp_params_static: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
    return BARD_OK;
  }
  return bard::launch_rnea_vjp_static(bm->m, B, q, qd, qdd, dtau, dparams, stream);
}

bard_status bard_model_inertial_params(const bard_model* bm, double* host_params) {
  if (!bm || !host_params) { set_error("bard_model_inertial_params: NULL argument"); return BARD_ERR_INVALID_ARG; }
  for (int i = 0; i < bm->m.nb; ++i)
    for (int k = 0; k < 10; ++k) host_params[10 * i + k] = bm->m.bc64[(size_t)bard::kBc64 * i + 42 + k];
  return BARD_OK;
}

bard_status bard_model_set_inertial_params(bard_model* bm, const double* host_params) {
  if (!bm || !host_params) { set_error("bard_model_set_inertial_params: NULL argument"); return BARD_ERR_INVALID_ARG; }
  bard::Model& m = bm->m;
  for (int k = 0; k < 10 * m.nb; ++k)
    if (!(host_params[k] == host_params[k])) { set_error("bard_model_set_inertial_params: NaN parameter"); return BARD_ERR_INVALID_ARG; }
  bard::DeviceGuard guard(m.device);
  if (m.d_blob) {                                            // as bard_model_set_frames: nothing that reads the tables may be in flight
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { set_error(std::string("bard_model_set_inertial_params: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
  }
  bard::drop_specialized_dynamics(m);
  bard::BodyConst* BC = reinterpret_cast<bard::BodyConst*>(m.blob.data() + sizeof(bard::BlobHeader));
  for (int i = 0; i < m.nb; ++i) {
    const double* th = host_params + 10 * i;
    double* c64 = &m.bc64[(size_t)bard::kBc64 * i];
    for (int k = 0; k < 10; ++k) c64[42 + k] = th[k];
    BC[i].mass = (float)th[0];
    for (int k = 0; k < 3; ++k) BC[i].h[k] = (float)th[1 + k];
    for (int k = 0; k < 6; ++k) BC[i].Io[k] = (float)th[4 + k];
  }
  if (m.d_blob) {
    const size_t bytes = sizeof(bard::BlobHeader) + sizeof(bard::BodyConst) * (size_t)m.nb;
    cudaError_t e = cudaMemcpy(m.d_blob, m.blob.data(), bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { set_error(std::string("bard_model_set_inertial_params: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
  }
  return BARD_OK;
}

const char* bard_status_string(bard_status s) {
  switch (s) {
    case BARD_OK: return "BARD_OK";
    case BARD_ERR_INVALID_ARG: return "BARD_ERR_INVALID_ARG";
    case BARD_ERR_TOPOLOGY: return "BARD_ERR_TOPOLOGY";
    case BARD_ERR_UNSUPPORTED: return "BARD_ERR_UNSUPPORTED";
    case BARD_ERR_ALLOC: return "BARD_ERR_ALLOC";
    case BARD_ERR_CUDA: return "BARD_ERR_CUDA";
  }
  return "BARD_ERR_UNKNOWN";
}

const char* bard_last_error(void) { return bard::g_err.c_str(); }

int64_t bard_launch_count(void) { return bard::g_launches.load(); }

}  // extern "C"
