// Internal definitions shared by the model builder (model.cu), the kernels (kernels.cu) and the C ABI
// (api.cu).  Nothing here is used by oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/bard.h"

namespace bard {

// Per-body constants as the kernels read them (fp32, 64 words = 256 B, 16-byte aligned so the whole
// table can be staged into shared memory with one cp.async.bulk).
//
// Joint transform (eq. (4)-(5)), unified over joint types through two scalars
// (u, w):  R_pc = R0 + u*A + w*B ,  t_pc = t0 + u*a + w*b
//   revolute : u = sin q, w = 1 - cos q
//   prismatic: u = q,     w = 0   (A = B = 0, a = R_pre * axis, b = 0)        "analogously"
//   fixed    : u = w = 0
//   free     : R_pc = R0 * R(quat), t_pc = R0 * p + t0   (R0 = R_pre, t0 = t_pre)
struct BodyConst {
  float R0[9], A[9], Bm[9];   // 0..26
  float t0[3], a[3], b[3];    // 27..35   (words 0..35 = the RODRIGUES table row)
  float Sw[3], Sl[3];         // 36..41   body-frame motion subspace [angular; linear] (revolute/prismatic)
  float mass;                 // 42
  float h[3];                 // 43..45   m * com
  float Io[6];                // 46..51   rotational inertia about the BODY ORIGIN: xx,xy,xz,yy,yz,zz
  int32_t type;               // 52
  int32_t parent;             // 53
  int32_t q_off, v_off;       // 54, 55
  int32_t src;                // 56  where the parent's state is: -1 world, -2 the previous body (registers), >=0 slot
  int32_t save;               // 57  slot this body's state is saved to for later children (-1: none)
  int32_t flags;              // 58  bit0: T_post is identity (a = b = 0, Sl = 0)
  int32_t level;              // 59
  uint32_t anc_lo, anc_hi;    // 60, 61  ancestor-or-self mask of this body
  int32_t pad[2];             // 62, 63
};
static_assert(sizeof(BodyConst) == 256, "BodyConst must be 64 words");

struct FrameConst {           // 8 words
  int32_t body;
  float   off[3];
  uint32_t anc_lo, anc_hi;    // ancestor-or-self mask of the frame's body
  int32_t pad[2];
};

// Header of the device blob; followed by BodyConst[nb], then FrameConst[BARD_MAX_FRAMES].
struct BlobHeader {           // 16 words
  int32_t nb, nq, nv, nlevels;
  int32_t nslots;             // number of parent-state slots the outward sweeps need
  int32_t nframes;
  int32_t jac_mask_lo, jac_mask_hi;  // union of the frames' ancestor masks
  float   g[3];               // gravity, world
  int32_t pad[5];
};
static_assert(sizeof(BlobHeader) == 64, "BlobHeader must be 16 words");

struct Model {
  int device = 0;
  int32_t nb = 0, nq = 0, nv = 0, nlevels = 0, nslots = 0, nframes = 0;
  std::vector<int32_t> parent, jtype, level_ptr, level_body, body_level, parent_slot, q_off, v_off, dof_body;
  std::vector<uint64_t> anc_mask;
  std::vector<float> rodrigues;       // nb*36
  std::vector<unsigned char> blob;    // host copy of the device blob
  void* d_blob = nullptr;
  size_t blob_bytes = 0;
  int sm_count = 148;
};

void set_error(const std::string& s);

// kernels.cu
bard_status launch_fk(const Model& m, int64_t B, const float* q, float* pose, void* stream);
bard_status launch_jacobian(const Model& m, int64_t B, const float* q, float* J, void* stream);
bard_status launch_rnea(const Model& m, int64_t B, const float* q, const float* qd, const float* qdd, float* tau,
                        void* stream);
bard_status launch_crba(const Model& m, int64_t B, const float* q, float* M, void* stream);

}  // namespace bard
