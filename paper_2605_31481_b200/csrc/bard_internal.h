// Internal definitions shared by the model builder (model.cu), the kernels (kernels.cu) and the C ABI
// (api.cu).  Nothing here is used by oracle/.
#pragma once
#include <algorithm>
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
  int32_t src;                // 56  where the parent's state is: -1 world, -2 registers of the same warp
                              //     (the task this warp processed just before), >=0 shared-memory slot
  int32_t save;               // 57  slot this body's state is saved to for children on other warps (-1: none)
  int32_t flags;              // 58  bit0: T_post is identity (a = b = 0, Sl = 0); bits 8..15: index among free-joint bodies
  int32_t level;              // 59
  uint32_t anc_lo, anc_hi;    // 60, 61  ancestor-or-self mask of this body
  int32_t child_begin;        // 62  first entry of this body's children in the CHILDREN table
  int32_t child_count;        // 63
};
static_assert(sizeof(BodyConst) == 256, "BodyConst must be 64 words");

struct FrameConst {           // 8 words
  int32_t body;
  float   off[3];
  uint32_t anc_lo, anc_hi;    // ancestor-or-self mask of the frame's body
  int32_t pad[2];
};

// Level-parallel schedule (eq. (6)): one TEAM of `team_warps` warps evaluates 32
// environments (lane = environment).  Bodies of one tree level are spread over the team's warps; the warps
// meet at a named barrier between levels.  Every warp walks its own flat task list
//   task = body | TASK_BAR (team barrier after this task) | TASK_NOOP (no body: barrier only)
// terminated by TASK_END; the inward sweeps of RNEA / CRBA walk the same list backwards.
enum : uint16_t { TASK_BODY_MASK = 0x00ff, TASK_BAR = 0x0100, TASK_NOOP = 0x0200, TASK_END = 0xffff };

// Device constants come in three sections, each a multiple of 16 bytes so that it can be staged into shared
// memory with one TMA bulk copy:
//   COMMON  BlobHeader | BodyConst[nb] | tasks | children          (all four operators)
//   M       MHeader | fill lists | rel masks | zero rows           (CRBA only; directly after COMMON)
//   J       JHeader | FrameConst[16] | columns | zero rows         (Jacobian only; own buffer, rewritten by
//                                                                   bard_model_set_frames)
struct BlobHeader {           // 16 words
  int32_t nb, nq, nv, nlevels;
  int32_t nslots;             // number of parent-state slots the outward sweeps need
  int32_t team_warps;         // L
  int32_t off_tasks;          // uint16 [team_warps][task_stride]   (byte offsets from the start of COMMON)
  int32_t task_stride;
  float   g[3];               // gravity, world
  int32_t off_children;       // uint8 [nb]: children lists, ascending, concatenated in body order
  int32_t off_dof_body;       // uint8 [nv]
  int32_t simple;             // 1: every joint is REVOLUTE with T_post = I, or FREE
  int32_t pad[2];
};
static_assert(sizeof(BlobHeader) == 64, "BlobHeader must be 16 words");

struct MHeader {              // 12 words; byte offsets from the start of the M section
  int32_t off_fill;           // uint8 [team_warps][fill_stride]: rows of M each warp fills, 0xff ends
  int32_t fill_stride;
  int32_t off_rel;            // uint64 [nv]: bit j set <=> j <= i and DOF j sits on an ancestor-or-self body of DOF i
  int32_t off_zrows;          // uint16 [nzrows]: flat indices i*nv+j of the structurally zero entries (both triangles)
  int32_t nzrows;             // padded to a multiple of 4 with 0xffff
  int32_t off_pairs;          // uint8: for row i the DOFs j <= i with M[i][j] != 0, EXCEPT the DOFs of free-joint
                              //        bodies that are proper ancestors of row i's body (those go through fanc)
  int32_t off_pair_ptr;       // uint16 [nv + 1]: row i's pairs are pairs[pair_ptr[i] .. pair_ptr[i+1])
  int32_t off_fanc;           // uint8: for row i the free-joint bodies that are proper ancestors of its body
  int32_t off_fanc_ptr;       // uint16 [nv + 1]
  int32_t pad[3];
};
struct JHeader {              // 8 words; byte offsets from the start of the J section
  int32_t nframes;
  uint32_t jmask_lo, jmask_hi;  // union of the frames' ancestor masks: bodies the Jacobian FK must visit
  int32_t off_cols;           // uint16 [ncols]: (frame << 8 | dof) of the non-zero columns
  int32_t ncols;
  int32_t off_zrows;          // uint16 [nzrows]: flat row indices (f*6+r)*nv+j of the zero rows, padded with 0xffff
  int32_t nzrows;
  int32_t off_bframes;        // uint16 [nb]: bit f set <=> frame f is attached to this body
};

struct Specialized;           // specialize.cu: model-specialised (NVRTC) kernels

// Launch and code-generation knobs.  Every one is a field of the MODEL: bard_model_create reads its default from the
// environment variable BARD_<KEY IN UPPER CASE> once, bard_model_set_option overrides it afterwards; no operator
// call reads the environment.  -1 = "auto" (the measured rule documented next to the knob's use).
#define BARD_OPTIONS(X)                                                                                        \
  /* team kernels (kernels.cu) */                                                                              \
  X(teams, 0)            /* tiles per CTA (0 = auto) */                                                        \
  X(pack, 0)             /* force N environments per lane (1 / 2; 0 = auto) */                                 \
  X(pack2_min_b, 32768)  /* smallest batch that runs two environments per lane */                              \
  X(pdl, 1)              /* programmatic dependent launch attribute on every launch */                         \
  /* which kernel family a call gets (specialize.cu, api.cu) */                                                \
  X(spec_min_b, -1)            /* smallest batch for the plain specialised kernels */                          \
  X(spec_block, 0)             /* force the CTA size of the specialised kernels */                             \
  X(spec_min_block, -1)        /* smallest CTA of a one-wave launch of the compute-bound generated kernels (-1: per kernel, 256 / 128; 0: off) */ \
  X(spec_roles_max_b, -1)      /* largest batch for the limb-role RNEA */                                      \
  X(spec_crba_roles_max_b, -1) /* largest / smallest batch for the limb-role CRBA */                           \
  X(spec_crba_roles_min_b, -1)                                                                                 \
  X(spec_fused_max_rows, 112)  /* the fused step kernel is used at every batch up to this many parked rows */  \
  X(spec_fused_small_b, -1)    /* ... and above it only up to this batch */                                    \
  X(spec_kin_min_b, -1)        /* smallest batch at which bard_step uses the kinematics-fused kernel + RNEA */ \
  X(step_fork_max_b, -1)       /* bard_step forks the four operators over side streams up to this batch (auto: step_fork_max_b() in specialize.cu) */ \
  X(step_light_max, 2000)      /* ... not measured: a one-/two-launch step of at most this many arithmetic statements per thread takes over from 3072 environments */ \
  X(step_calibrate, 1)         /* bard_model_specialize(BARD_OP_FUSED) times the forked and the one-/two-launch step at B = 4096 and sets the fork regime from that */ \
  X(step_kin_fork, 1)          /* bard_step = kinematics-fused kernel + RNEA: RNEA on a side stream (1) or after it (0) */ \
  X(step_mode, -1)             /* bard_step: -1 auto, 0 four launches in sequence, 1 forked, 2 one-launch kernel */ \
  /* read by bard_model_specialize (code generation) */                                                        \
  X(spec_prefetch, 2)          /* bodies of input-load lookahead */                                            \
  X(spec_prefetch_rnea, 3)     /* ... of the generated RNEA kernel */                                          \
  X(spec_sync, -1)             /* bodies between CTA barriers (0 = none) */                                    \
  X(spec_l2pf, -1)             /* up-front L2 prefetch: 0 never, 1 always, 2 two kernels */                    \
  X(spec_roles, 2)             /* limb roles */                                                                \
  X(spec_zero_role, 1)         /* CRBA limb roles: a group of warps that only stores M's structural zeros */   \
  X(spec_maxreg, 0)            /* --maxrregcount of the NVRTC compile (0 = none) */                            \
  X(spec_step4, 1)             /* build the side-by-side step kernel */                                        \
  X(spec_step4_max_rows, 72)                                                                                   \
  X(spec_ldnc, 1)              /* non-coherent (ld.global.nc) input loads in the generated kernels; 0 = coherent */ \
  X(spec_max_block, 512)       /* __launch_bounds__ of the generated kernels (448: 144 registers instead of 128) */ \
  X(spec_solo_smem, 1)         /* one-wave launches ask for > half of the shared memory: one CTA per SM also under PDL */ \
  X(spec_vjp_min_b, -1)        /* smallest batch for the generated RNEA VJP kernel (auto: 0) */                \
  X(spec_kin, 1)               /* build the kinematics-fused kernel (FK + Jacobian + CRBA) with BARD_OP_FUSED */ \
  X(spec_classical, 1)         /* RNEA of simple models in the classical Newton-Euler form about the COM (fewer FLOPs) */ \
  X(spec_pack, 1)              /* RNEA: 2 = also build the kernel with two environments per thread (FFMA2); it loses: off */ \
  X(spec_pack_min_b, -1)       /* ... and the batch range it is launched in */                                  \
  X(spec_pack_max_b, -1)
struct Options {
#define BARD_OPT_FIELD(name, dflt) int64_t name = dflt;
  BARD_OPTIONS(BARD_OPT_FIELD)
#undef BARD_OPT_FIELD
};
void options_from_env(Options& o);
bool option_ref(Options& o, const char* key, int64_t** ref);

struct Model {
  int device = 0;
  Options opt;
  Specialized* spec = nullptr;
  int64_t fork_max_cal[2] = {-1, -1}; // bard_step's fork regime as bard_model_specialize measured it (-1: not measured): [0] plain calls, [1] under stream capture
  int32_t nb = 0, nq = 0, nv = 0, nlevels = 0, nslots = 0, nframes = 0, nfree = 0;
  int32_t team_warps = 1;             // L: warps that share one 32-environment tile (level-parallel schedule)
  int32_t crba_warps = 1;             // Lc >= L: CRBA adds warps that only join the fill of M
  bool simple = false;
  std::vector<int32_t> warp_of;       // body -> warp of its team
  std::vector<int32_t> free_index;    // body -> index among free-joint bodies (-1 otherwise)
  std::vector<int32_t> parent, jtype, level_ptr, level_body, body_level, parent_slot, q_off, v_off, dof_body;
  std::vector<uint64_t> anc_mask;
  std::vector<float> rodrigues;       // nb*36
  std::vector<unsigned char> blob;    // host copy of COMMON + M
  std::vector<unsigned char> jblob;   // host copy of J
  void* d_blob = nullptr;             // COMMON + M
  void* d_jblob = nullptr;            // J (allocated for the largest frame set)
  size_t common_bytes = 0, m_bytes = 0, j_bytes = 0;
  int sm_count = 148;
  // where rnea_kernel parks the staged input rows (shared-memory row of q / qd / qdd row r); built once with the model
  uint16_t rowmap_q[128] = {}, rowmap_qd[64] = {}, rowmap_qdd[64] = {};
  // fp64 copy of the per-body constants (the fp32 BodyConst rows are these, rounded once): R0 A B t0 a b (36),
  // Sw Sl (6), mass, h (3), Io (6) = 52 doubles per body; gravity.  Read by the fp64 code generator.
  std::vector<double> bc64;
  double g64[3] = {0, 0, 0};
  std::vector<double> frame_off64;    // nframes * 3
};
constexpr int kBc64 = 52;

// Makes the model's device current for the duration of a call (and restores the caller's): one cudaGetDevice, and a
// cudaSetDevice only when a process drives several GPUs and the caller's current device is another one.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device);
  ~DeviceGuard();
};

constexpr size_t kJBlobMax = sizeof(JHeader) + sizeof(FrameConst) * BARD_MAX_FRAMES +
                             2 * (size_t)BARD_MAX_FRAMES * BARD_MAX_DOF + 2 * 6 * (size_t)BARD_MAX_FRAMES * BARD_MAX_DOF +
                             2 * (size_t)BARD_MAX_BODIES + 96;

void set_error(const std::string& s);
// Set (per host thread) by bard_step while it enqueues operators that are meant to run SIDE BY SIDE on several streams:
// their launches must not ask for the shared memory that keeps an SM to one CTA (see solo_smem).
bool& launching_side_by_side();
// A launch whose grid fits one CTA per SM asks for more than half of the SM's shared memory, so that the plan (one CTA per
// SM) also holds under programmatic dependent launch, where the next grid's CTAs are dispatched as resources free up:
// where two CTAs fit an SM, the first SMs to finish take two of the next grid's CTAs and the last ones none (measured on
// back-to-back trains: humanoid FK at B = 65 536 13 -> 23 us, quadruped Jacobian 18.8 -> 26.8 us, team CRBA at 4096 10.9 -> 15.2 us).
inline size_t solo_smem(const Model& m, unsigned grid, size_t smem) {
  return (grid <= (unsigned)m.sm_count && m.opt.spec_solo_smem && !launching_side_by_side()) ? std::max<size_t>(smem, 116 * 1024) : smem;
}

// kernels.cu
bard_status launch_fk(const Model& m, int64_t B, const float* q, float* pose, void* stream);
bard_status launch_jacobian(const Model& m, int64_t B, const float* q, float* J, void* stream);
bard_status launch_rnea(const Model& m, int64_t B, const float* q, const float* qd, const float* qdd, float* tau,
                        void* stream);
bard_status launch_crba(const Model& m, int64_t B, const float* q, float* M, void* stream);
bard_status launch_euler(const Model& m, int64_t B, float dt, const float* q, const float* qd, const float* qdd, float* q_out, float* qd_out,
                         void* stream);


// specialize.cu
bard_status specialize(Model& M, uint32_t ops);
void free_specialized(Specialized* s);
const std::string* specialized_source(const Model& M, uint32_t op);
bool launch_specialized(const Model& M, uint32_t op, int64_t B, const float* q, const float* qd, const float* qdd, float* pose,
                        float* J, float* tau, float* Mo, void* stream, bard_status& st);
bard_status specialize_f64(Model& M, uint32_t ops);
const std::string* f64_source(const Model& M, uint32_t op);
bard_status launch_f64(const Model& M, uint32_t op, int64_t B, const void* q, const void* qd, const void* qdd, void* pose, void* J,
                       void* tau, void* Mo, void* stream);

// layout.cu: [rows][cols] -> [cols][rows] at HBM speed (elem = 4 or 8 bytes), one launch
bard_status launch_transpose(const void* src, void* dst, int64_t rows, int64_t cols, int elem, void* stream);
bool kin_available(const Model& M, int64_t B);
int64_t step_fork_max_b(const Model& M, bool capturing);
bool launch_kin(const Model& M, int64_t B, const float* q, float* pose, float* J, float* Mo, void* stream, bard_status& st);
void drop_specialized_jacobian(Model& M);
void drop_specialized_dynamics(Model& M);      // kernels with the inertial parameters folded in as literals

// aba_generic.cu: the table-driven ABA (no NVRTC; a free joint anywhere)
size_t aba_generic_workspace_floats(const Model& M, int64_t B);
bard_status launch_aba_generic(const Model& M, int64_t B, const float* q, const float* qd, const float* tau, float* qdd, float* ws, void* stream);
bool aba_is_specialized(const Model& M);

// vjp.cu
size_t rnea_vjp_workspace_floats(const Model& M, int64_t B);
bard_status launch_rnea_vjp(const Model& M, int64_t B, const float* q, const float* qd, const float* qdd, const float* dtau,
                            float* dparams, float* ws, void* stream);
bard_status launch_aba(const Model& M, int64_t B, const float* q, const float* qd, const float* tau, float* qdd, float* ws, void* stream);
// the generated VJP kernel (specialize.cu) and the sum over its CTAs' columns, partials[np][ncta] (vjp.cu)
bool launch_vjp_specialized(const Model& M, int64_t B, const float* q, const float* qd, const float* qdd, const float* dtau,
                            float* dparams, float* ws, void* stream, bard_status& st);
bard_status launch_vjp_reduce_columns(const float* partials, int ncta, int np, float* dparams, void* stream);
// vjp_static.cu: launch_rnea_vjp with the library's static scratch array (no allocation; one array per device, shared)
bard_status launch_rnea_vjp_static(const Model& M, int64_t B, const float* q, const float* qd, const float* qdd, const float* dtau,
                                   float* dparams, void* stream);

}  // namespace bard
