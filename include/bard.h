/*
 * bard.h -- C ABI of the B200-native batched rigid-body operator library (libbard.so).
 *
 * Hot path of "Batched Differentiable Rigid Body Dynamics in PyTorch for GPU-Accelerated Robot
 * Learning" (arxiv 2605.31481, /root/reference/PAPER.md): forward kinematics, geometric Jacobians,
 * RNEA inverse dynamics and the CRBA mass matrix (operator list PAPER.md:37) for B independent
 * robot states per call.  The model is immutable and built once; every operator is
 * one asynchronous kernel launch on the caller's stream.
 *
 * Conventions (readings of the paper are listed in DESIGN.md "Readings"):
 *   - bodies i = 0..nb-1, one joint per body, parent[i] in {-1, 0..i-1}; -1 = world.
 *   - T_pc,i = T_pre,i * T_J(q_i) * T_post,i maps child to parent coordinates (eq. (1)).
 *   - joint types: revolute (nq=nv=1), prismatic (1,1), fixed (0,0), free (nq=7, nv=6).
 *     free joint: q = [p(3), quat x,y,z,w] (normalised inside the kernels), qd = body-frame twist
 *     [v_lin(3); omega(3)], qdd its component-wise derivative, tau = [force(3); moment(3)].
 *   - spatial order at the boundary is [linear; angular] (row order of eq. (7)).
 *   - DEVICE I/O LAYOUT: structure of arrays, batch fastest: component c of env b is ptr[c*B + b].
 *       q[nq][B]  qd[nv][B]  qdd[nv][B]           inputs,  fp32, device memory
 *       pose[nb][12][B]   c = 0..8 R row-major (body->world), 9..11 p (world)
 *       J[nframes][6][nv][B]  rows 0-2 linear, 3-5 angular; geometric Jacobian at the frame origin,
 *                             world axes (eq. (7) shifted to the frame origin)
 *       tau[nv][B]        M[nv][nv][B]  (full symmetric matrix, every element written once)
 *
 * Ownership: the caller owns every q/qd/qdd/output DEVICE buffer.  The library owns only the model
 * (host struct + one device constant blob), freed by bard_model_destroy.  Host arrays in
 * bard_model_desc are copied by bard_model_create.
 *
 * Execution: operator calls enqueue exactly one kernel on `stream`, allocate nothing and never
 * synchronise.  B == 0 returns BARD_OK without a launch.  Outputs are fully overwritten.
 * Devices: a model lives on the device given to bard_model_create; `stream` and every device pointer of
 * a call must belong to that device.  The calling thread's current device may be any: every call makes the
 * model's device current for its duration and restores the caller's.
 * Threads: operator calls on one model from several host threads / on several streams are legal (the
 * model is immutable between bard_model_create / set_frames / set_option / specialize calls).
 *
 * Errors: return codes only; bard_last_error() gives thread-local detail text.
 */
#ifndef BARD_H
#define BARD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bard_model bard_model;     /* opaque */
typedef void* bard_stream;                /* a cudaStream_t (NULL = default stream) */

typedef enum {
  BARD_OK = 0,
  BARD_ERR_INVALID_ARG = 1,   /* NULL pointer, negative B, nb < 1, bad joint type, zero axis, mass < 0,
                                 non-identity T_post on a free joint, bad frame body */
  BARD_ERR_TOPOLOGY = 2,      /* parent[i] >= i or < -1 (topological numbering is required) */
  BARD_ERR_UNSUPPORTED = 3,   /* nb > BARD_MAX_BODIES or nv > BARD_MAX_DOF or B too large */
  BARD_ERR_ALLOC = 4,
  BARD_ERR_CUDA = 5           /* failed cudaMalloc/cudaMemcpy/launch; text in bard_last_error() */
} bard_status;

typedef enum {
  BARD_JOINT_REVOLUTE = 0, BARD_JOINT_PRISMATIC = 1, BARD_JOINT_FIXED = 2, BARD_JOINT_FREE = 3
} bard_joint_type;

#define BARD_MAX_BODIES 64
#define BARD_MAX_DOF    64
#define BARD_MAX_FRAMES 16

/* Robot description (all HOST pointers, fp64; copied by bard_model_create). */
typedef struct {
  int32_t        nb;
  const int32_t* parent;      /* [nb]   -1 = world; parent[i] < i                                  */
  const int32_t* joint_type;  /* [nb]   bard_joint_type                                            */
  const double*  axis;        /* [nb*3] joint frame; normalised by the builder;
                                 ignored for FIXED / FREE                                          */
  const double*  T_pre;       /* [nb*12] rows [R|t]: the paper's T_joint (parent body -> joint)    */
  const double*  T_post;      /* [nb*12] or NULL = identity: the paper's T_link; identity for FREE */
  const double*  mass;        /* [nb]   >= 0 (massless links are legal; bard_aba needs positive inertia under every DOF) */
  const double*  com;         /* [nb*3] body frame                                                 */
  const double*  inertia;     /* [nb*6] xx,xy,xz,yy,yz,zz about the COM, body axes                 */
  double         gravity[3];  /* world frame, e.g. (0,0,-9.81)                                     */
} bard_model_desc;

/* Tables exported for bit-exact checks of the level schedule and index tables. */
enum {
  BARD_TAB_LEVEL_PTR = 0,   /* int32 [nlevels+1]                                              */
  BARD_TAB_LEVEL_BODY = 1,  /* int32 [nb]  bodies sorted by (level, body index)                */
  BARD_TAB_BODY_LEVEL = 2,  /* int32 [nb]                                                     */
  BARD_TAB_PARENT_SLOT = 3, /* int32 [nb]  slot in LEVEL_BODY of the parent of LEVEL_BODY[s]  */
  BARD_TAB_Q_OFF = 4,       /* int32 [nb+1]                                                   */
  BARD_TAB_V_OFF = 5,       /* int32 [nb+1]                                                   */
  BARD_TAB_DOF_BODY = 6,    /* int32 [nv]                                                     */
  BARD_TAB_ANC_MASK = 7,    /* uint64 [nb] bit j set <=> j == i or j is an ancestor of i      */
  BARD_TAB_RODRIGUES = 8    /* float [nb*36] R0 A B (3x3 row-major) t0 a b, eq. (2)-(3)       */
};

/* Build the immutable model on `cuda_device`: validation, q/v offsets, level schedule, ancestor sets,
 * Rodrigues constants (eq. (2)-(3); fp64 on the host, rounded once to fp32), motion
 * subspaces, compact spatial inertias; one upload of the constant blob.  *out is set on BARD_OK only.
 * cuda_device < 0 builds a HOST-ONLY model (no CUDA call): tables and dims can be queried, every
 * operator call on it returns BARD_ERR_INVALID_ARG. */
bard_status bard_model_create(const bard_model_desc* desc, int cuda_device, bard_model** out);
void        bard_model_destroy(bard_model* m);
bard_status bard_model_dims(const bard_model* m, int32_t* nb, int32_t* nq, int32_t* nv, int32_t* nlevels);
/* Copy table `table_id` to host_dst (cap bytes).  *need receives the size in bytes; if cap < need
 * nothing is copied and BARD_ERR_INVALID_ARG is returned (call with cap 0 to query). */
bard_status bard_model_get_table(const bard_model* m, int table_id, void* host_dst, size_t cap, size_t* need);
/* Choose the Jacobian frames: frame f is rigidly attached to body[f] at `offset` (body coordinates,
 * [nframes*3], NULL = zeros).  A build-time call: it SYNCHRONISES the model's device first (the J tables are
 * rewritten in place and the generated Jacobian / step kernels are unloaded, so no kernel that reads them -- on any
 * stream, blocking or not, including bard_step's internal side streams -- may still be in flight), then uploads.
 * Not thread-safe against concurrent operator calls on the same model from other host threads. */
bard_status bard_model_set_frames(bard_model* m, int32_t nframes, const int32_t* body, const double* offset);

/* Launch / code-generation knobs are fields of the model, never global state: bard_model_create reads the default of
 * option "x" once from the environment variable BARD_X (upper case), bard_model_set_option overrides it; no operator
 * call reads the environment.  Keys (int64 values, -1 = the documented automatic rule): teams, pack, pack2_min_b,
 * pdl (team kernels); spec_min_b, spec_block, spec_roles_max_b, spec_crba_roles_max_b, spec_crba_roles_min_b,
 * spec_fused_max_rows, spec_fused_small_b, spec_kin_min_b, spec_pack_min_b, spec_pack_max_b, step_fork_max_b, step_kin_fork, step_mode (which kernel a call gets: take effect at
 * the next operator call); spec_prefetch, spec_sync, spec_l2pf, spec_roles, spec_zero_role, spec_maxreg, spec_step4,
 * spec_step4_max_rows, spec_pack, spec_classical, spec_kin (code generation: take effect at the next bard_model_specialize).
 * section 10.  Unknown key: BARD_ERR_INVALID_ARG.  Not thread-safe against concurrent operator calls on the model. */
bard_status bard_model_set_option(bard_model* m, const char* key, int64_t value);
bard_status bard_model_get_option(const bard_model* m, const char* key, int64_t* value);

/* Operators, as bits of the `ops` mask of bard_model_specialize. */
enum { BARD_OP_FK = 1, BARD_OP_JACOBIAN = 2, BARD_OP_RNEA = 4, BARD_OP_CRBA = 8,
       BARD_OP_STEP = 15,     /* all four, each as its own kernel                                   */
       BARD_OP_FUSED = 16,    /* the fused kernel behind bard_step                                  */
       BARD_OP_ABA = 32,      /* forward dynamics (bard_aba): exists only as a specialised kernel   */
       BARD_OP_RNEA_ROLES = 64,   /* bard_model_specialized_source only: the limb-role RNEA kernel  */
       BARD_OP_CRBA_ROLES = 128,  /* bard_model_specialized_source only: the limb-role CRBA kernel */
       BARD_OP_RNEA_PACK2 = 256,  /* bard_model_specialized_source only: the RNEA kernel with two environments per thread */
       BARD_OP_KIN = 512,         /* bard_model_specialized_source only: the kinematics-fused kernel (FK + Jacobian + CRBA) */
       BARD_OP_RNEA_VJP = 1024 }; /* the generated kernel behind bard_rnea_vjp_params (the table-driven one serves without it) */

/* Model-specialised kernels (optional, once per model, takes seconds): writes straight-line CUDA source of
 * the operators in `ops` (BARD_OP_FUSED: one kernel that evaluates all four, see bard_step) for THIS model -- constants as literals, the tree walked depth first so that the
 * inward pass of a subtree follows its outward pass (eq. (6)) and only the bodies on
 * the current root-to-leaf path hold parked state -- compiles it for sm_100a with NVRTC (libnvrtc.so.12 of the
 * CUDA toolkit, loaded with dlopen) and loads the cubin.  Afterwards bard_<op> calls with a large batch
 * launch the specialised kernel (thresholds measured per operator -- chains: any B; teams of <= 4 warps: FK / Jacobian any B,
 * RNEA / CRBA B >= 4096; wider teams: Jacobian B >= 5000, FK B >= 16385, CRBA B >= 18945, RNEA B >= 32768), smaller ones
 * the level-parallel team kernel; results agree to rounding.  BARD_OP_RNEA on a single-rooted tree that branches
 * also builds a limb-role RNEA kernel (the subtrees below the first branching body dealt to two groups of warps
 * of the CTA, siblings' forces summed in ascending child order through shared memory: PAPER.md:91), which
 * bard_rnea launches for B <= 256 x SM count, below the thresholds above too.  The Jacobian is generated for the frames the
 * model has at the time of the call: bard_model_set_frames drops it (specialise again afterwards).  Unknown
 * bits: BARD_ERR_INVALID_ARG.  On a host-only model the source is generated and compiled but not loaded.  NVRTC missing or a compile error:
 * BARD_ERR_CUDA with the log in bard_last_error; the model stays usable.  Not thread-safe against concurrent
 * operator calls on the same model. */
bard_status bard_model_specialize(bard_model* m, uint32_t ops);
/* The generated source of one specialised operator (NUL-terminated) into host_dst; query with cap 0. */
bard_status bard_model_specialized_source(const bard_model* m, uint32_t op, char* host_dst, size_t cap, size_t* need);

/* FK (eq. (1)-(5), level-ordered outward propagation). */
bard_status bard_fk(const bard_model* m, int64_t B, const float* q, float* pose, bard_stream stream);
/* Geometric Jacobian of the frames chosen by bard_model_set_frames (eq. (7)). */
bard_status bard_jacobian(const bard_model* m, int64_t B, const float* q, float* J, bard_stream stream);
/* RNEA: outward velocity/acceleration pass (eq. (6)) and inward force pass
 * fused in one launch; gravity enters as a_world = -g. */
bard_status bard_rnea(const bard_model* m, int64_t B, const float* q, const float* qd, const float* qdd,
                      float* tau, bard_stream stream);
/* CRBA: composite-inertia backward sweep (the X^T M X update of PAPER.md:103) and mass-matrix fill. */
bard_status bard_crba(const bard_model* m, int64_t B, const float* q, float* M, bard_stream stream);

/* The three operators that depend on q alone -- poses, Jacobians and the mass matrix -- of one batch.  They share joint
 * transforms, world poses and screws (the paper's tiered cache: one FK evaluation shared by the queries): if
 * the model was specialised with BARD_OP_FUSED and B is above bard_step's fork regime (below), ONE kernel walks the tree once and stores all three
 * (the kernel bard_step launches beside bard_rnea on the larger robots); otherwise bard_fk, bard_jacobian and bard_crba in
 * sequence on `stream`.  Outputs and layouts as for the three calls. */
bard_status bard_kinematics(const bard_model* m, int64_t B, const float* q, float* pose, float* J, float* M, bard_stream stream);

/* One simulation step's worth of operators on one batch: poses, Jacobians, torques and mass matrix of the same
 * (q, qd, qdd) -- the paper's tiered cache and "full pipeline" restated on chip.  The form is chosen
 * per call from the batch size (option step_mode forces one):
 *   B <= step_fork_max_b: one operator's grid does not fill the machine, so bard_fk, bard_jacobian, bard_rnea and
 *     bard_crba are FORKED over three internal side streams and joined back into `stream`: the step costs its longest
 *     operator, not the sum; the fork-join is ordered after everything already in `stream`, is complete before anything
 *     enqueued later, and can be captured into a CUDA graph (one capture at a time per model);
 *   above, if the model was specialised with BARD_OP_FUSED: ONE launch -- the fused kernel that evaluates the joint
 *     transforms and FK once per body and shares them between the four operators (robots with a small parked state) --
 *     or TWO: the kinematics-fused kernel (FK + Jacobian + CRBA in one walk: they share q, poses and screws) and
 *     bard_rnea on an internal side stream (ALU-bound beside an HBM-bound kernel), joined back into `stream`;
 *   otherwise the four operators in sequence on `stream`.
 * Where the fork regime ends (option step_fork_max_b, -1 = automatic; bard_model_get_option(m, "step_fork_regime" /
 * "step_fork_regime_captured", &v) reads the current answer for plain calls / calls under stream capture): 256 x SM count on
 * a model without generated kernels.  bard_model_specialize(model, ... | BARD_OP_FUSED) on a device model MEASURES it: it times
 * the forked step and the one- / two-launch step at B = 4096 and 16 384 on the model's device as plain calls (scratch buffers
 * it allocates and frees: a build-time call, a few ms) and lets the one- / two-launch form take over from 3072 environments
 * if it is already faster at 4096 (a 7-DOF arm's fused kernel, an 11-DOF spined quadruped -- short walks, and no fork-join on
 * the host: sixteen API calls), from 8192 if it is faster at 16 384, else from 128 x SM count.  Under stream capture the host
 * cost does not exist and forking pays a little longer: bard_step asks the stream (cudaStreamIsCapturing) and then forks up
 * to at least 8192 (so a captured call and a plain call of the same batch may take different forms: their results agree to
 * rounding, not bit for bit; step_fork_max_b or step_mode pins one form).  Option step_calibrate = 0 replaces the measurement by a static rule on the length of the generated walk
 * (step_light_max).
 * Outputs and layouts as for the four calls. */
bard_status bard_step(const bard_model* m, int64_t B, const float* q, const float* qd, const float* qdd,
                      float* pose, float* J, float* tau, float* M, bard_stream stream);

/* Explicit Euler step on the configuration manifold, IN PLACE (BASELINE.json config 2: "q advanced by explicit
 * Euler from random qdd"; the paper's RL loop calls the operators once per simulated step):
 *   qd += dt qdd ;  q (+)= dt qd
 * revolute / prismatic: q += dt qd; free joint (q = [p, quat xyzw], qd = body-frame twist [v; omega]):
 * p += dt R(quat) v, quat += dt/2 quat (x) (omega, 0), renormalised.  One kernel launch, asynchronous. */
bard_status bard_euler_step(const bard_model* m, int64_t B, float dt, float* q, float* qd, const float* qdd,
                            bard_stream stream);
/* The same step OUT OF PLACE: (q, qd, qdd) -> (q_out, qd_out) (q_out == q and qd_out == qd is the in-place step; partial
 * overlap is not allowed).  With two or three state buffers a rollout can integrate step k on one stream WHILE the
 * operators of step k still read (q, qd) on another -- the next state depends on (q, qd, qdd) only (BASELINE.json config
 * 2: "q advanced by explicit Euler from random qdd"), so the integrator leaves the critical path (bench.py,
 * `config2_rollout.pipelined`). */
bard_status bard_euler_step_to(const bard_model* m, int64_t B, float dt, const float* q, const float* qd, const float* qdd,
                               float* q_out, float* qd_out, bard_stream stream);

/* ABA forward dynamics, the paper's fifth operator: qdd = M(q)^-1 (tau - C(q, qd)) by the
 * articulated-body algorithm -- three passes, the 6x6 update I^A_parent += X^T I^a X of PAPER.md:103 on the way up.
 * tau[nv][B] in, qdd[nv][B] out (free joint: [linear; angular] blocks as everywhere), gravity as in bard_rnea.
 * Two kernels: after bard_model_specialize(model, BARD_OP_ABA) the generated one (per-body state on chip; a free joint
 * must sit on a root body: BARD_ERR_UNSUPPORTED at specialisation otherwise); without it the table-driven one (any model,
 * a free joint anywhere, no NVRTC; per-body state in the workspace: ~12 KB of traffic per environment, 4-7x slower).  `workspace`: a caller-owned
 * device buffer of bard_aba_workspace_floats(model, B) floats -- 10 nv B with the generated kernel, 48 nb B without: ask
 * AFTER specialising.  Every body with a DOF needs a positive-definite articulated inertia (a massless subtree under a
 * joint divides by zero).  One launch, asynchronous. */
size_t      bard_aba_workspace_floats(const bard_model* m, int64_t B);
bard_status bard_aba(const bard_model* m, int64_t B, const float* q, const float* qd, const float* tau, float* qdd,
                     float* workspace, bard_stream stream);

/* Precision and layout variants of the four operators.
 *   dtype : BARD_F32 (default) or BARD_F64 -- the whole recursion in double, model constants as the builder's unrounded
 *           doubles: the instantiation that reproduces the paper's fp64 agreement table (Table 1)
 *           against the fp64 oracle (<= 1e-11 on the BASELINE robots).  Needs bard_model_specialize_variant(model, ops,
 *           BARD_F64, layout) first (NVRTC, as bard_model_specialize); BARD_ERR_UNSUPPORTED otherwise.
 *   layout: BARD_LAYOUT_SOA (default: [rows][B], batch fastest) or BARD_LAYOUT_AOS -- the paper's batch-first layout
 *           (PAPER.md:103): q (B, nq), qd / qdd / tau (B, nv), pose (B, nb, 12), J (B, nframes, 6, nv), M (B, nv, nv),
 *           contiguous, so PyTorch callers pass their (B, n) tensors as they are.  Served by tiled transposes around
 *           the SoA kernels (1 + number of input arrays extra launches) through `workspace`: a caller-owned device
 *           buffer of bard_variant_workspace_bytes(model, op, dtype, layout, B) bytes (0 / NULL for SoA).  B <= 2 097 120.
 * All launches are asynchronous on `stream`; pointers are device pointers to float or double according to dtype.
 * (BARD_F32, BARD_LAYOUT_SOA) is the plain operator call.  bard_model_set_frames / set_inertial_params drop the fp64
 * kernels that depend on them, like the plain ones. */
enum { BARD_F32 = 0, BARD_F64 = 1 };
enum { BARD_LAYOUT_SOA = 0, BARD_LAYOUT_AOS = 1 };
bard_status bard_model_specialize_variant(bard_model* m, uint32_t ops, int dtype, int layout);
bard_status bard_model_variant_source(const bard_model* m, uint32_t op, int dtype, int layout, char* host_dst, size_t cap, size_t* need);
size_t      bard_variant_workspace_bytes(const bard_model* m, uint32_t op, int dtype, int layout, int64_t B);
bard_status bard_fk_v      (const bard_model* m, int dtype, int layout, int64_t B, const void* q, void* pose, void* workspace, bard_stream stream);
bard_status bard_jacobian_v(const bard_model* m, int dtype, int layout, int64_t B, const void* q, void* J, void* workspace, bard_stream stream);
bard_status bard_rnea_v    (const bard_model* m, int dtype, int layout, int64_t B, const void* q, const void* qd, const void* qdd,
                            void* tau, void* workspace, bard_stream stream);
bard_status bard_crba_v    (const bard_model* m, int dtype, int layout, int64_t B, const void* q, void* M, void* workspace, bard_stream stream);

/* Reverse-mode derivative of RNEA with respect to the inertial parameters (the paper's
 * differentiable "functional mode", and its use: link masses identified through RNEA).
 * theta[nb][10] per link: m, h = m c (3), Io = Ic + m [c]x [c]x^T (xx,xy,xz,yy,yz,zz about the BODY ORIGIN, body axes);
 * tau is linear in theta.  Given the loss cotangent dtau[nv][B] (device, SoA like tau):
 *   dparams[i][k] = sum_b sum_j dtau[j][b] * d tau[j][b] / d theta[i][k]            (device, [nb*10] floats, fully overwritten)
 * One outward pass per environment (dtau is pushed outward like a velocity; no inward pass), then a DETERMINISTIC batch
 * reduction: fixed order inside a warp, warps and CTAs summed in ascending order (the last stage in fp64) -- the
 * same bits on every call with the same B and the same kernel.  Two kernels, two launches either way: a table-driven one
 * (any model, no bard_model_specialize needed) and, after bard_model_specialize(model, BARD_OP_RNEA_VJP), a generated
 * one (humanoid at B = 65 536: 20.7 us against 62 us; the two agree to rounding; the gradient does not depend on theta,
 * so bard_model_set_inertial_params keeps it).
 * `workspace`: caller-owned device buffer of bard_rnea_vjp_workspace_floats(model, B) floats (the same for both kernels:
 * nb * 10 floats x min(ceil(B / 32), 4 x SM count)).  B == 0 writes zeros. */
size_t      bard_rnea_vjp_workspace_floats(const bard_model* m, int64_t B);
bard_status bard_rnea_vjp_params(const bard_model* m, int64_t B, const float* q, const float* qd, const float* qdd,
                                 const float* dtau, float* dparams, float* workspace, bard_stream stream);
/* The same operation for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments without `workspace`, same kernels, same bits.  The scratch is a
 * static device array inside the library of BARD_VJP_STATIC_SCRATCH_FLOATS floats (1 MiB, held by every GPU that loads
 * the library until the process exits); a call with bard_rnea_vjp_workspace_floats(model, B) above that is refused with
 * BARD_ERR_UNSUPPORTED and a message (on a 148-SM GPU: more than 44 bodies at more than ~18 600 environments) -- use
 * bard_rnea_vjp_params then.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 * EVERY call on a device shares that one array: calls ordered on one stream are safe (nothing in the array has to start at
 * zero: each call overwrites every entry it later reads), calls that OVERLAP on the GPU (two streams without an ordering
 * between them) race on it and may return wrong sums.  The first call on a device looks the array's device address up
 * (cudaGetSymbolAddress, once per device): make that call outside stream capture. */
#define BARD_VJP_STATIC_SCRATCH_FLOATS 262144
bard_status bard_rnea_vjp_params_static(const bard_model* m, int64_t B, const float* q, const float* qd, const float* qdd,
                                        const float* dtau, float* dparams, bard_stream stream);
/* The model's theta (HOST, [nb*10] doubles) as bard_model_create derived it from (mass, com, inertia) -- and its
 * replacement, for optimisation loops over the inertial parameters (system identification): a build-time call like
 * bard_model_set_frames (SYNCHRONISES the device, rewrites the constant tables, drops the generated RNEA / CRBA / step /
 * ABA kernels, which have theta folded in as literals: the team kernels serve until bard_model_specialize runs again). */
bard_status bard_model_inertial_params(const bard_model* m, double* host_params);
bard_status bard_model_set_inertial_params(bard_model* m, const double* host_params);

/* Utility for the roofline report: the device's plain-FP32 FMA throughput in TFLOP/s, measured
 * with an FFMA-chain kernel (synchronous: allocates, launches, waits).  No operator depends on it. */
bard_status bard_measure_fp32_peak(int cuda_device, double* tflops);

const char* bard_status_string(bard_status s);
const char* bard_last_error(void);
/* Number of kernel launches this process has enqueued through the library (bench.py's gpu_launches). */
int64_t     bard_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif
