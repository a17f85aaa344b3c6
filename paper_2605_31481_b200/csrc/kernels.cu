// sm_100a kernels for the four operators -- level-parallel team schedule.
//
// Mapping.  A TEAM of L warps evaluates 32 environments: lane = environment, so the 32 lanes of every warp
// touch 32 adjacent floats of one SoA row (batch fastest) and each global load/store instruction moves one
// full 128-byte line.  The bodies of one tree level (eq. (6)) are spread over the team's L
// warps by the host schedule (model.cu); whole warps work on different bodies of the same environments, so
// there is no divergence and an idle warp costs no issue slots.  Warps of a team meet at a named barrier
// (bar.sync id, 32 L) between levels and exchange per-environment state through shared-memory columns
// state[row][lane] (bank-conflict free); a body that continues on its parent's warp reads it from registers.
// A CTA holds TEAMS teams that share one copy of the model constants.
//
// Staging.  The model constant blob (a few KB, identical for all environments) is copied into shared memory
// once per CTA with one TMA bulk copy (cp.async.bulk + mbarrier) and read with warp-uniform (broadcast)
// loads.  The team's input rows (q, and qd / qdd for RNEA) are staged with cp.async (LDGSTS) so that all
// input lines are in flight at once instead of one DRAM round trip per body.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdint>
#include <cstdlib>

#include "bard_internal.h"

namespace bard {

extern std::atomic<int64_t> g_launches;

namespace {

constexpr int W = 32;   // environments per team = lanes per warp = floats per state row

// ----------------------------------------------------------------------------- small vector algebra
struct V3 { float x, y, z; };
struct M3 { float m[9]; };   // row-major

__device__ __forceinline__ V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ V3 operator*(float s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ V3 cross(V3 a, V3 b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
__device__ __forceinline__ float dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ V3 mul(const M3& R, V3 v) {          // R v
  return {R.m[0] * v.x + R.m[1] * v.y + R.m[2] * v.z, R.m[3] * v.x + R.m[4] * v.y + R.m[5] * v.z,
          R.m[6] * v.x + R.m[7] * v.y + R.m[8] * v.z};
}
__device__ __forceinline__ V3 mulT(const M3& R, V3 v) {         // R^T v
  return {R.m[0] * v.x + R.m[3] * v.y + R.m[6] * v.z, R.m[1] * v.x + R.m[4] * v.y + R.m[7] * v.z,
          R.m[2] * v.x + R.m[5] * v.y + R.m[8] * v.z};
}
__device__ __forceinline__ M3 mul(const M3& a, const M3& b) {
  M3 c;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      c.m[3 * i + j] = a.m[3 * i] * b.m[j] + a.m[3 * i + 1] * b.m[3 + j] + a.m[3 * i + 2] * b.m[6 + j];
  return c;
}
// symmetric 3x3 (xx,xy,xz,yy,yz,zz) times vector
__device__ __forceinline__ V3 symmul(const float* I, V3 v) {
  return {I[0] * v.x + I[1] * v.y + I[2] * v.z, I[1] * v.x + I[3] * v.y + I[4] * v.z,
          I[2] * v.x + I[4] * v.y + I[5] * v.z};
}
__device__ __forceinline__ V3 ld3(const float* p) { return {p[0], p[1], p[2]}; }
// state rows: element k of a per-environment vector lives at s[k * W]
__device__ __forceinline__ V3 ldrow3(const float* s) { return {s[0], s[W], s[2 * W]}; }
__device__ __forceinline__ void strow3(float* s, V3 v) { s[0] = v.x; s[W] = v.y; s[2 * W] = v.z; }

// ----------------------------------------------------------------------------- staging
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void blob_issue(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  const uint32_t bar_a = smem_u32(bar);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(bar_a)
                 : "memory");
  }
}
__device__ __forceinline__ void blob_wait(uint64_t* bar) {
  const uint32_t bar_a = smem_u32(bar);
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar_a)
        : "memory");
  }
}
__device__ __forceinline__ void cp_async4(float* sdst, const float* gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(sdst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

// Per-thread view of the CTA: which team / warp of the team / environment, and where things are in smem.
struct Ctx {
  const BlobHeader* H;
  const BodyConst* bodies;
  const FrameConst* frames;
  const uint16_t* tasks;    // this warp's task list
  const uint8_t* children;
  float* st;                // this team's state rows, already offset by the lane
  int64_t e;                // environment (may be >= B in the ragged tail: loads clamp, stores are skipped)
  int64_t el;               // clamped environment for loads
  int team, w, L;
  bool valid;
};

__device__ __forceinline__ void team_sync(const Ctx& c) {
  if (c.L > 1) asm volatile("bar.sync %0, %1;" ::"r"(c.team + 1), "r"(c.L * 32) : "memory");
}

// Shared memory: [16 B mbarrier][blob][team 0 rows][team 1 rows]...  The first `nin` rows of a team are its
// staged inputs: row r of input array k (q, qd, qdd) comes from in_k[r * B + e].
__device__ __forceinline__ Ctx setup(unsigned char* smem, const void* gblob, uint32_t blob_bytes, int L, int team_rows,
                                     int64_t B, const float* in0, int n0, const float* in1, int n1, const float* in2,
                                     int n2) {
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem);
  unsigned char* blob = smem + 16;
  Ctx c;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  c.L = L;
  c.team = warp / L;
  c.w = warp - c.team * L;
  const int teams = (blockDim.x >> 5) / L;
  c.e = ((int64_t)blockIdx.x * teams + c.team) * W + lane;
  c.valid = c.e < B;
  c.el = c.valid ? c.e : B - 1;
  c.st = reinterpret_cast<float*>(blob + blob_bytes) + (size_t)c.team * team_rows * W + lane;
  blob_issue(blob, gblob, blob_bytes, bar);
  // stage the team's input rows; warp w takes rows w, w + L, ...
  for (int r = c.w; r < n0; r += L) cp_async4(c.st + r * W, in0 + (int64_t)r * B + c.el);
  for (int r = c.w; r < n1; r += L) cp_async4(c.st + (n0 + r) * W, in1 + (int64_t)r * B + c.el);
  for (int r = c.w; r < n2; r += L) cp_async4(c.st + (n0 + n1 + r) * W, in2 + (int64_t)r * B + c.el);
  cp_async_wait_all();
  __syncthreads();          // mbarrier init visible to all; staged rows visible to the other warps
  blob_wait(bar);
  c.H = reinterpret_cast<const BlobHeader*>(blob);
  c.bodies = reinterpret_cast<const BodyConst*>(blob + sizeof(BlobHeader));
  c.frames = reinterpret_cast<const FrameConst*>(blob + sizeof(BlobHeader) + sizeof(BodyConst) * c.H->nb);
  c.tasks = reinterpret_cast<const uint16_t*>(blob + c.H->off_tasks) + c.w * c.H->task_stride;
  c.children = blob + c.H->off_children;
  return c;
}

// ----------------------------------------------------------------------------- joint transform (a1)
// (u, w) of eq. (4)-(5): revolute (sin q, 1 - cos q); prismatic (q, 0); fixed (0, 0).
__device__ __forceinline__ void joint_uw(int type, float qv, float& u, float& w) {
  if (type == BARD_JOINT_REVOLUTE) {
    float s, c;
    sincosf(qv, &s, &c);
    u = s;
    w = 1.0f - c;
  } else if (type == BARD_JOINT_PRISMATIC) {
    u = qv;
    w = 0.f;
  } else {
    u = 0.f;
    w = 0.f;
  }
}
// R_pc = R0 + u A + w B ; t_pc = t0 + u a + w b   (eq. (4)-(5))
__device__ __forceinline__ void joint_Rt(const BodyConst& c, float u, float w, M3& R, V3& t) {
  const float4* c4 = reinterpret_cast<const float4*>(&c);      // words 0..35 with nine 16-byte broadcast loads
  float k[36];
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    const float4 v = c4[i];
    k[4 * i] = v.x; k[4 * i + 1] = v.y; k[4 * i + 2] = v.z; k[4 * i + 3] = v.w;
  }
#pragma unroll
  for (int i = 0; i < 9; ++i) R.m[i] = fmaf(w, k[18 + i], fmaf(u, k[9 + i], k[i]));
  if (c.flags & 1) {
    t = {fmaf(u, k[30], k[27]), fmaf(u, k[31], k[28]), fmaf(u, k[32], k[29])};   // revolute, T_post = I: a = b = 0
  } else {
    t = {fmaf(w, k[33], fmaf(u, k[30], k[27])), fmaf(w, k[34], fmaf(u, k[31], k[28])),
         fmaf(w, k[35], fmaf(u, k[32], k[29]))};
  }
}
// free joint: q = [p, quat xyzw]; R_pc = R0 R(quat/|quat|), t_pc = R0 p + t0.  qs = staged q rows of the team.
__device__ __forceinline__ void free_Rt(const BodyConst& c, const float* qs, M3& R, V3& t) {
  const float* qp = qs + c.q_off * W;
  V3 p = ldrow3(qp);
  float x = qp[3 * W], y = qp[4 * W], z = qp[5 * W], s = qp[6 * W];
  float n = rsqrtf(x * x + y * y + z * z + s * s);
  x *= n; y *= n; z *= n; s *= n;
  M3 Rq = {{1.f - 2.f * (y * y + z * z), 2.f * (x * y - z * s), 2.f * (x * z + y * s),
            2.f * (x * y + z * s), 1.f - 2.f * (x * x + z * z), 2.f * (y * z - x * s),
            2.f * (x * z - y * s), 2.f * (y * z + x * s), 1.f - 2.f * (x * x + y * y)}};
  M3 R0;
#pragma unroll
  for (int k = 0; k < 9; ++k) R0.m[k] = c.R0[k];
  R = mul(R0, Rq);
  t = mul(R0, p) + ld3(c.t0);
}
// local transform of a body from the staged q rows
__device__ __forceinline__ void local_Rt(const BodyConst& c, const float* qs, M3& R, V3& t, float& u, float& w) {
  if (c.type == BARD_JOINT_FREE) {
    u = 0.f; w = 0.f;
    free_Rt(c, qs, R, t);
  } else {
    const float qv = (c.type == BARD_JOINT_FIXED) ? 0.f : qs[c.q_off * W];
    joint_uw(c.type, qv, u, w);
    joint_Rt(c, u, w, R, t);
  }
}

// World pose of a body from its parent's (registers `cur`, a slot, or the world) -- a2.
struct Pose { M3 R; V3 p; };

__device__ __forceinline__ Pose compose_world(const BodyConst& c, const Pose& cur, const float* slots, const M3& R,
                                              V3 t) {
  Pose out;
  if (c.src == -1) {
    out.R = R;
    out.p = t;
    return out;
  }
  Pose par;
  if (c.src == -2) {
    par = cur;
  } else {
    const float* s = slots + c.src * 12 * W;
#pragma unroll
    for (int k = 0; k < 9; ++k) par.R.m[k] = s[k * W];
    par.p = ldrow3(s + 9 * W);
  }
  out.R = mul(par.R, R);
  out.p = mul(par.R, t) + par.p;
  return out;
}
__device__ __forceinline__ void save_pose(const BodyConst& c, const Pose& P, float* slots) {
  if (c.save >= 0) {
    float* s = slots + c.save * 12 * W;
#pragma unroll
    for (int k = 0; k < 9; ++k) s[k * W] = P.R.m[k];
    strow3(s + 9 * W, P.p);
  }
}

// ============================================================================= FK kernel (a1 + a2)
// team rows: q[nq] | pose slots[12 nslots]
__global__ void __launch_bounds__(256) fk_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int L, int team_rows,
                                                 int nq, int64_t B, const float* __restrict__ q,
                                                 float* __restrict__ pose) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gblob, blob_bytes, L, team_rows, B, q, nq, nullptr, 0, nullptr, 0);
  const float* qs = C.st;
  float* slots = C.st + nq * W;
  Pose cur;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) break;
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const BodyConst& c = C.bodies[i];
      M3 R; V3 t; float u, w;
      local_Rt(c, qs, R, t, u, w);
      cur = compose_world(c, cur, slots, R, t);
      save_pose(c, cur, slots);
      if (C.valid) {
        float* o = pose + (int64_t)i * 12 * B + C.e;
#pragma unroll
        for (int j = 0; j < 9; ++j) __stcs(o + j * B, cur.R.m[j]);
        __stcs(o + 9 * B, cur.p.x); __stcs(o + 10 * B, cur.p.y); __stcs(o + 11 * B, cur.p.z);
      }
    }
    if (tk & TASK_BAR) team_sync(C);
  }
}

// World-origin screws of a body's DOFs, s = [omega; v0] with v0 = R l + p x omega: for a revolute joint
// with T_post = I this is exactly the column [p_k x (R_k a'_k); R_k a'_k] of eq. (7).
// Stored as 6 rows per DOF at dof[(v * 6 + k) * W].
__device__ __forceinline__ void store_screws(const BodyConst& c, const Pose& P, float* dof) {
  if (c.type == BARD_JOINT_FIXED) return;
  float* d = dof + c.v_off * 6 * W;
  if (c.type == BARD_JOINT_FREE) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      V3 col = {P.R.m[k], P.R.m[3 + k], P.R.m[6 + k]};   // R e_k
      float* dl = d + k * 6 * W;                         // linear DOF k: omega = 0, v0 = R e_k
      strow3(dl, {0.f, 0.f, 0.f});
      strow3(dl + 3 * W, col);
      float* da = d + (3 + k) * 6 * W;                   // angular DOF k: omega = R e_k, v0 = p x omega
      strow3(da, col);
      strow3(da + 3 * W, cross(P.p, col));
    }
    return;
  }
  V3 om = mul(P.R, ld3(c.Sw));
  V3 v0 = cross(P.p, om);
  if (!(c.flags & 1) || c.type == BARD_JOINT_PRISMATIC) v0 = v0 + mul(P.R, ld3(c.Sl));
  strow3(d, om);
  strow3(d + 3 * W, v0);
}
// ============================================================================= Jacobian kernel (a3)
// team rows: q[nq] | pose slots[12 nslots] | screws[6 nv] | frame origins[3 nframes]
// Phase 1: level-parallel FK over the union of the frames' ancestor paths, screws and frame origins to smem.
// Phase 2: the nframes * nv columns are dealt round-robin to the team's warps; each writes its 6 rows.
__global__ void __launch_bounds__(256) jacobian_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int L,
                                                       int team_rows, int nq, int64_t B, const float* __restrict__ q,
                                                       float* __restrict__ J) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gblob, blob_bytes, L, team_rows, B, q, nq, nullptr, 0, nullptr, 0);
  const int nv = C.H->nv, nframes = C.H->nframes;
  const float* qs = C.st;
  float* slots = C.st + nq * W;
  float* dof = slots + C.H->nslots * 12 * W;
  float* pe = dof + nv * 6 * W;
  const uint64_t jmask = ((uint64_t)(uint32_t)C.H->jac_mask_hi << 32) | (uint32_t)C.H->jac_mask_lo;
  Pose cur;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) break;
    const int i = tk & TASK_BODY_MASK;
    if (!(tk & TASK_NOOP) && ((jmask >> i) & 1)) {
      const BodyConst& c = C.bodies[i];
      M3 R; V3 t; float u, w;
      local_Rt(c, qs, R, t, u, w);
      cur = compose_world(c, cur, slots, R, t);
      save_pose(c, cur, slots);
      store_screws(c, cur, dof);
      for (int f = 0; f < nframes; ++f)
        if (C.frames[f].body == i) strow3(pe + 3 * f * W, cur.p + mul(cur.R, ld3(C.frames[f].off)));
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  const uint8_t* dof_body = reinterpret_cast<const uint8_t*>(C.H) + C.H->off_dof_body;
  const int64_t rs = (int64_t)nv * B;
  for (int col = C.w; col < nframes * nv; col += L) {
    const int f = col / nv, j = col - f * nv;
    const FrameConst& fc = C.frames[f];
    const uint64_t anc = ((uint64_t)fc.anc_hi << 32) | fc.anc_lo;
    V3 lin = {0.f, 0.f, 0.f}, ang = {0.f, 0.f, 0.f};
    if ((anc >> dof_body[j]) & 1) {
      const float* d = dof + j * 6 * W;
      ang = ldrow3(d);
      lin = ldrow3(d + 3 * W) + cross(ang, ldrow3(pe + 3 * f * W));   // shift the world-origin column to the frame origin
    }
    if (C.valid) {
      float* o = J + ((int64_t)f * 6 * nv + j) * B + C.e;
      __stcs(o, lin.x); __stcs(o + rs, lin.y); __stcs(o + 2 * rs, lin.z);
      __stcs(o + 3 * rs, ang.x); __stcs(o + 4 * rs, ang.y); __stcs(o + 5 * rs, ang.z);
    }
  }
}

// ============================================================================= RNEA kernel (a4 + a5)
// Body-frame recursion, internal order [angular; linear].
// team rows: q[nq] | qd[nv] | qdd[nv] | motion slots[12 nslots] (v.w v.v a.w a.v) | force[6 nb] (n f) | uw[2 nb]
// Outward (level-parallel, eq. (6)): v, a of the parent come from the registers of this warp's
// previous task, a shared-memory slot, or the world (v = 0, a = -g: gravity trick); the net body force f_i and
// the joint scalars (u, w) are parked in shared memory.
// Inward (PAPER.md:91 keeps this pass sequential because siblings collide on the parent; here it is
// level-parallel too): a body first adds the forces its children left -- already expressed in ITS frame -- in
// ascending child order (deterministic, no atomics), emits tau_i = S_i^T f_i, then overwrites its own force
// rows with X_up^T f_i for its parent, rebuilding T_pc from (u, w) with eq. (4)-(5).
struct Motion { V3 w, v; };   // [angular; linear]

__global__ void __launch_bounds__(256) rnea_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int L, int team_rows,
                                                   int nq, int nv, int64_t B, const float* __restrict__ q,
                                                   const float* __restrict__ qd, const float* __restrict__ qdd,
                                                   float* __restrict__ tau) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gblob, blob_bytes, L, team_rows, B, q, nq, qd, nv, qdd, nv);
  const int nb = C.H->nb;
  const float* qs = C.st;
  const float* qds = qs + nq * W;
  const float* qdds = qds + nv * W;
  float* slots = C.st + (nq + 2 * nv) * W;
  float* bst = slots + C.H->nslots * 12 * W;
  float* uw = bst + nb * 6 * W;
  const V3 g = ld3(C.H->g);
  Motion cv, ca;                                               // this warp's previous body: velocity / acceleration
  int ntask = 0;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) { ntask = k; break; }
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const BodyConst& c = C.bodies[i];
      M3 R; V3 t; float u, w;
      local_Rt(c, qs, R, t, u, w);
      // joint velocity / acceleration in the body frame: S qd, S qdd
      Motion vJ = {{0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}}, aJ = vJ;
      if (c.type == BARD_JOINT_FREE) {
        const float* d1 = qds + c.v_off * W;
        const float* d2 = qdds + c.v_off * W;
        vJ = {ldrow3(d1 + 3 * W), ldrow3(d1)};
        aJ = {ldrow3(d2 + 3 * W), ldrow3(d2)};
      } else if (c.type != BARD_JOINT_FIXED) {
        const float qd_i = qds[c.v_off * W], qdd_i = qdds[c.v_off * W];
        const V3 sw = ld3(c.Sw), sl = ld3(c.Sl);
        vJ = {qd_i * sw, qd_i * sl};
        aJ = {qdd_i * sw, qdd_i * sl};
      }
      // X_up [w; v] = [R^T w ; R^T (v + w x t)]   (Pluecker motion transform with (E, r) = (R^T, t))
      Motion v, a;
      if (c.src == -1) {                                       // world parent: v_p = 0, a_p = [0; -g]
        v = vJ;                                                // (v x vJ = 0 since v = vJ)
        a.w = aJ.w;
        a.v = mulT(R, {-g.x, -g.y, -g.z}) + aJ.v;
      } else {
        Motion pv, pa;
        if (c.src == -2) {
          pv = cv; pa = ca;
        } else {
          const float* s = slots + c.src * 12 * W;
          pv = {ldrow3(s), ldrow3(s + 3 * W)};
          pa = {ldrow3(s + 6 * W), ldrow3(s + 9 * W)};
        }
        v.w = mulT(R, pv.w) + vJ.w;
        v.v = mulT(R, pv.v + cross(pv.w, t)) + vJ.v;
        a.w = mulT(R, pa.w) + aJ.w + cross(v.w, vJ.w);
        a.v = mulT(R, pa.v + cross(pa.w, t)) + aJ.v + cross(v.w, vJ.v) + cross(v.v, vJ.w);
      }
      // f = I a + v x* (I v),  I = (m, h, Io) about the body origin
      const V3 h = ld3(c.h);
      const float m = c.mass;
      const V3 n1 = symmul(c.Io, v.w) + cross(h, v.v);
      const V3 f1 = m * v.v - cross(h, v.w);
      const V3 n2 = symmul(c.Io, a.w) + cross(h, a.v);
      const V3 f2 = m * a.v - cross(h, a.w);
      const V3 n = n2 + cross(v.w, n1) + cross(v.v, f1);
      const V3 f = f2 + cross(v.w, f1);
      float* b = bst + i * 6 * W;
      strow3(b, n); strow3(b + 3 * W, f);
      uw[(2 * i) * W] = u; uw[(2 * i + 1) * W] = w;
      if (c.save >= 0) {
        float* s = slots + c.save * 12 * W;
        strow3(s, v.w); strow3(s + 3 * W, v.v); strow3(s + 6 * W, a.w); strow3(s + 9 * W, a.v);
      }
      cv = v; ca = a;
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  // inward pass, deepest level first: the same task list walked backwards
  for (int k = ntask - 1; k >= 0; --k) {
    const uint32_t tk = C.tasks[k];
    if ((tk & TASK_BAR) && k != ntask - 1) team_sync(C);
    if (tk & TASK_NOOP) continue;
    const int i = tk & TASK_BODY_MASK;
    const BodyConst& c = C.bodies[i];
    float* b = bst + i * 6 * W;
    V3 n = ldrow3(b), f = ldrow3(b + 3 * W);
    for (int cc = 0; cc < c.child_count; ++cc) {
      const float* cb = bst + C.children[c.child_begin + cc] * 6 * W;
      n = n + ldrow3(cb); f = f + ldrow3(cb + 3 * W);
    }
    if (C.valid) {
      float* to = tau + (int64_t)c.v_off * B + C.e;
      if (c.type == BARD_JOINT_FREE) {
        __stcs(to, f.x); __stcs(to + B, f.y); __stcs(to + 2 * B, f.z);
        __stcs(to + 3 * B, n.x); __stcs(to + 4 * B, n.y); __stcs(to + 5 * B, n.z);
      } else if (c.type != BARD_JOINT_FIXED) {
        __stcs(to, dot(ld3(c.Sw), n) + dot(ld3(c.Sl), f));
      }
    }
    if (c.parent >= 0) {
      M3 R; V3 t;
      if (c.type == BARD_JOINT_FREE) free_Rt(c, qs, R, t);
      else joint_Rt(c, uw[(2 * i) * W], uw[(2 * i + 1) * W], R, t);
      const V3 fp = mul(R, f);
      strow3(b, mul(R, n) + cross(t, fp));
      strow3(b + 3 * W, fp);
    }
  }
}

// ============================================================================= CRBA kernel (a6 + a7)
// World-frame formulation: every composite inertia is expressed about the WORLD origin in world axes
// (m, h, I: 10 floats), so the backward sweep  I^c_parent += X^T I^c_child X degenerates to
// ten additions (X = identity between world-frame quantities), and M_ij = s_j . (I^c_i s_i) for every
// ancestor DOF j needs no transform along the walk.  The screws s are the eq. (7) columns (store_screws).
// team rows: q[nq] | pose slots[12 nslots] | screws[6 nv] | inertia[10 nb]
// Phase 1 (outward, level-parallel): FK, screws, world-frame body inertias.
// Phase 2 (inward, level-parallel): a body adds its children's composites in ascending child order.
// Phase 3: the rows of M are dealt to the team's warps (host LPT schedule); both M[i][j] and M[j][i] are
//          written by the warp that owns row i >= j, every element exactly once.
__global__ void __launch_bounds__(256) crba_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int L, int team_rows,
                                                   int nq, int64_t B, const float* __restrict__ q,
                                                   float* __restrict__ Mout) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gblob, blob_bytes, L, team_rows, B, q, nq, nullptr, 0, nullptr, 0);
  const int nv = C.H->nv;
  const float* qs = C.st;
  float* slots = C.st + nq * W;
  float* dof = slots + C.H->nslots * 12 * W;                   // 6 rows per DOF
  float* ic = dof + nv * 6 * W;                                // 10 rows per body: m h(3) I(6)
  Pose cur;
  int ntask = 0;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) { ntask = k; break; }
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const BodyConst& c = C.bodies[i];
      M3 R; V3 t; float u, w;
      local_Rt(c, qs, R, t, u, w);
      cur = compose_world(c, cur, slots, R, t);
      save_pose(c, cur, slots);
      store_screws(c, cur, dof);
      // body inertia about the world origin: h' = R h + m p ; with h'' = R h + m p / 2:
      // I' = R Io R^T + 2 (p . h'') 1 - (h'' p^T + p h''^T)
      const float m = c.mass;
      const V3 hr = mul(cur.R, ld3(c.h));
      const V3 p = cur.p;
      const V3 hh = hr + (0.5f * m) * p;
      const V3 r0 = {cur.R.m[0], cur.R.m[1], cur.R.m[2]}, r1 = {cur.R.m[3], cur.R.m[4], cur.R.m[5]},
               r2 = {cur.R.m[6], cur.R.m[7], cur.R.m[8]};
      const V3 a0 = symmul(c.Io, r0), a1 = symmul(c.Io, r1), a2 = symmul(c.Io, r2);
      const float d = 2.f * dot(p, hh);
      float* o = ic + i * 10 * W;
      o[0] = m;
      strow3(o + W, hr + m * p);
      o[4 * W] = dot(r0, a0) + d - 2.f * hh.x * p.x;             // xx
      o[5 * W] = dot(r0, a1) - (hh.x * p.y + p.x * hh.y);        // xy
      o[6 * W] = dot(r0, a2) - (hh.x * p.z + p.x * hh.z);        // xz
      o[7 * W] = dot(r1, a1) + d - 2.f * hh.y * p.y;             // yy
      o[8 * W] = dot(r1, a2) - (hh.y * p.z + p.y * hh.z);        // yz
      o[9 * W] = dot(r2, a2) + d - 2.f * hh.z * p.z;             // zz
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  // composite sweep, deepest level first
  for (int k = ntask - 1; k >= 0; --k) {
    const uint32_t tk = C.tasks[k];
    if ((tk & TASK_BAR) && k != ntask - 1) team_sync(C);
    if (tk & TASK_NOOP) continue;
    const BodyConst& c = C.bodies[tk & TASK_BODY_MASK];
    if (c.child_count == 0) continue;
    float* d = ic + (tk & TASK_BODY_MASK) * 10 * W;
    float acc[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) acc[j] = d[j * W];
    for (int cc = 0; cc < c.child_count; ++cc) {
      const float* s = ic + C.children[c.child_begin + cc] * 10 * W;
#pragma unroll
      for (int j = 0; j < 10; ++j) acc[j] += s[j * W];
    }
#pragma unroll
    for (int j = 0; j < 10; ++j) d[j * W] = acc[j];
  }
  team_sync(C);
  // fill
  const uint8_t* dof_body = reinterpret_cast<const uint8_t*>(C.H) + C.H->off_dof_body;
  const uint8_t* rows = reinterpret_cast<const uint8_t*>(C.H) + C.H->off_fill + C.w * C.H->fill_stride;
  for (int k = 0;; ++k) {
    const int i = rows[k];
    if (i == 0xff) break;
    const int bi = dof_body[i];
    const BodyConst& ci = C.bodies[bi];
    const uint64_t anc = ((uint64_t)ci.anc_hi << 32) | ci.anc_lo;
    const float* I = ic + bi * 10 * W;
    const float m = I[0];
    const V3 h = ldrow3(I + W);
    const float Iw[6] = {I[4 * W], I[5 * W], I[6 * W], I[7 * W], I[8 * W], I[9 * W]};
    const float* si = dof + i * 6 * W;
    const V3 om = ldrow3(si), v0 = ldrow3(si + 3 * W);
    const V3 Fn = symmul(Iw, om) + cross(h, v0);             // F = I^c_i s_i  (moment about the world origin)
    const V3 Ff = m * v0 - cross(h, om);                     //               (force)
    float* row = Mout + (int64_t)i * nv * B + C.e;           // M[i][.]
    float* colp = Mout + (int64_t)i * B + C.e;               // M[.][i]
    for (int j = 0; j <= i; ++j) {
      float val = 0.f;
      if ((anc >> dof_body[j]) & 1) {
        const float* sj = dof + j * 6 * W;
        val = dot(ldrow3(sj), Fn) + dot(ldrow3(sj + 3 * W), Ff);
      }
      if (C.valid) {
        __stcs(row + (int64_t)j * B, val);
        if (j != i) __stcs(colp + (int64_t)j * nv * B, val);
      }
    }
  }
}

// ----------------------------------------------------------------------------- launchers
struct LaunchCfg { int teams, threads, team_rows; size_t smem; unsigned grid; };

constexpr size_t kSmemMax = 227 * 1024;

int env_int(const char* name, int dflt) {
  const char* v = std::getenv(name);
  return v ? std::atoi(v) : dflt;
}

// TEAMS per CTA: two 32-environment teams share one blob copy when the team is narrow; fewer if the state
// does not fit.  Small CTAs keep the last wave short at B = 65 536 (2048 tiles over 148 SMs).
bool pick_cfg(const Model& m, int64_t B, int team_rows, LaunchCfg& cfg) {
  const int L = m.team_warps;
  static const int want = env_int("BARD_TEAMS", 0);            // tuning knob for experiments
  int teams = want > 0 ? want : (L <= 4 ? 2 : 1);
  teams = std::max(1, std::min(teams, 8 / L));
  const size_t fixed = 16 + m.blob_bytes;
  const size_t per_team = (size_t)team_rows * W * sizeof(float);
  while (teams > 1 && (fixed + per_team * teams) * 2 + 2048 > kSmemMax) --teams;   // keep >= 2 CTAs per SM
  cfg.teams = teams;
  cfg.threads = teams * L * 32;
  cfg.team_rows = team_rows;
  cfg.smem = fixed + per_team * teams;
  cfg.grid = (unsigned)((B + (int64_t)teams * W - 1) / ((int64_t)teams * W));
  return cfg.smem <= kSmemMax;
}

template <int ID, typename K>   // ID: one static per kernel (several kernels share a signature)
bard_status prep(K kernel, const char* name, bool fits) {
  if (!fits) { set_error(std::string(name) + ": per-environment state does not fit in shared memory"); return BARD_ERR_UNSUPPORTED; }
  static thread_local int done_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  if (done_dev != dev) {
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
    if (e != cudaSuccess) { set_error(std::string(name) + ": " + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
    done_dev = dev;
  }
  return BARD_OK;
}
bard_status finish(const char* name) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_error(std::string(name) + ": " + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
  g_launches.fetch_add(1);
  return BARD_OK;
}

}  // namespace

bard_status launch_fk(const Model& m, int64_t B, const float* q, float* pose, void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.nq + 12 * m.nslots, cfg);
  bard_status s = prep<0>(fk_kernel, "bard_fk", fits);
  if (s != BARD_OK) return s;
  fk_kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(m.d_blob, (uint32_t)m.blob_bytes, m.team_warps,
                                                                       cfg.team_rows, m.nq, B, q, pose);
  return finish("bard_fk");
}
bard_status launch_jacobian(const Model& m, int64_t B, const float* q, float* J, void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.nq + 12 * m.nslots + 6 * m.nv + 3 * m.nframes, cfg);
  bard_status s = prep<1>(jacobian_kernel, "bard_jacobian", fits);
  if (s != BARD_OK) return s;
  jacobian_kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(
      m.d_blob, (uint32_t)m.blob_bytes, m.team_warps, cfg.team_rows, m.nq, B, q, J);
  return finish("bard_jacobian");
}
bard_status launch_rnea(const Model& m, int64_t B, const float* q, const float* qd, const float* qdd, float* tau,
                        void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.nq + 2 * m.nv + 12 * m.nslots + 8 * m.nb, cfg);
  bard_status s = prep<2>(rnea_kernel, "bard_rnea", fits);
  if (s != BARD_OK) return s;
  rnea_kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(
      m.d_blob, (uint32_t)m.blob_bytes, m.team_warps, cfg.team_rows, m.nq, m.nv, B, q, qd, qdd, tau);
  return finish("bard_rnea");
}
bard_status launch_crba(const Model& m, int64_t B, const float* q, float* M, void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.nq + 12 * m.nslots + 6 * m.nv + 10 * m.nb, cfg);
  bard_status s = prep<3>(crba_kernel, "bard_crba", fits);
  if (s != BARD_OK) return s;
  crba_kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(
      m.d_blob, (uint32_t)m.blob_bytes, m.team_warps, cfg.team_rows, m.nq, B, q, M);
  return finish("bard_crba");
}

}  // namespace bard
