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
// Staging.  The model constant sections (a few KB, identical for all environments) are copied into shared
// memory once per CTA with TMA bulk copies (cp.async.bulk + mbarrier) and read with warp-uniform (broadcast)
// 16-byte loads.  The team's input rows (q, and qd / qdd for RNEA) are staged with cp.async (LDGSTS) so that
// all input lines are in flight at once instead of one DRAM round trip per body.
//
// Stores.  Output rows are B floats apart (B is a run-time value), so every store address is
// base + row * 4B, formed by ONE mad.wide.u32 (IMAD.WIDE) from a 32-bit row index; structurally zero rows of
// J and M are written by a separate pass, four rows per 16-byte store instruction.
//
// Every kernel exists in two instantiations: SIMPLE (every joint is a revolute joint with T_post = I or a
// free joint -- all BASELINE configs) and the general one (prismatic / fixed joints, T_post != I).
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
// Written as fused multiply-add chains: acc + R v, acc + a x b, ... so that almost every FP instruction
// is an FFMA.
struct V3 { float x, y, z; };
struct M3 { float m[9]; };   // row-major

__device__ __forceinline__ V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ V3 operator*(float s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ V3 axpy(float s, V3 a, V3 acc) {      // acc + s a
  return {fmaf(s, a.x, acc.x), fmaf(s, a.y, acc.y), fmaf(s, a.z, acc.z)};
}
__device__ __forceinline__ V3 cross(V3 a, V3 b) {
  return {fmaf(a.y, b.z, -a.z * b.y), fmaf(a.z, b.x, -a.x * b.z), fmaf(a.x, b.y, -a.y * b.x)};
}
__device__ __forceinline__ V3 cross_acc(V3 a, V3 b, V3 acc) {    // acc + a x b
  return {fmaf(-a.z, b.y, fmaf(a.y, b.z, acc.x)), fmaf(-a.x, b.z, fmaf(a.z, b.x, acc.y)),
          fmaf(-a.y, b.x, fmaf(a.x, b.y, acc.z))};
}
__device__ __forceinline__ float dot(V3 a, V3 b) { return fmaf(a.z, b.z, fmaf(a.y, b.y, a.x * b.x)); }
__device__ __forceinline__ float dot_acc(V3 a, V3 b, float acc) { return fmaf(a.z, b.z, fmaf(a.y, b.y, fmaf(a.x, b.x, acc))); }
__device__ __forceinline__ V3 mul(const M3& R, V3 v) {           // R v
  return {fmaf(R.m[2], v.z, fmaf(R.m[1], v.y, R.m[0] * v.x)), fmaf(R.m[5], v.z, fmaf(R.m[4], v.y, R.m[3] * v.x)),
          fmaf(R.m[8], v.z, fmaf(R.m[7], v.y, R.m[6] * v.x))};
}
__device__ __forceinline__ V3 mul_acc(const M3& R, V3 v, V3 acc) {   // acc + R v
  return {fmaf(R.m[2], v.z, fmaf(R.m[1], v.y, fmaf(R.m[0], v.x, acc.x))),
          fmaf(R.m[5], v.z, fmaf(R.m[4], v.y, fmaf(R.m[3], v.x, acc.y))),
          fmaf(R.m[8], v.z, fmaf(R.m[7], v.y, fmaf(R.m[6], v.x, acc.z)))};
}
__device__ __forceinline__ V3 mulT(const M3& R, V3 v) {          // R^T v
  return {fmaf(R.m[6], v.z, fmaf(R.m[3], v.y, R.m[0] * v.x)), fmaf(R.m[7], v.z, fmaf(R.m[4], v.y, R.m[1] * v.x)),
          fmaf(R.m[8], v.z, fmaf(R.m[5], v.y, R.m[2] * v.x))};
}
__device__ __forceinline__ V3 mulT_acc(const M3& R, V3 v, V3 acc) {  // acc + R^T v
  return {fmaf(R.m[6], v.z, fmaf(R.m[3], v.y, fmaf(R.m[0], v.x, acc.x))),
          fmaf(R.m[7], v.z, fmaf(R.m[4], v.y, fmaf(R.m[1], v.x, acc.y))),
          fmaf(R.m[8], v.z, fmaf(R.m[5], v.y, fmaf(R.m[2], v.x, acc.z)))};
}
__device__ __forceinline__ M3 mul(const M3& a, const M3& b) {
  M3 c;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      c.m[3 * i + j] = fmaf(a.m[3 * i + 2], b.m[6 + j], fmaf(a.m[3 * i + 1], b.m[3 + j], a.m[3 * i] * b.m[j]));
  return c;
}
// symmetric 3x3 (xx,xy,xz,yy,yz,zz) times vector
__device__ __forceinline__ V3 symmul(const float* I, V3 v) {
  return {fmaf(I[2], v.z, fmaf(I[1], v.y, I[0] * v.x)), fmaf(I[4], v.z, fmaf(I[3], v.y, I[1] * v.x)),
          fmaf(I[5], v.z, fmaf(I[4], v.y, I[2] * v.x))};
}
// state rows: element k of a per-environment vector lives at s[k * W]
__device__ __forceinline__ V3 ldrow3(const float* s) { return {s[0], s[W], s[2 * W]}; }
__device__ __forceinline__ void strow3(float* s, V3 v) { s[0] = v.x; s[W] = v.y; s[2 * W] = v.z; }

// sin and cos of x together: Cody-Waite reduction by pi/2 in three FMA steps, then the classic
// single-precision minimax polynomials on [-pi/4, pi/4] (Cephes sinf / cosf coefficients) and a quadrant
// fix-up.  About 1 ulp for |x| <= 1e4 rad; degrades gracefully (never NaN for finite x) up to ~6e6.
__device__ __forceinline__ void sincos_fast(float x, float& s, float& c) {
  const float kb = fmaf(x, 0.636619772367581343f, 12582912.0f);   // round(x * 2/pi) in the low mantissa bits
  const float k = kb - 12582912.0f;
  const int qd = __float_as_int(kb);
  float r = fmaf(k, -1.57079637050628662109375f, x);
  r = fmaf(k, 4.371138828673793e-8f, r);
  r = fmaf(k, 1.7151245100058819e-15f, r);
  const float r2 = r * r;
  float ps = fmaf(r2, -1.9515295891e-4f, 8.3321608736e-3f);
  ps = fmaf(ps, r2, -1.6666654611e-1f);
  ps = fmaf(ps * r2, r, r);                                       // sin r
  float pc = fmaf(r2, 2.443315711809948e-5f, -1.388731625493765e-3f);
  pc = fmaf(pc, r2, 4.166664568298827e-2f);
  pc = fmaf(pc * r2, r2, fmaf(r2, -0.5f, 1.0f));                  // cos r
  const float ss = (qd & 1) ? pc : ps;
  const float cc = (qd & 1) ? ps : pc;
  s = __int_as_float(__float_as_int(ss) ^ ((qd & 2) << 30));
  c = __int_as_float(__float_as_int(cc) ^ (((qd + 1) & 2) << 30));
}

// ----------------------------------------------------------------------------- staging and addressing
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint32_t bar_a) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(bar_a)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar_a) {
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
// base + row * B4 bytes in one IMAD.WIDE (B4 = 4 B < 2^32, checked by the C ABI)
__device__ __forceinline__ float* rowptr(float* base, uint32_t row, uint32_t B4) {
  uint64_t a;
  asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(a) : "r"(row), "r"(B4), "l"(reinterpret_cast<uint64_t>(base)));
  return reinterpret_cast<float*>(a);
}

// ----------------------------------------------------------------------------- per-thread view of the CTA
// Shared memory: [16 B mbarrier][COMMON][extra section: M or J tables, or nothing][team 0 rows][team 1 rows]...
// The first rows of a team are its staged inputs: row r of input array k (q, qd, qdd) is in_k[r * B + e].
struct Ctx {
  const unsigned char* common;   // BlobHeader | BodyConst[nb] | tasks | children | dof_body
  const unsigned char* extra;    // MHeader... or JHeader...
  const BodyConst* bodies;
  const uint16_t* tasks;         // this warp's task list
  float* st;                     // this team's state rows, already offset by the lane
  uint32_t e;                    // environment of this lane (may be >= B in the ragged tail: stores are skipped)
  int team, w, L, lane;
  bool valid;
};

__device__ __forceinline__ void team_sync(const Ctx& c) {
  if (c.L > 1) asm volatile("bar.sync %0, %1;" ::"r"(c.team + 1), "r"(c.L * 32) : "memory");
}

__device__ __forceinline__ Ctx setup(unsigned char* smem, const void* gcommon, uint32_t cbytes, const void* gextra,
                                     uint32_t xbytes, int L, int team_rows, uint32_t B, const float* in0, int n0,
                                     const float* in1, int n1, const float* in2, int n2) {
  const uint32_t bar_a = smem_u32(smem);
  unsigned char* blob = smem + 16;
  Ctx c;
  const int warp = threadIdx.x >> 5;
  c.lane = threadIdx.x & 31;
  c.L = L;
  c.team = warp / L;
  c.w = warp - c.team * L;
  const int teams = (blockDim.x >> 5) / L;
  c.e = (blockIdx.x * teams + c.team) * W + c.lane;
  c.valid = c.e < B;
  const uint32_t el = c.valid ? c.e : B - 1;                 // clamped environment for loads
  c.st = reinterpret_cast<float*>(blob + cbytes + xbytes) + c.team * team_rows * W + c.lane;
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(cbytes + xbytes) : "memory");
    bulk_g2s(blob, gcommon, cbytes, bar_a);
    if (xbytes) bulk_g2s(blob + cbytes, gextra, xbytes, bar_a);
  }
  // stage the team's input rows; warp w takes rows w, w + L, ...
  const uint32_t B4 = B * 4u;
  for (int r = c.w; r < n0; r += L) cp_async4(c.st + r * W, rowptr(const_cast<float*>(in0) + el, r, B4));
  for (int r = c.w; r < n1; r += L) cp_async4(c.st + (n0 + r) * W, rowptr(const_cast<float*>(in1) + el, r, B4));
  for (int r = c.w; r < n2; r += L) cp_async4(c.st + (n0 + n1 + r) * W, rowptr(const_cast<float*>(in2) + el, r, B4));
  cp_async_wait_all();
  __syncthreads();          // mbarrier init visible to all; staged rows visible to the other warps
  mbar_wait(bar_a);
  c.common = blob;
  c.extra = blob + cbytes;
  const BlobHeader* H = reinterpret_cast<const BlobHeader*>(blob);
  c.bodies = reinterpret_cast<const BodyConst*>(blob + sizeof(BlobHeader));
  c.tasks = reinterpret_cast<const uint16_t*>(blob + H->off_tasks) + c.w * H->task_stride;
  return c;
}

// Integer fields of a BodyConst with three 16-byte broadcast loads.
struct Meta { int type, parent, q_off, v_off, src, save, flags, level; uint32_t anc_lo, anc_hi; int child_begin, child_count; };
__device__ __forceinline__ Meta load_meta(const BodyConst& c) {
  const int4* p = reinterpret_cast<const int4*>(&c) + 13;
  const int4 a = p[0], b = p[1], d = p[2];
  return {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, (uint32_t)d.x, (uint32_t)d.y, d.z, d.w};
}
// words 36..51: Sw Sl mass h Io
struct Inertia { V3 Sw, Sl; float mass; V3 h; float Io[6]; };
__device__ __forceinline__ Inertia load_inertia(const BodyConst& c) {
  const float4* p = reinterpret_cast<const float4*>(&c) + 9;
  const float4 a = p[0], b = p[1], d = p[2], e = p[3];
  return {{a.x, a.y, a.z}, {a.w, b.x, b.y}, b.z, {b.w, d.x, d.y}, {d.z, d.w, e.x, e.y, e.z, e.w}};
}

// ----------------------------------------------------------------------------- joint transform (a1)
// R_pc = R0 + u A + w B ; t_pc = t0 + u a + w b   (eq. (4)-(5)), constants read with
// 16-byte broadcast loads.  (u, w): revolute (sin q, 1 - cos q); prismatic (q, 0); fixed (0, 0).
template <bool SIMPLE>
__device__ __forceinline__ void joint_Rt(const BodyConst& c, int flags, float u, float w, M3& R, V3& t) {
  const float4* c4 = reinterpret_cast<const float4*>(&c);
  float k[36];
#pragma unroll
  for (int i = 0; i < (SIMPLE ? 8 : 9); ++i) {
    const float4 v = c4[i];
    k[4 * i] = v.x; k[4 * i + 1] = v.y; k[4 * i + 2] = v.z; k[4 * i + 3] = v.w;
  }
#pragma unroll
  for (int i = 0; i < 9; ++i) R.m[i] = fmaf(w, k[18 + i], fmaf(u, k[9 + i], k[i]));
  if (SIMPLE || (flags & 1)) {
    t = {k[27], k[28], k[29]};                                 // T_post = I: a = b = 0
  } else {
    t = {fmaf(w, k[33], fmaf(u, k[30], k[27])), fmaf(w, k[34], fmaf(u, k[31], k[28])),
         fmaf(w, k[35], fmaf(u, k[32], k[29]))};
  }
}
// free joint: q = [p, quat xyzw]; R_pc = R0 R(quat/|quat|), t_pc = R0 p + t0.  qs = staged q rows of the joint.
__device__ __forceinline__ void free_Rt(const BodyConst& c, const float* qp, M3& R, V3& t) {
  const V3 p = ldrow3(qp);
  float x = qp[3 * W], y = qp[4 * W], z = qp[5 * W], s = qp[6 * W];
  const float n = rsqrtf(fmaf(x, x, fmaf(y, y, fmaf(z, z, s * s))));
  x *= n; y *= n; z *= n; s *= n;
  const M3 Rq = {{1.f - 2.f * (y * y + z * z), 2.f * (x * y - z * s), 2.f * (x * z + y * s),
                  2.f * (x * y + z * s), 1.f - 2.f * (x * x + z * z), 2.f * (y * z - x * s),
                  2.f * (x * z - y * s), 2.f * (y * z + x * s), 1.f - 2.f * (x * x + y * y)}};
  M3 R0;
#pragma unroll
  for (int k = 0; k < 9; ++k) R0.m[k] = c.R0[k];
  R = mul(R0, Rq);
  t = mul_acc(R0, p, V3{c.t0[0], c.t0[1], c.t0[2]});
}
// local transform of a body from the team's staged q rows
template <bool SIMPLE>
__device__ __forceinline__ void local_Rt(const BodyConst& c, const Meta& m, const float* qs, M3& R, V3& t, float& u,
                                         float& w) {
  if (m.type == BARD_JOINT_FREE) {
    u = 0.f; w = 0.f;
    free_Rt(c, qs + m.q_off * W, R, t);
    return;
  }
  if (SIMPLE || m.type == BARD_JOINT_REVOLUTE) {
    float s, co;
    sincos_fast(qs[m.q_off * W], s, co);
    u = s; w = 1.0f - co;
  } else if (m.type == BARD_JOINT_PRISMATIC) {
    u = qs[m.q_off * W]; w = 0.f;
  } else {
    u = 0.f; w = 0.f;
  }
  joint_Rt<SIMPLE>(c, m.flags, u, w, R, t);
}

// World pose of a body from its parent's (registers `cur`, a slot, or the world) -- a2.
struct Pose { M3 R; V3 p; };

__device__ __forceinline__ Pose compose_world(int src, const Pose& cur, const float* slots, const M3& R, V3 t) {
  Pose out;
  if (src == -1) {
    out.R = R;
    out.p = t;
    return out;
  }
  Pose par;
  if (src == -2) {
    par = cur;
  } else {
    const float* s = slots + src * 12 * W;
#pragma unroll
    for (int k = 0; k < 9; ++k) par.R.m[k] = s[k * W];
    par.p = ldrow3(s + 9 * W);
  }
  out.R = mul(par.R, R);
  out.p = mul_acc(par.R, t, par.p);
  return out;
}
__device__ __forceinline__ void save_pose(int save, const Pose& P, float* slots) {
  if (save >= 0) {
    float* s = slots + save * 12 * W;
#pragma unroll
    for (int k = 0; k < 9; ++k) s[k * W] = P.R.m[k];
    strow3(s + 9 * W, P.p);
  }
}

// ============================================================================= FK kernel (a1 + a2)
// team rows: q[nq] | pose slots[12 nslots]
template <bool SIMPLE>
__global__ void __launch_bounds__(256) fk_kernel(const void* __restrict__ gcommon, uint32_t cbytes, int L, int team_rows,
                                                 int nq, uint32_t B, const float* __restrict__ q,
                                                 float* __restrict__ pose) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gcommon, cbytes, nullptr, 0, L, team_rows, B, q, nq, nullptr, 0, nullptr, 0);
  const float* qs = C.st;
  float* slots = C.st + nq * W;
  const uint32_t B4 = B * 4u;
  float* out_e = pose + C.e;
  Pose cur;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) break;
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const BodyConst& c = C.bodies[i];
      const Meta m = load_meta(c);
      M3 R; V3 t; float u, w;
      local_Rt<SIMPLE>(c, m, qs, R, t, u, w);
      cur = compose_world(m.src, cur, slots, R, t);
      save_pose(m.save, cur, slots);
      if (C.valid) {
        float* o = rowptr(out_e, i * 12, B4);
#pragma unroll
        for (int j = 0; j < 9; ++j) __stcs(rowptr(o, j, B4), cur.R.m[j]);
        __stcs(rowptr(o, 9, B4), cur.p.x); __stcs(rowptr(o, 10, B4), cur.p.y); __stcs(rowptr(o, 11, B4), cur.p.z);
      }
    }
    if (tk & TASK_BAR) team_sync(C);
  }
}

// World-origin screws of a body's DOFs, s = [omega; v0] with v0 = R l + p x omega: for a revolute joint
// with T_post = I this is exactly the column [p_k x (R_k a'_k); R_k a'_k] of eq. (7).
// Stored as 6 rows per DOF at dof[(v * 6 + k) * W].
template <bool SIMPLE>
__device__ __forceinline__ void store_screws(const BodyConst& c, const Meta& m, const Pose& P, float* dof) {
  if (!SIMPLE && m.type == BARD_JOINT_FIXED) return;
  float* d = dof + m.v_off * 6 * W;
  if (m.type == BARD_JOINT_FREE) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const V3 col = {P.R.m[k], P.R.m[3 + k], P.R.m[6 + k]};   // R e_k
      float* dl = d + k * 6 * W;                               // linear DOF k: omega = 0, v0 = R e_k
      strow3(dl, {0.f, 0.f, 0.f});
      strow3(dl + 3 * W, col);
      float* da = d + (3 + k) * 6 * W;                         // angular DOF k: omega = R e_k, v0 = p x omega
      strow3(da, col);
      strow3(da + 3 * W, cross(P.p, col));
    }
    return;
  }
  const float4* p4 = reinterpret_cast<const float4*>(&c) + 9;  // Sw Sl
  const float4 a = p4[0];
  const V3 om = mul(P.R, V3{a.x, a.y, a.z});
  V3 v0 = cross(P.p, om);
  if (!SIMPLE && (!(m.flags & 1) || m.type == BARD_JOINT_PRISMATIC)) {
    const float4 b = p4[1];
    v0 = mul_acc(P.R, V3{a.w, b.x, b.y}, v0);
  }
  strow3(d, om);
  strow3(d + 3 * W, v0);
}

// Structurally zero output rows (flat row indices, list padded to a multiple of 4 with 0xffff): the team's
// warps take groups of four rows; 8 lanes x 16 bytes cover the 32 environments of one row, so one store
// instruction clears four rows.  Needs B % 4 == 0 and a 16-byte aligned output (else one row per instruction).
__device__ __forceinline__ void zero_rows(const Ctx& C, const uint16_t* zr, int nz, float* out, uint32_t B, uint32_t B4,
                                          bool vec_ok) {
  if (vec_ok) {
    const int sub = C.lane >> 3;
    const uint32_t ev = C.e - C.lane + (C.lane & 7) * 4;
    float* base = out + ev;
    const bool ok = ev < B;
    for (int g = C.w * 4; g < nz; g += C.L * 4) {
      const uint32_t row = zr[g + sub];
      if (ok && row != 0xffffu) __stcs(reinterpret_cast<float4*>(rowptr(base, row, B4)), make_float4(0.f, 0.f, 0.f, 0.f));
    }
  } else {
    float* base = out + C.e;
    for (int g = C.w; g < nz; g += C.L) {
      const uint32_t row = zr[g];
      if (C.valid && row != 0xffffu) __stcs(rowptr(base, row, B4), 0.f);
    }
  }
}

// ============================================================================= Jacobian kernel (a3)
// team rows: q[nq] | pose slots[12 nslots] | screws[6 nv] | frame origins[3 nframes]
// Phase 1: level-parallel FK over the union of the frames' ancestor paths, screws and frame origins to smem.
// Phase 2: the non-zero columns (frame, dof) are dealt round-robin to the team's warps; each writes its 6 rows.
// Phase 3: the zero rows.
template <bool SIMPLE>
__global__ void __launch_bounds__(256) jacobian_kernel(const void* __restrict__ gcommon, uint32_t cbytes,
                                                       const void* __restrict__ gj, uint32_t jbytes, int L,
                                                       int team_rows, int nq, int nv, int nslots, uint32_t B,
                                                       const float* __restrict__ q, float* __restrict__ J, int vec_ok) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gcommon, cbytes, gj, jbytes, L, team_rows, B, q, nq, nullptr, 0, nullptr, 0);
  const JHeader* JH = reinterpret_cast<const JHeader*>(C.extra);
  const FrameConst* frames = reinterpret_cast<const FrameConst*>(C.extra + sizeof(JHeader));
  const int nframes = JH->nframes;
  const float* qs = C.st;
  float* slots = C.st + nq * W;
  float* dof = slots + nslots * 12 * W;
  float* pe = dof + nv * 6 * W;
  const uint32_t jm_lo = JH->jmask_lo, jm_hi = JH->jmask_hi;
  const uint32_t B4 = B * 4u;
  Pose cur;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) break;
    const int i = tk & TASK_BODY_MASK;
    if (!(tk & TASK_NOOP) && (((i < 32 ? jm_lo : jm_hi) >> (i & 31)) & 1)) {
      const BodyConst& c = C.bodies[i];
      const Meta m = load_meta(c);
      M3 R; V3 t; float u, w;
      local_Rt<SIMPLE>(c, m, qs, R, t, u, w);
      cur = compose_world(m.src, cur, slots, R, t);
      save_pose(m.save, cur, slots);
      store_screws<SIMPLE>(c, m, cur, dof);
      for (int f = 0; f < nframes; ++f) {
        const float4 fr = *reinterpret_cast<const float4*>(&frames[f]);   // body, off[3]
        if (__float_as_int(fr.x) == i) strow3(pe + 3 * f * W, mul_acc(cur.R, V3{fr.y, fr.z, fr.w}, cur.p));
      }
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  const uint16_t* cols = reinterpret_cast<const uint16_t*>(C.extra + JH->off_cols);
  const int ncols = JH->ncols;
  float* out_e = J + C.e;
  const uint32_t nvu = nv;
  for (int idx = C.w; idx < ncols; idx += L) {
    const uint32_t cj = cols[idx];
    const uint32_t f = cj >> 8, j = cj & 255u;
    const float* d = dof + j * 6 * W;
    const V3 ang = ldrow3(d);
    const V3 lin = cross_acc(ang, ldrow3(pe + 3 * f * W), ldrow3(d + 3 * W));   // shift the world-origin column to the frame origin
    if (C.valid) {
      float* o = rowptr(out_e, f * 6 * nvu + j, B4);
      __stcs(o, lin.x); __stcs(rowptr(o, nvu, B4), lin.y); __stcs(rowptr(o, 2 * nvu, B4), lin.z);
      __stcs(rowptr(o, 3 * nvu, B4), ang.x); __stcs(rowptr(o, 4 * nvu, B4), ang.y); __stcs(rowptr(o, 5 * nvu, B4), ang.z);
    }
  }
  zero_rows(C, reinterpret_cast<const uint16_t*>(C.extra + JH->off_zrows), JH->nzrows, J, B, B4, vec_ok != 0);
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
template <bool SIMPLE>
__global__ void __launch_bounds__(256) rnea_kernel(const void* __restrict__ gcommon, uint32_t cbytes, int L, int team_rows,
                                                   int nq, int nv, int nb, int nslots, uint32_t B,
                                                   const float* __restrict__ q, const float* __restrict__ qd,
                                                   const float* __restrict__ qdd, float* __restrict__ tau) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gcommon, cbytes, nullptr, 0, L, team_rows, B, q, nq, qd, nv, qdd, nv);
  const BlobHeader* H = reinterpret_cast<const BlobHeader*>(C.common);
  const uint8_t* children = C.common + H->off_children;
  const float* qs = C.st;
  const float* qds = qs + nq * W;
  const float* qdds = qds + nv * W;
  float* slots = C.st + (nq + 2 * nv) * W;
  float* bst = slots + nslots * 12 * W;
  float* uw = bst + nb * 6 * W;
  const V3 ng = {-H->g[0], -H->g[1], -H->g[2]};
  const uint32_t B4 = B * 4u;
  V3 cvw, cvv, caw, cav;                                       // this warp's previous body: v and a
  int ntask = 0;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) { ntask = k; break; }
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const BodyConst& c = C.bodies[i];
      const Meta m = load_meta(c);
      const Inertia in = load_inertia(c);
      M3 R; V3 t; float u, w;
      local_Rt<SIMPLE>(c, m, qs, R, t, u, w);
      // joint velocity / acceleration in the body frame: S qd, S qdd
      const bool is_free = m.type == BARD_JOINT_FREE;
      const bool haslin = is_free || !SIMPLE;
      V3 vJw = {0.f, 0.f, 0.f}, vJv = vJw, aJw = vJw, aJv = vJw;
      if (is_free) {
        const float* d1 = qds + m.v_off * W;
        const float* d2 = qdds + m.v_off * W;
        vJw = ldrow3(d1 + 3 * W); vJv = ldrow3(d1);
        aJw = ldrow3(d2 + 3 * W); aJv = ldrow3(d2);
      } else if (SIMPLE || m.type != BARD_JOINT_FIXED) {
        const float qd_i = qds[m.v_off * W], qdd_i = qdds[m.v_off * W];
        vJw = qd_i * in.Sw; aJw = qdd_i * in.Sw;
        if (!SIMPLE) { vJv = qd_i * in.Sl; aJv = qdd_i * in.Sl; }
      }
      // X_up [w; v] = [R^T w ; R^T (v + w x t)]   (Pluecker motion transform with (E, r) = (R^T, t))
      V3 vw, vv, aw, av;
      if (m.src == -1) {                                       // world parent: v_p = 0, a_p = [0; -g]; v x vJ = 0
        vw = vJw; vv = vJv; aw = aJw;
        av = haslin ? mulT_acc(R, ng, aJv) : mulT(R, ng);
      } else {
        V3 pvw, pvv, paw, pav;
        if (m.src == -2) {
          pvw = cvw; pvv = cvv; paw = caw; pav = cav;
        } else {
          const float* s = slots + m.src * 12 * W;
          pvw = ldrow3(s); pvv = ldrow3(s + 3 * W); paw = ldrow3(s + 6 * W); pav = ldrow3(s + 9 * W);
        }
        vw = mulT_acc(R, pvw, vJw);
        const V3 tv = cross_acc(pvw, t, pvv);
        const V3 ta = cross_acc(paw, t, pav);
        aw = cross_acc(vw, vJw, mulT_acc(R, paw, aJw));
        if (haslin) {
          vv = mulT_acc(R, tv, vJv);
          av = cross_acc(vw, vJv, cross_acc(vv, vJw, mulT_acc(R, ta, aJv)));
        } else {
          vv = mulT(R, tv);
          av = cross_acc(vv, vJw, mulT(R, ta));
        }
      }
      // f = I a + v x* (I v),  I = (m, h, Io) about the body origin
      const V3 n1 = cross_acc(in.h, vv, symmul(in.Io, vw));
      const V3 f1 = cross_acc(vw, in.h, in.mass * vv);
      const V3 n2 = cross_acc(in.h, av, symmul(in.Io, aw));
      const V3 f2 = cross_acc(aw, in.h, in.mass * av);
      const V3 n = cross_acc(vv, f1, cross_acc(vw, n1, n2));
      const V3 f = cross_acc(vw, f1, f2);
      float* b = bst + i * 6 * W;
      strow3(b, n); strow3(b + 3 * W, f);
      uw[(2 * i) * W] = u; uw[(2 * i + 1) * W] = w;
      if (m.save >= 0) {
        float* s = slots + m.save * 12 * W;
        strow3(s, vw); strow3(s + 3 * W, vv); strow3(s + 6 * W, aw); strow3(s + 9 * W, av);
      }
      cvw = vw; cvv = vv; caw = aw; cav = av;
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  // inward pass, deepest level first: the same task list walked backwards
  float* tau_e = tau + C.e;
  for (int k = ntask - 1; k >= 0; --k) {
    const uint32_t tk = C.tasks[k];
    if ((tk & TASK_BAR) && k != ntask - 1) team_sync(C);
    if (tk & TASK_NOOP) continue;
    const int i = tk & TASK_BODY_MASK;
    const BodyConst& c = C.bodies[i];
    const Meta m = load_meta(c);
    float* b = bst + i * 6 * W;
    V3 n = ldrow3(b), f = ldrow3(b + 3 * W);
    for (int cc = 0; cc < m.child_count; ++cc) {
      const float* cb = bst + children[m.child_begin + cc] * 6 * W;
      n = n + ldrow3(cb); f = f + ldrow3(cb + 3 * W);
    }
    if (C.valid) {
      float* to = rowptr(tau_e, m.v_off, B4);
      if (m.type == BARD_JOINT_FREE) {
        __stcs(to, f.x); __stcs(rowptr(to, 1, B4), f.y); __stcs(rowptr(to, 2, B4), f.z);
        __stcs(rowptr(to, 3, B4), n.x); __stcs(rowptr(to, 4, B4), n.y); __stcs(rowptr(to, 5, B4), n.z);
      } else if (SIMPLE || m.type != BARD_JOINT_FIXED) {
        const float4* p4 = reinterpret_cast<const float4*>(&c) + 9;
        const float4 a4 = p4[0];
        float tv = dot(V3{a4.x, a4.y, a4.z}, n);
        if (!SIMPLE) { const float4 b4 = p4[1]; tv = dot_acc(V3{a4.w, b4.x, b4.y}, f, tv); }
        __stcs(to, tv);
      }
    }
    if (m.parent >= 0) {
      M3 R; V3 t;
      if (m.type == BARD_JOINT_FREE) free_Rt(c, qs + m.q_off * W, R, t);
      else joint_Rt<SIMPLE>(c, m.flags, uw[(2 * i) * W], uw[(2 * i + 1) * W], R, t);
      const V3 fp = mul(R, f);
      strow3(b, cross_acc(t, fp, mul(R, n)));
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
// Phase 3: the rows of M are dealt to the team's warps (host LPT schedule); the warp that owns row i walks
//          the set bits of rel[i] (DOFs j <= i on ancestor bodies) and writes M[i][j] and M[j][i].
// Phase 4: the structurally zero entries.  Every element of M is written exactly once.
template <bool SIMPLE>
__global__ void __launch_bounds__(256) crba_kernel(const void* __restrict__ gcommon, uint32_t cbytes, uint32_t mbytes, int L,
                                                   int team_rows, int nq, int nv, int nslots, uint32_t B,
                                                   const float* __restrict__ q, float* __restrict__ Mout, int vec_ok) {
  extern __shared__ __align__(16) unsigned char smem[];
  const Ctx C = setup(smem, gcommon, cbytes, static_cast<const unsigned char*>(gcommon) + cbytes, mbytes, L, team_rows, B,
                      q, nq, nullptr, 0, nullptr, 0);
  const BlobHeader* H = reinterpret_cast<const BlobHeader*>(C.common);
  const MHeader* MH = reinterpret_cast<const MHeader*>(C.extra);
  const uint8_t* children = C.common + H->off_children;
  const float* qs = C.st;
  float* slots = C.st + nq * W;
  float* dof = slots + nslots * 12 * W;                        // 6 rows per DOF
  float* ic = dof + nv * 6 * W;                                // 10 rows per body: m h(3) I(6)
  const uint32_t B4 = B * 4u;
  Pose cur;
  int ntask = 0;
  for (int k = 0;; ++k) {
    const uint32_t tk = C.tasks[k];
    if (tk == TASK_END) { ntask = k; break; }
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const BodyConst& c = C.bodies[i];
      const Meta m = load_meta(c);
      M3 R; V3 t; float u, w;
      local_Rt<SIMPLE>(c, m, qs, R, t, u, w);
      cur = compose_world(m.src, cur, slots, R, t);
      save_pose(m.save, cur, slots);
      store_screws<SIMPLE>(c, m, cur, dof);
      // body inertia about the world origin: h' = R h + m p ; with h'' = R h + m p / 2:
      // I' = R Io R^T + 2 (p . h'') 1 - (h'' p^T + p h''^T)
      const Inertia in = load_inertia(c);
      const float ms = in.mass;
      const V3 p = cur.p;
      const V3 hr = mul(cur.R, in.h);
      const V3 hh = axpy(0.5f * ms, p, hr);
      const V3 r0 = {cur.R.m[0], cur.R.m[1], cur.R.m[2]}, r1 = {cur.R.m[3], cur.R.m[4], cur.R.m[5]},
               r2 = {cur.R.m[6], cur.R.m[7], cur.R.m[8]};
      const V3 a0 = symmul(in.Io, r0), a1 = symmul(in.Io, r1), a2 = symmul(in.Io, r2);
      const float d = 2.f * dot(p, hh);
      float* o = ic + i * 10 * W;
      o[0] = ms;
      strow3(o + W, axpy(ms, p, hr));
      o[4 * W] = fmaf(-2.f * hh.x, p.x, dot_acc(r0, a0, d));                 // xx
      o[5 * W] = fmaf(-hh.x, p.y, fmaf(-p.x, hh.y, dot(r0, a1)));            // xy
      o[6 * W] = fmaf(-hh.x, p.z, fmaf(-p.x, hh.z, dot(r0, a2)));            // xz
      o[7 * W] = fmaf(-2.f * hh.y, p.y, dot_acc(r1, a1, d));                 // yy
      o[8 * W] = fmaf(-hh.y, p.z, fmaf(-p.y, hh.z, dot(r1, a2)));            // yz
      o[9 * W] = fmaf(-2.f * hh.z, p.z, dot_acc(r2, a2, d));                 // zz
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  // composite sweep, deepest level first
  for (int k = ntask - 1; k >= 0; --k) {
    const uint32_t tk = C.tasks[k];
    if ((tk & TASK_BAR) && k != ntask - 1) team_sync(C);
    if (tk & TASK_NOOP) continue;
    const int i = tk & TASK_BODY_MASK;
    const int2 ch = *reinterpret_cast<const int2*>(&C.bodies[i].child_begin);
    if (ch.y == 0) continue;
    float* d = ic + i * 10 * W;
    float acc[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) acc[j] = d[j * W];
    for (int cc = 0; cc < ch.y; ++cc) {
      const float* s = ic + children[ch.x + cc] * 10 * W;
#pragma unroll
      for (int j = 0; j < 10; ++j) acc[j] += s[j * W];
    }
#pragma unroll
    for (int j = 0; j < 10; ++j) d[j * W] = acc[j];
  }
  team_sync(C);
  // fill
  const uint8_t* dof_body = C.common + H->off_dof_body;
  const uint8_t* rows = C.extra + MH->off_fill + C.w * MH->fill_stride;
  const uint2* rel = reinterpret_cast<const uint2*>(C.extra + MH->off_rel);
  float* out_e = Mout + C.e;
  const uint32_t nvu = nv;
  for (int k = 0;; ++k) {
    const uint32_t i = rows[k];
    if (i == 0xffu) break;
    const float* I = ic + dof_body[i] * 10 * W;
    const float ms = I[0];
    const V3 h = ldrow3(I + W);
    const float Iw[6] = {I[4 * W], I[5 * W], I[6 * W], I[7 * W], I[8 * W], I[9 * W]};
    const float* si = dof + i * 6 * W;
    const V3 om = ldrow3(si), v0 = ldrow3(si + 3 * W);
    const V3 Fn = cross_acc(h, v0, symmul(Iw, om));          // F = I^c_i s_i  (moment about the world origin)
    const V3 Ff = cross_acc(om, h, ms * v0);                 //               (force)  m v0 - h x om
    float* rowp = rowptr(out_e, i * nvu, B4);                // M[i][.]
    float* colp = rowptr(out_e, i, B4);                      // M[.][i]
    const uint2 rm = rel[i];
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      uint32_t bits = half ? rm.y : rm.x;
      while (bits) {
        const uint32_t j = (uint32_t)(__ffs(bits) - 1) + 32u * half;
        bits &= bits - 1;
        const float* sj = dof + j * 6 * W;
        const float val = dot_acc(ldrow3(sj + 3 * W), Ff, dot(ldrow3(sj), Fn));
        if (C.valid) {
          __stcs(rowptr(rowp, j, B4), val);
          if (j != i) __stcs(rowptr(colp, j * nvu, B4), val);
        }
      }
    }
  }
  zero_rows(C, reinterpret_cast<const uint16_t*>(C.extra + MH->off_zrows), MH->nzrows, Mout, B, B4, vec_ok != 0);
}

// ----------------------------------------------------------------------------- launchers
struct LaunchCfg { int teams, threads, team_rows; size_t smem; unsigned grid; };

constexpr size_t kSmemMax = 227 * 1024;

int env_int(const char* name, int dflt) {
  const char* v = std::getenv(name);
  return v ? std::atoi(v) : dflt;
}

// TEAMS per CTA: two 32-environment teams share one copy of the constants when the team is narrow; fewer if
// the state does not fit.  Small CTAs keep the last wave short at B = 65 536 (2048 tiles over 148 SMs).
bool pick_cfg(const Model& m, int64_t B, size_t const_bytes, int team_rows, LaunchCfg& cfg) {
  const int L = m.team_warps;
  static const int want = env_int("BARD_TEAMS", 0);            // tuning knob for experiments
  int teams = want > 0 ? want : (L <= 4 ? 2 : 1);
  teams = std::max(1, std::min(teams, 8 / L));
  const size_t fixed = 16 + const_bytes;
  const size_t per_team = (size_t)team_rows * W * sizeof(float);
  while (teams > 1 && (fixed + per_team * teams) * 2 + 2048 > kSmemMax) --teams;   // keep >= 2 CTAs per SM
  cfg.teams = teams;
  cfg.threads = teams * L * 32;
  cfg.team_rows = team_rows;
  cfg.smem = fixed + per_team * teams;
  cfg.grid = (unsigned)((B + (int64_t)teams * W - 1) / ((int64_t)teams * W));
  return cfg.smem <= kSmemMax;
}

template <int ID, typename K>   // ID: one static per kernel instantiation (several kernels share a signature)
bard_status prep(K kernel, const char* name, bool fits) {
  if (!fits) { set_error(std::string(name) + ": per-environment state does not fit in shared memory"); return BARD_ERR_UNSUPPORTED; }
  static thread_local int done_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  if (done_dev != dev) {
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
    if (e == cudaSuccess)   // all of the unified L1/shared array as shared memory: occupancy is smem-bound
      e = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
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
bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

bard_status launch_fk(const Model& m, int64_t B, const float* q, float* pose, void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.common_bytes, m.nq + 12 * m.nslots, cfg);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_fk", fits);
    if (s != BARD_OK) return s;
    kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(m.d_blob, (uint32_t)m.common_bytes, m.team_warps,
                                                                      cfg.team_rows, m.nq, (uint32_t)B, q, pose);
    return finish("bard_fk");
  };
  return m.simple ? go(fk_kernel<true>, std::integral_constant<int, 0>()) : go(fk_kernel<false>, std::integral_constant<int, 1>());
}
bard_status launch_jacobian(const Model& m, int64_t B, const float* q, float* J, void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.common_bytes + m.j_bytes, m.nq + 12 * m.nslots + 6 * m.nv + 3 * m.nframes, cfg);
  const int vec_ok = (B % 4 == 0) && aligned16(J);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_jacobian", fits);
    if (s != BARD_OK) return s;
    kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(
        m.d_blob, (uint32_t)m.common_bytes, m.d_jblob, (uint32_t)m.j_bytes, m.team_warps, cfg.team_rows, m.nq, m.nv,
        m.nslots, (uint32_t)B, q, J, vec_ok);
    return finish("bard_jacobian");
  };
  return m.simple ? go(jacobian_kernel<true>, std::integral_constant<int, 2>())
                  : go(jacobian_kernel<false>, std::integral_constant<int, 3>());
}
bard_status launch_rnea(const Model& m, int64_t B, const float* q, const float* qd, const float* qdd, float* tau,
                        void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.common_bytes, m.nq + 2 * m.nv + 12 * m.nslots + 8 * m.nb, cfg);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_rnea", fits);
    if (s != BARD_OK) return s;
    kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(m.d_blob, (uint32_t)m.common_bytes, m.team_warps,
                                                                      cfg.team_rows, m.nq, m.nv, m.nb, m.nslots,
                                                                      (uint32_t)B, q, qd, qdd, tau);
    return finish("bard_rnea");
  };
  return m.simple ? go(rnea_kernel<true>, std::integral_constant<int, 4>())
                  : go(rnea_kernel<false>, std::integral_constant<int, 5>());
}
bard_status launch_crba(const Model& m, int64_t B, const float* q, float* M, void* stream) {
  LaunchCfg cfg;
  const bool fits = pick_cfg(m, B, m.common_bytes + m.m_bytes, m.nq + 12 * m.nslots + 6 * m.nv + 10 * m.nb, cfg);
  const int vec_ok = (B % 4 == 0) && aligned16(M);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_crba", fits);
    if (s != BARD_OK) return s;
    kernel<<<cfg.grid, cfg.threads, cfg.smem, (cudaStream_t)stream>>>(
        m.d_blob, (uint32_t)m.common_bytes, (uint32_t)m.m_bytes, m.team_warps, cfg.team_rows, m.nq, m.nv, m.nslots,
        (uint32_t)B, q, M, vec_ok);
    return finish("bard_crba");
  };
  return m.simple ? go(crba_kernel<true>, std::integral_constant<int, 6>())
                  : go(crba_kernel<false>, std::integral_constant<int, 7>());
}

}  // namespace bard
