// sm_100a kernels for the four operators.  One thread evaluates one environment; a warp's 32 environments
// are adjacent in memory (SoA, batch fastest), so every global load/store instruction moves one full
// 128-byte line per warp.  The model constant blob (a few KB, identical for all envs) is staged into
// shared memory once per CTA with a TMA bulk copy (cp.async.bulk + mbarrier) and is then read with
// warp-uniform (broadcast) shared loads.  Per-environment state that must survive across bodies lives
// in shared-memory columns  state[slot][tid]  (bank-conflict free); everything else stays in registers.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "bard_internal.h"

namespace bard {

extern std::atomic<int64_t> g_launches;

namespace {

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

// ----------------------------------------------------------------------------- constant staging (TMA bulk copy)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Copies `bytes` (multiple of 16) of the model blob from global to shared memory with one
// cp.async.bulk issued by thread 0 and completed on an mbarrier; every thread waits on the barrier.
__device__ __forceinline__ void stage_blob(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  const uint32_t bar_a = smem_u32(bar);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(bar_a)
                 : "memory");
  }
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
#pragma unroll
  for (int k = 0; k < 9; ++k) R.m[k] = fmaf(w, c.Bm[k], fmaf(u, c.A[k], c.R0[k]));
  if (c.flags & 1) {
    t = {fmaf(u, c.a[0], c.t0[0]), fmaf(u, c.a[1], c.t0[1]), fmaf(u, c.a[2], c.t0[2])};  // revolute: a = 0
  } else {
    t = {fmaf(w, c.b[0], fmaf(u, c.a[0], c.t0[0])), fmaf(w, c.b[1], fmaf(u, c.a[1], c.t0[1])),
         fmaf(w, c.b[2], fmaf(u, c.a[2], c.t0[2]))};
  }
}
// free joint: q = [p, quat xyzw]; R_pc = R0 R(quat/|quat|), t_pc = R0 p + t0
__device__ __forceinline__ void free_Rt(const BodyConst& c, const float* __restrict__ q, int64_t B, int64_t e, M3& R,
                                        V3& t) {
  const float* qp = q + (int64_t)c.q_off * B + e;
  V3 p = {qp[0], qp[B], qp[2 * B]};
  float x = qp[3 * B], y = qp[4 * B], z = qp[5 * B], s = qp[6 * B];
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
// local transform of body i for env e
__device__ __forceinline__ void local_Rt(const BodyConst& c, const float* __restrict__ q, int64_t B, int64_t e, M3& R,
                                         V3& t, float& u, float& w) {
  if (c.type == BARD_JOINT_FREE) {
    u = 0.f; w = 0.f;
    free_Rt(c, q, B, e, R, t);
  } else {
    float qv = (c.type == BARD_JOINT_FIXED) ? 0.f : q[(int64_t)c.q_off * B + e];
    joint_uw(c.type, qv, u, w);
    joint_Rt(c, u, w, R, t);
  }
}

struct Smem {
  const BlobHeader* H;
  const BodyConst* bodies;
  const FrameConst* frames;
  float* state;   // [nstate][blockDim.x]
};

__device__ __forceinline__ Smem setup_smem(unsigned char* smem, const void* gblob, uint32_t blob_bytes) {
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem);
  unsigned char* dst = smem + 16;
  stage_blob(dst, gblob, blob_bytes, bar);
  Smem s;
  s.H = reinterpret_cast<const BlobHeader*>(dst);
  s.bodies = reinterpret_cast<const BodyConst*>(dst + sizeof(BlobHeader));
  s.frames = reinterpret_cast<const FrameConst*>(dst + sizeof(BlobHeader) + sizeof(BodyConst) * s.H->nb);
  s.state = reinterpret_cast<float*>(dst + blob_bytes);
  return s;
}

// World pose of body i from its parent's (registers `cur`, a slot, or the world) -- a2.
struct Pose { M3 R; V3 p; };

__device__ __forceinline__ Pose compose_world(const BodyConst& c, const Pose& cur, const float* slots, int T,
                                              const M3& R, V3 t) {
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
    const float* s = slots + (size_t)c.src * 12 * T;
#pragma unroll
    for (int k = 0; k < 9; ++k) par.R.m[k] = s[k * T];
    par.p = {s[9 * T], s[10 * T], s[11 * T]};
  }
  out.R = mul(par.R, R);
  out.p = mul(par.R, t) + par.p;
  return out;
}
__device__ __forceinline__ void save_pose(const BodyConst& c, const Pose& P, float* slots, int T) {
  if (c.save >= 0) {
    float* s = slots + (size_t)c.save * 12 * T;
#pragma unroll
    for (int k = 0; k < 9; ++k) s[k * T] = P.R.m[k];
    s[9 * T] = P.p.x; s[10 * T] = P.p.y; s[11 * T] = P.p.z;
  }
}

// ============================================================================= FK kernel
__global__ void __launch_bounds__(128) fk_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int64_t B,
                                                 const float* __restrict__ q, float* __restrict__ pose) {
  extern __shared__ __align__(16) unsigned char smem[];
  Smem S = setup_smem(smem, gblob, blob_bytes);
  const int T = blockDim.x;
  const int64_t e = (int64_t)blockIdx.x * T + threadIdx.x;
  if (e >= B) return;
  float* slots = S.state + threadIdx.x;
  const int nb = S.H->nb;
  Pose cur;
  for (int i = 0; i < nb; ++i) {
    const BodyConst& c = S.bodies[i];
    M3 R; V3 t; float u, w;
    local_Rt(c, q, B, e, R, t, u, w);
    cur = compose_world(c, cur, slots, T, R, t);
    save_pose(c, cur, slots, T);
    float* o = pose + (int64_t)i * 12 * B + e;
#pragma unroll
    for (int k = 0; k < 9; ++k) __stcs(o + k * B, cur.R.m[k]);
    __stcs(o + 9 * B, cur.p.x); __stcs(o + 10 * B, cur.p.y); __stcs(o + 11 * B, cur.p.z);
  }
}


// World-origin screws of body i's DOFs, s = [omega; v0] with v0 = R l + p x omega: for a revolute joint
// with T_post = I this is exactly the column [p_k x (R_k a'_k); R_k a'_k] of eq. (7).
// Stored as 6 floats per DOF at dof[(v*6 + k) * T].
__device__ __forceinline__ void store_screws(const BodyConst& c, const Pose& P, float* dof, int T) {
  if (c.type == BARD_JOINT_FIXED) return;
  float* d = dof + (size_t)c.v_off * 6 * T;
  if (c.type == BARD_JOINT_FREE) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      V3 col = {P.R.m[k], P.R.m[3 + k], P.R.m[6 + k]};   // R e_k
      float* dl = d + (size_t)k * 6 * T;                 // linear DOF k: omega = 0, v0 = R e_k
      dl[0] = 0.f; dl[T] = 0.f; dl[2 * T] = 0.f; dl[3 * T] = col.x; dl[4 * T] = col.y; dl[5 * T] = col.z;
      float* da = d + (size_t)(3 + k) * 6 * T;           // angular DOF k: omega = R e_k, v0 = p x omega
      V3 v0 = cross(P.p, col);
      da[0] = col.x; da[T] = col.y; da[2 * T] = col.z; da[3 * T] = v0.x; da[4 * T] = v0.y; da[5 * T] = v0.z;
    }
    return;
  }
  V3 om = mul(P.R, ld3(c.Sw));
  V3 v0 = cross(P.p, om);
  if (!(c.flags & 1) || c.type == BARD_JOINT_PRISMATIC) v0 = v0 + mul(P.R, ld3(c.Sl));
  d[0] = om.x; d[T] = om.y; d[2 * T] = om.z; d[3 * T] = v0.x; d[4 * T] = v0.y; d[5 * T] = v0.z;
}
__device__ __forceinline__ int dof_count(int type) {
  return type == BARD_JOINT_FREE ? 6 : (type == BARD_JOINT_FIXED ? 0 : 1);
}

// ============================================================================= Jacobian kernel (a3)
__global__ void __launch_bounds__(128) jacobian_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int64_t B,
                                                       const float* __restrict__ q, float* __restrict__ J) {
  extern __shared__ __align__(16) unsigned char smem[];
  Smem S = setup_smem(smem, gblob, blob_bytes);
  const int T = blockDim.x;
  const int64_t e = (int64_t)blockIdx.x * T + threadIdx.x;
  if (e >= B) return;
  const int nb = S.H->nb, nv = S.H->nv, nframes = S.H->nframes;
  float* slots = S.state + threadIdx.x;
  float* dof = slots + (size_t)S.H->nslots * 12 * T;
  float* pe = dof + (size_t)nv * 6 * T;                       // frame origins, 3 floats per frame
  const uint64_t jmask = ((uint64_t)(uint32_t)S.H->jac_mask_hi << 32) | (uint32_t)S.H->jac_mask_lo;
  Pose cur;
  for (int i = 0; i < nb; ++i) {
    if (!((jmask >> i) & 1)) continue;                        // only the union of the frames' ancestor paths
    const BodyConst& c = S.bodies[i];
    M3 R; V3 t; float u, w;
    local_Rt(c, q, B, e, R, t, u, w);
    cur = compose_world(c, cur, slots, T, R, t);
    save_pose(c, cur, slots, T);
    store_screws(c, cur, dof, T);
    for (int f = 0; f < nframes; ++f) {
      if (S.frames[f].body == i) {
        V3 p = cur.p + mul(cur.R, ld3(S.frames[f].off));
        pe[(3 * f) * T] = p.x; pe[(3 * f + 1) * T] = p.y; pe[(3 * f + 2) * T] = p.z;
      }
    }
  }
  for (int f = 0; f < nframes; ++f) {
    const FrameConst& fc = S.frames[f];
    const uint64_t anc = ((uint64_t)fc.anc_hi << 32) | fc.anc_lo;
    const V3 p = {pe[(3 * f) * T], pe[(3 * f + 1) * T], pe[(3 * f + 2) * T]};
    float* Jf = J + (int64_t)f * 6 * nv * B + e;
    for (int i = 0; i < nb; ++i) {
      const BodyConst& c = S.bodies[i];
      const int nd = dof_count(c.type);
      const bool on_path = (anc >> i) & 1;
      for (int k = 0; k < nd; ++k) {
        const int j = c.v_off + k;
        V3 lin = {0.f, 0.f, 0.f}, ang = {0.f, 0.f, 0.f};
        if (on_path) {
          const float* d = dof + (size_t)j * 6 * T;
          ang = {d[0], d[T], d[2 * T]};
          V3 v0 = {d[3 * T], d[4 * T], d[5 * T]};
          lin = v0 + cross(ang, p);                           // shift the world-origin column to the frame origin
        }
        float* o = Jf + (int64_t)j * B;
        const int64_t rs = (int64_t)nv * B;
        __stcs(o, lin.x); __stcs(o + rs, lin.y); __stcs(o + 2 * rs, lin.z);
        __stcs(o + 3 * rs, ang.x); __stcs(o + 4 * rs, ang.y); __stcs(o + 5 * rs, ang.z);
      }
    }
  }
}


// ============================================================================= RNEA kernel (a4 + a5)
// Body-frame recursion, internal order [angular; linear].  Outward: v, a of the parent come from the
// registers of the previous body, a shared-memory slot, or the world (v = 0, a = -g: gravity trick).
// The net body force f_i and the two joint scalars (u, w) are parked in shared memory (8 floats per body);
// the inward pass rebuilds T_pc from (u, w) with eq. (4)-(5) instead of keeping 12 floats per body.
struct Motion { V3 w, v; };   // [angular; linear]

__global__ void __launch_bounds__(128) rnea_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int64_t B,
                                                   const float* __restrict__ q, const float* __restrict__ qd,
                                                   const float* __restrict__ qdd, float* __restrict__ tau) {
  extern __shared__ __align__(16) unsigned char smem[];
  Smem S = setup_smem(smem, gblob, blob_bytes);
  const int T = blockDim.x;
  const int64_t e = (int64_t)blockIdx.x * T + threadIdx.x;
  if (e >= B) return;
  const int nb = S.H->nb;
  float* slots = S.state + threadIdx.x;                        // 12 floats per slot: v.w v.v a.w a.v
  float* bst = slots + (size_t)S.H->nslots * 12 * T;           // 8 floats per body: n(3) f(3) u w
  const V3 g = ld3(S.H->g);
  Motion cv, ca;                                               // previous body's velocity / acceleration
  for (int i = 0; i < nb; ++i) {
    const BodyConst& c = S.bodies[i];
    M3 R; V3 t; float u, w;
    local_Rt(c, q, B, e, R, t, u, w);
    Motion pv, pa;
    if (c.src == -1) {
      pv = {{0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}};
      pa = {{0.f, 0.f, 0.f}, {-g.x, -g.y, -g.z}};
    } else if (c.src == -2) {
      pv = cv; pa = ca;
    } else {
      const float* s = slots + (size_t)c.src * 12 * T;
      pv = {{s[0], s[T], s[2 * T]}, {s[3 * T], s[4 * T], s[5 * T]}};
      pa = {{s[6 * T], s[7 * T], s[8 * T]}, {s[9 * T], s[10 * T], s[11 * T]}};
    }
    // joint velocity / acceleration in the body frame: S qd, S qdd
    Motion vJ = {{0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}}, aJ = vJ;
    if (c.type == BARD_JOINT_FREE) {
      const float* d1 = qd + (int64_t)c.v_off * B + e;
      const float* d2 = qdd + (int64_t)c.v_off * B + e;
      vJ = {{d1[3 * B], d1[4 * B], d1[5 * B]}, {d1[0], d1[B], d1[2 * B]}};
      aJ = {{d2[3 * B], d2[4 * B], d2[5 * B]}, {d2[0], d2[B], d2[2 * B]}};
    } else if (c.type != BARD_JOINT_FIXED) {
      const float qd_i = qd[(int64_t)c.v_off * B + e], qdd_i = qdd[(int64_t)c.v_off * B + e];
      const V3 sw = ld3(c.Sw), sl = ld3(c.Sl);
      vJ = {qd_i * sw, qd_i * sl};
      aJ = {qdd_i * sw, qdd_i * sl};
    }
    // X_up [w; v] = [R^T w ; R^T (v + w x t)]   (Pluecker motion transform with (E, r) = (R^T, t))
    Motion v, a;
    v.w = mulT(R, pv.w) + vJ.w;
    v.v = mulT(R, pv.v + cross(pv.w, t)) + vJ.v;
    a.w = mulT(R, pa.w) + aJ.w + cross(v.w, vJ.w);
    a.v = mulT(R, pa.v + cross(pa.w, t)) + aJ.v + cross(v.w, vJ.v) + cross(v.v, vJ.w);
    // f = I a + v x* (I v),  I = (m, h, Io) about the body origin
    const V3 h = ld3(c.h);
    const float m = c.mass;
    const V3 n1 = symmul(c.Io, v.w) + cross(h, v.v);
    const V3 f1 = m * v.v - cross(h, v.w);
    const V3 n2 = symmul(c.Io, a.w) + cross(h, a.v);
    const V3 f2 = m * a.v - cross(h, a.w);
    const V3 n = n2 + cross(v.w, n1) + cross(v.v, f1);
    const V3 f = f2 + cross(v.w, f1);
    float* b = bst + (size_t)i * 8 * T;
    b[0] = n.x; b[T] = n.y; b[2 * T] = n.z; b[3 * T] = f.x; b[4 * T] = f.y; b[5 * T] = f.z;
    b[6 * T] = u; b[7 * T] = w;
    if (c.save >= 0) {
      float* s = slots + (size_t)c.save * 12 * T;
      s[0] = v.w.x; s[T] = v.w.y; s[2 * T] = v.w.z; s[3 * T] = v.v.x; s[4 * T] = v.v.y; s[5 * T] = v.v.z;
      s[6 * T] = a.w.x; s[7 * T] = a.w.y; s[8 * T] = a.w.z; s[9 * T] = a.v.x; s[10 * T] = a.v.y; s[11 * T] = a.v.z;
    }
    cv = v; ca = a;
  }
  // inward pass: tau_i = S_i^T f_i ; f_parent += X_up^T f_i, children in descending index order
  for (int i = nb - 1; i >= 0; --i) {
    const BodyConst& c = S.bodies[i];
    const float* b = bst + (size_t)i * 8 * T;
    const V3 n = {b[0], b[T], b[2 * T]}, f = {b[3 * T], b[4 * T], b[5 * T]};
    float* to = tau + (int64_t)c.v_off * B + e;
    if (c.type == BARD_JOINT_FREE) {
      __stcs(to, f.x); __stcs(to + B, f.y); __stcs(to + 2 * B, f.z);
      __stcs(to + 3 * B, n.x); __stcs(to + 4 * B, n.y); __stcs(to + 5 * B, n.z);
    } else if (c.type != BARD_JOINT_FIXED) {
      __stcs(to, dot(ld3(c.Sw), n) + dot(ld3(c.Sl), f));
    }
    if (c.parent >= 0) {
      M3 R; V3 t;
      if (c.type == BARD_JOINT_FREE) free_Rt(c, q, B, e, R, t);
      else joint_Rt(c, b[6 * T], b[7 * T], R, t);
      const V3 fp = mul(R, f);
      const V3 np = mul(R, n) + cross(t, fp);
      float* pb = bst + (size_t)c.parent * 8 * T;
      pb[0] += np.x; pb[T] += np.y; pb[2 * T] += np.z; pb[3 * T] += fp.x; pb[4 * T] += fp.y; pb[5 * T] += fp.z;
    }
  }
}


// ============================================================================= CRBA kernel (a6 + a7)
// World-frame formulation: every composite inertia is expressed about the WORLD origin in world axes
// (m, h, I: 10 floats), so the backward sweep  I^c_parent += X^T I^c_child X degenerates to
// ten additions (X = identity between world-frame quantities), and M_ij = s_j . (I^c_i s_i) for every
// ancestor DOF j needs no transform along the walk.  The screws s are the eq. (7) columns (store_screws).
__global__ void __launch_bounds__(128) crba_kernel(const void* __restrict__ gblob, uint32_t blob_bytes, int64_t B,
                                                   const float* __restrict__ q, float* __restrict__ Mout) {
  extern __shared__ __align__(16) unsigned char smem[];
  Smem S = setup_smem(smem, gblob, blob_bytes);
  const int T = blockDim.x;
  const int64_t e = (int64_t)blockIdx.x * T + threadIdx.x;
  if (e >= B) return;
  const int nb = S.H->nb, nv = S.H->nv;
  float* slots = S.state + threadIdx.x;
  float* dof = slots + (size_t)S.H->nslots * 12 * T;           // 6 floats per DOF
  float* ic = dof + (size_t)nv * 6 * T;                        // 10 floats per body: m h(3) I(6)
  Pose cur;
  for (int i = 0; i < nb; ++i) {
    const BodyConst& c = S.bodies[i];
    M3 R; V3 t; float u, w;
    local_Rt(c, q, B, e, R, t, u, w);
    cur = compose_world(c, cur, slots, T, R, t);
    save_pose(c, cur, slots, T);
    store_screws(c, cur, dof, T);
    // body inertia about the world origin: h' = R h + m p ; with h'' = R h + m p / 2:
    // I' = R Io R^T + 2 (p . h'') 1 - (h'' p^T + p h''^T)
    const float m = c.mass;
    const V3 hr = mul(cur.R, ld3(c.h));
    const V3 p = cur.p;
    const V3 hh = hr + (0.5f * m) * p;
    // R Io R^T (symmetric): columns of Io R^T are Io * (rows of R)
    const V3 r0 = {cur.R.m[0], cur.R.m[1], cur.R.m[2]}, r1 = {cur.R.m[3], cur.R.m[4], cur.R.m[5]},
             r2 = {cur.R.m[6], cur.R.m[7], cur.R.m[8]};
    const V3 a0 = symmul(c.Io, r0), a1 = symmul(c.Io, r1), a2 = symmul(c.Io, r2);
    const float d = 2.f * dot(p, hh);
    float* o = ic + (size_t)i * 10 * T;
    o[0] = m;
    o[T] = hr.x + m * p.x; o[2 * T] = hr.y + m * p.y; o[3 * T] = hr.z + m * p.z;
    o[4 * T] = dot(r0, a0) + d - 2.f * hh.x * p.x;             // xx
    o[5 * T] = dot(r0, a1) - (hh.x * p.y + p.x * hh.y);        // xy
    o[6 * T] = dot(r0, a2) - (hh.x * p.z + p.x * hh.z);        // xz
    o[7 * T] = dot(r1, a1) + d - 2.f * hh.y * p.y;             // yy
    o[8 * T] = dot(r1, a2) - (hh.y * p.z + p.y * hh.z);        // yz
    o[9 * T] = dot(r2, a2) + d - 2.f * hh.z * p.z;             // zz
  }
  // composite sweep, children into parents in descending index order
  for (int i = nb - 1; i > 0; --i) {
    const int par = S.bodies[i].parent;
    if (par < 0) continue;
    const float* s = ic + (size_t)i * 10 * T;
    float* d = ic + (size_t)par * 10 * T;
#pragma unroll
    for (int k = 0; k < 10; ++k) d[k * T] += s[k * T];
  }
  // fill: row DOF i, column DOF j <= i; both M[i][j] and M[j][i] are written here, exactly once each
  for (int bi = 0; bi < nb; ++bi) {
    const BodyConst& ci = S.bodies[bi];
    const int ndi = dof_count(ci.type);
    if (ndi == 0) continue;
    const uint64_t anc = ((uint64_t)ci.anc_hi << 32) | ci.anc_lo;
    const float* I = ic + (size_t)bi * 10 * T;
    const float m = I[0];
    const V3 h = {I[T], I[2 * T], I[3 * T]};
    const float Iw[6] = {I[4 * T], I[5 * T], I[6 * T], I[7 * T], I[8 * T], I[9 * T]};
    for (int ki = 0; ki < ndi; ++ki) {
      const int i = ci.v_off + ki;
      const float* si = dof + (size_t)i * 6 * T;
      const V3 om = {si[0], si[T], si[2 * T]}, v0 = {si[3 * T], si[4 * T], si[5 * T]};
      const V3 Fn = symmul(Iw, om) + cross(h, v0);             // F = I^c_i s_i  (moment about the world origin)
      const V3 Ff = m * v0 - cross(h, om);                     //               (force)
      for (int bj = 0; bj <= bi; ++bj) {
        const BodyConst& cj = S.bodies[bj];
        const int ndj = dof_count(cj.type);
        const bool rel = (anc >> bj) & 1;
        for (int kj = 0; kj < ndj; ++kj) {
          const int j = cj.v_off + kj;
          if (j > i) break;
          float val = 0.f;
          if (rel) {
            const float* sj = dof + (size_t)j * 6 * T;
            const V3 oj = {sj[0], sj[T], sj[2 * T]}, vj = {sj[3 * T], sj[4 * T], sj[5 * T]};
            val = dot(oj, Fn) + dot(vj, Ff);
          }
          __stcs(Mout + ((int64_t)i * nv + j) * B + e, val);
          if (j != i) __stcs(Mout + ((int64_t)j * nv + i) * B + e, val);
        }
      }
    }
  }
}

// ----------------------------------------------------------------------------- launchers
struct LaunchCfg { int threads; size_t smem; };

// Largest CTA (<= 128 threads, multiple of 32) such that at least `want_ctas` CTAs fit in one SM's shared memory.
LaunchCfg pick_cfg(const Model& m, size_t state_floats_per_thread) {
  const size_t fixed = 16 + m.blob_bytes;
  const size_t sm_budget = 227 * 1024;
  int best = 32;
  for (int t : {128, 64, 32}) {
    size_t need = fixed + state_floats_per_thread * 4 * t + 1024;   // +1 KB driver reservation per CTA
    if (need * 2 <= sm_budget || t == 32) { best = t; break; }
  }
  return {best, fixed + state_floats_per_thread * 4 * best};
}

template <typename K>
bard_status prep(K kernel, const LaunchCfg& cfg, const char* name) {
  if (cfg.smem > 227 * 1024) { set_error(std::string(name) + ": model state does not fit in shared memory"); return BARD_ERR_UNSUPPORTED; }
  if (cfg.smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
    if (e != cudaSuccess) { set_error(std::string(name) + ": " + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
  }
  return BARD_OK;
}
bard_status finish(const char* name) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_error(std::string(name) + ": " + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
  g_launches.fetch_add(1);
  return BARD_OK;
}
unsigned grid_for(int64_t B, int threads) { return (unsigned)((B + threads - 1) / threads); }

}  // namespace

bard_status launch_fk(const Model& m, int64_t B, const float* q, float* pose, void* stream) {
  LaunchCfg cfg = pick_cfg(m, (size_t)m.nslots * 12);
  bard_status s = prep(fk_kernel, cfg, "bard_fk");
  if (s != BARD_OK) return s;
  fk_kernel<<<grid_for(B, cfg.threads), cfg.threads, cfg.smem, (cudaStream_t)stream>>>(m.d_blob, (uint32_t)m.blob_bytes, B, q, pose);
  return finish("bard_fk");
}
bard_status launch_jacobian(const Model& m, int64_t B, const float* q, float* J, void* stream) {
  LaunchCfg cfg = pick_cfg(m, (size_t)m.nslots * 12 + (size_t)m.nv * 6 + (size_t)m.nframes * 3);
  bard_status s = prep(jacobian_kernel, cfg, "bard_jacobian");
  if (s != BARD_OK) return s;
  jacobian_kernel<<<grid_for(B, cfg.threads), cfg.threads, cfg.smem, (cudaStream_t)stream>>>(m.d_blob, (uint32_t)m.blob_bytes, B, q, J);
  return finish("bard_jacobian");
}
bard_status launch_rnea(const Model& m, int64_t B, const float* q, const float* qd, const float* qdd, float* tau,
                        void* stream) {
  LaunchCfg cfg = pick_cfg(m, (size_t)m.nslots * 12 + (size_t)m.nb * 8);
  bard_status s = prep(rnea_kernel, cfg, "bard_rnea");
  if (s != BARD_OK) return s;
  rnea_kernel<<<grid_for(B, cfg.threads), cfg.threads, cfg.smem, (cudaStream_t)stream>>>(m.d_blob, (uint32_t)m.blob_bytes, B, q, qd, qdd, tau);
  return finish("bard_rnea");
}
bard_status launch_crba(const Model& m, int64_t B, const float* q, float* M, void* stream) {
  LaunchCfg cfg = pick_cfg(m, (size_t)m.nslots * 12 + (size_t)m.nv * 6 + (size_t)m.nb * 10);
  bard_status s = prep(crba_kernel, cfg, "bard_crba");
  if (s != BARD_OK) return s;
  crba_kernel<<<grid_for(B, cfg.threads), cfg.threads, cfg.smem, (cudaStream_t)stream>>>(m.d_blob, (uint32_t)m.blob_bytes, B, q, M);
  return finish("bard_crba");
}

}  // namespace bard
