// Table-driven ABA (forward dynamics, the paper's fifth operator: PAPER.md:37, 91, 125) for models that were not
// specialised with BARD_OP_ABA -- any model, no NVRTC, a free joint anywhere in the tree (missing 4).
//
// Featherstone's three passes (RBDA table 7.1), body frames, [angular; linear], one thread per environment:
//   pass 1 (outward, depth-first preorder): v_i = X v_p + S qd ; c_i = v_i x S qd ; p^A_i = v_i x* I_i v_i ; I^A_i = I_i
//   pass 2 (inward, reverse preorder):      U = I^A S ; D = S^T U ; u = tau - S^T p^A ;
//        I^a = I^A - U D^-1 U^T ; p^a = p^A + I^a c + U D^-1 u ; I^A_parent += X^T I^a X (block form of the "bottleneck
//        6x6 update" of PAPER.md:103: rotate the three 3x3 blocks, translate) ; p^A_parent += X^T p^a
//   pass 3 (outward): a' = X a_p + c ; qdd = D^-1 (u - U^T a') ; a = a' + S qdd            (a_world = -g)
// A 6-DOF joint (S = 1_6) transmits nothing to its parent but the applied wrench: I^a = 0, p^a = tau, and its body's
// acceleration is a = (I^A)^-1 (tau - p^A) whatever the parent does (LDL^T, 6x6); qdd = a - a'.
//
// Per-body state lives in the caller's workspace, SoA rows [48 nb][B] (row = 48 body + k): v 0..5, c 6..11, I^A 12..32
// (A: 6 symmetric, H: 9, M: 6 symmetric of I^A = [[A, H], [H^T, M]]), p^A 33..38, U 39..44 (a free joint: its a), D^-1 45,
// u 46.  Every row is written and read back by the same thread; a child adds into its parent's rows (read-modify-write, the
// children of a body in reverse preorder, i.e. a fixed order: deterministic).  The generated kernel (specialize.cu) keeps all
// of this on chip; this one trades ~12 KB of workspace traffic per environment for needing no compiler (humanoid at B = 65 536: 406 us against 61 us).
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <string>

#include "bard_internal.h"
#include "dfs.h"

namespace bard {
extern std::atomic<int64_t> g_launches;

namespace {

constexpr int kRows = 48;
extern __shared__ __align__(16) float asm_[];

struct Sym3 { float xx, xy, xz, yy, yz, zz; };
__device__ __forceinline__ V3f mul(const Sym3& s, V3f v) {
  return {fmaf(s.xz, v.z, fmaf(s.xy, v.y, s.xx * v.x)), fmaf(s.yz, v.z, fmaf(s.yy, v.y, s.xy * v.x)), fmaf(s.zz, v.z, fmaf(s.yz, v.y, s.xz * v.x))};
}
__device__ __forceinline__ V3f mulH(const float* H, V3f v) {          // H v (row-major 3x3)
  return {fmaf(H[2], v.z, fmaf(H[1], v.y, H[0] * v.x)), fmaf(H[5], v.z, fmaf(H[4], v.y, H[3] * v.x)), fmaf(H[8], v.z, fmaf(H[7], v.y, H[6] * v.x))};
}
__device__ __forceinline__ V3f mulHT(const float* H, V3f v) {         // H^T v
  return {fmaf(H[6], v.z, fmaf(H[3], v.y, H[0] * v.x)), fmaf(H[7], v.z, fmaf(H[4], v.y, H[1] * v.x)), fmaf(H[8], v.z, fmaf(H[5], v.y, H[2] * v.x))};
}
// R S R^T for a symmetric S (given as full 3x3 in m) -> symmetric
__device__ __forceinline__ Sym3 rot_sym(const float* R, const Sym3& s) {
  const float S[9] = {s.xx, s.xy, s.xz, s.xy, s.yy, s.yz, s.xz, s.yz, s.zz};
  float RS[9];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) RS[3 * a + b] = fmaf(R[3 * a + 2], S[6 + b], fmaf(R[3 * a + 1], S[3 + b], R[3 * a] * S[b]));
  auto e = [&](int a, int b) { return fmaf(RS[3 * a + 2], R[3 * b + 2], fmaf(RS[3 * a + 1], R[3 * b + 1], RS[3 * a] * R[3 * b])); };
  return {e(0, 0), e(0, 1), e(0, 2), e(1, 1), e(1, 2), e(2, 2)};
}
__device__ __forceinline__ void rot_gen(const float* R, const float* H, float* out) {      // R H R^T
  float RH[9];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) RH[3 * a + b] = fmaf(R[3 * a + 2], H[6 + b], fmaf(R[3 * a + 1], H[3 + b], R[3 * a] * H[b]));
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) out[3 * a + b] = fmaf(RH[3 * a + 2], R[3 * b + 2], fmaf(RH[3 * a + 1], R[3 * b + 1], RH[3 * a] * R[3 * b]));
}

struct Joint { float R[9]; V3f t; };
// the joint transform of body c from q (as pass 1 computed it: same expressions, same bits)
__device__ __forceinline__ void joint_of(const BodyConst& c, const float* __restrict__ q, uint32_t B, uint32_t e, Joint& J) {
  if (c.type == BARD_JOINT_FREE) { free_Rt(c, q, c.q_off * B + e, B, J.R, J.t); return; }
  float u = 0.f, w = 0.f;
  if (c.type == BARD_JOINT_REVOLUTE) {
    float s, co;
    sincos_fast(q[c.q_off * B + e], s, co);
    u = s; w = 1.f - co;
  } else if (c.type == BARD_JOINT_PRISMATIC) {
    u = q[c.q_off * B + e];
  }
  joint_Rt_uw(c, u, w, J.R, J.t);
}

__global__ void __launch_bounds__(128) aba_generic_kernel(const unsigned char* __restrict__ blob, uint32_t cwords, int nb, DfsTab tab, uint32_t B,
                                                          const float* __restrict__ q, const float* __restrict__ qd,
                                                          const float* __restrict__ tau, float* __restrict__ qdd, float* __restrict__ ws) {
  // shared: [COMMON (BlobHeader | BodyConst[nb])][slots: nslots x 6 x blockDim]
  float* cst = asm_;
  float* slots = asm_ + cwords;
  for (uint32_t i = threadIdx.x; i < cwords; i += blockDim.x) cst[i] = reinterpret_cast<const float*>(blob)[i];
  __syncthreads();
  const BlobHeader* Hd = reinterpret_cast<const BlobHeader*>(cst);
  const BodyConst* BC = reinterpret_cast<const BodyConst*>(cst + sizeof(BlobHeader) / 4);
  const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= B) return;                                       // (no barrier below)
  auto W = [&](int body, int k) -> float& { return ws[((size_t)(kRows * body + k)) * B + e]; };
  auto slot = [&](int s, int k) -> float& { return slots[((size_t)s * 6 + k) * blockDim.x + threadIdx.x]; };

  // ---- pass 1
  V3f cw_ = {0, 0, 0}, cv_ = {0, 0, 0};                     // state of the previous body: its velocity
  for (int pos = 0; pos < nb; ++pos) {
    const int i = tab.order[pos];
    const BodyConst& c = BC[i];
    V3f pw = {0, 0, 0}, pv = {0, 0, 0};
    const int ld = tab.load[pos];
    if (ld == -1) { pw = cw_; pv = cv_; }
    else if (ld >= 0) { pw = {slot(ld, 0), slot(ld, 1), slot(ld, 2)}; pv = {slot(ld, 3), slot(ld, 4), slot(ld, 5)}; }
    Joint J;
    joint_of(c, q, B, e, J);
    V3f jw = {0, 0, 0}, jv = {0, 0, 0};
    if (c.type == BARD_JOINT_FREE) {
      const uint32_t vo = c.v_off * B + e;
      jv = {qd[vo], qd[vo + B], qd[vo + 2 * B]}; jw = {qd[vo + 3 * B], qd[vo + 4 * B], qd[vo + 5 * B]};
    } else if (c.type != BARD_JOINT_FIXED) {
      const float x = qd[c.v_off * B + e];
      jw = scale(x, V3f{c.Sw[0], c.Sw[1], c.Sw[2]}); jv = scale(x, V3f{c.Sl[0], c.Sl[1], c.Sl[2]});
    }
    const V3f vw = mulT(J.R, pw) + jw, vv = mulT(J.R, pv + cross(pw, J.t)) + jv;
    const V3f ccw = cross(vw, jw), ccv = cross(vw, jv) + cross(vv, jw);
    // I v and p^A = v x* (I v) with I = (m, h, Io)
    const V3f h = {c.h[0], c.h[1], c.h[2]};
    const Sym3 Io = {c.Io[0], c.Io[1], c.Io[2], c.Io[3], c.Io[4], c.Io[5]};
    const V3f n1 = mul(Io, vw) + cross(h, vv), f1 = scale(c.mass, vv) - cross(h, vw);
    const V3f pn = cross(vw, n1) + cross(vv, f1), pf = cross(vw, f1);
    const float vals[39] = {vw.x, vw.y, vw.z, vv.x, vv.y, vv.z, ccw.x, ccw.y, ccw.z, ccv.x, ccv.y, ccv.z,
                            Io.xx, Io.xy, Io.xz, Io.yy, Io.yz, Io.zz,                         // A
                            0.f, -h.z, h.y, h.z, 0.f, -h.x, -h.y, h.x, 0.f,                 // H = [h]x
                            c.mass, 0.f, 0.f, c.mass, 0.f, c.mass,                           // M
                            pn.x, pn.y, pn.z, pf.x, pf.y, pf.z};
#pragma unroll
    for (int k = 0; k < 39; ++k) W(i, k) = vals[k];
    const int sv = tab.save[pos];
    if (sv >= 0) { slot(sv, 0) = vw.x; slot(sv, 1) = vw.y; slot(sv, 2) = vw.z; slot(sv, 3) = vv.x; slot(sv, 4) = vv.y; slot(sv, 5) = vv.z; }
    cw_ = vw; cv_ = vv;
  }

  // ---- pass 2
  for (int pos = nb - 1; pos >= 0; --pos) {
    const int i = tab.order[pos];
    const BodyConst& c = BC[i];
    Sym3 A = {W(i, 12), W(i, 13), W(i, 14), W(i, 15), W(i, 16), W(i, 17)};
    float H[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) H[k] = W(i, 18 + k);
    Sym3 M = {W(i, 27), W(i, 28), W(i, 29), W(i, 30), W(i, 31), W(i, 32)};
    V3f pn = {W(i, 33), W(i, 34), W(i, 35)}, pf = {W(i, 36), W(i, 37), W(i, 38)};
    const V3f ccw = {W(i, 6), W(i, 7), W(i, 8)}, ccv = {W(i, 9), W(i, 10), W(i, 11)};
    if (c.type == BARD_JOINT_FREE) {
      // a = (I^A)^-1 (tau - p^A) by LDL^T of the dense 6x6; the parent receives I^a = 0, p^a = tau
      const uint32_t vo = c.v_off * B + e;
      const V3f tf = {tau[vo], tau[vo + B], tau[vo + 2 * B]}, tn = {tau[vo + 3 * B], tau[vo + 4 * B], tau[vo + 5 * B]};   // API: [force; moment]
      float Am[6][6];
      const float As[9] = {A.xx, A.xy, A.xz, A.xy, A.yy, A.yz, A.xz, A.yz, A.zz}, Ms[9] = {M.xx, M.xy, M.xz, M.xy, M.yy, M.yz, M.xz, M.yz, M.zz};
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) { Am[a][b] = As[3 * a + b]; Am[a][3 + b] = H[3 * a + b]; Am[3 + a][b] = H[3 * b + a]; Am[3 + a][3 + b] = Ms[3 * a + b]; }
      float rhs[6] = {tn.x - pn.x, tn.y - pn.y, tn.z - pn.z, tf.x - pf.x, tf.y - pf.y, tf.z - pf.z};
      float L[6][6], d[6];
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        float s = Am[j][j];
#pragma unroll
        for (int k = 0; k < 6; ++k) if (k < j) s = fmaf(-L[j][k] * d[k], L[j][k], s);
        d[j] = s;
        const float inv = 1.f / s;
#pragma unroll
        for (int r = 0; r < 6; ++r) if (r > j) {
          float t = Am[r][j];
#pragma unroll
          for (int k = 0; k < 6; ++k) if (k < j) t = fmaf(-L[r][k] * d[k], L[j][k], t);
          L[r][j] = t * inv;
        }
      }
#pragma unroll
      for (int r = 0; r < 6; ++r)
#pragma unroll
        for (int k = 0; k < 6; ++k) if (k < r) rhs[r] = fmaf(-L[r][k], rhs[k], rhs[r]);
#pragma unroll
      for (int r = 0; r < 6; ++r) rhs[r] /= d[r];
#pragma unroll
      for (int r = 5; r >= 0; --r)
#pragma unroll
        for (int k = 0; k < 6; ++k) if (k > r) rhs[r] = fmaf(-L[k][r], rhs[k], rhs[r]);
#pragma unroll
      for (int k = 0; k < 6; ++k) W(i, 39 + k) = rhs[k];
      A = {0, 0, 0, 0, 0, 0}; M = A;
#pragma unroll
      for (int k = 0; k < 9; ++k) H[k] = 0.f;
      pn = tn; pf = tf;
    } else if (c.type != BARD_JOINT_FIXED) {
      const V3f sw = {c.Sw[0], c.Sw[1], c.Sw[2]}, sl = {c.Sl[0], c.Sl[1], c.Sl[2]};
      const V3f Uw = mul(A, sw) + mulH(H, sl), Ul = mulHT(H, sw) + mul(M, sl);
      const float D = dot(sw, Uw) + dot(sl, Ul), Dinv = 1.f / D;
      const float u = tau[c.v_off * B + e] - dot(sw, pn) - dot(sl, pf);
      W(i, 39) = Uw.x; W(i, 40) = Uw.y; W(i, 41) = Uw.z; W(i, 42) = Ul.x; W(i, 43) = Ul.y; W(i, 44) = Ul.z; W(i, 45) = Dinv; W(i, 46) = u;
      if (c.parent >= 0) {
        const V3f dw = scale(Dinv, Uw), dl = scale(Dinv, Ul);
        A = {A.xx - dw.x * Uw.x, A.xy - dw.x * Uw.y, A.xz - dw.x * Uw.z, A.yy - dw.y * Uw.y, A.yz - dw.y * Uw.z, A.zz - dw.z * Uw.z};
        M = {M.xx - dl.x * Ul.x, M.xy - dl.x * Ul.y, M.xz - dl.x * Ul.z, M.yy - dl.y * Ul.y, M.yz - dl.y * Ul.z, M.zz - dl.z * Ul.z};
        const float uw3[3] = {dw.x, dw.y, dw.z}, ul3[3] = {Ul.x, Ul.y, Ul.z};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
          for (int b = 0; b < 3; ++b) H[3 * a + b] = fmaf(-uw3[a], ul3[b], H[3 * a + b]);
        const float k = Dinv * u;
        pn = pn + mul(A, ccw) + mulH(H, ccv) + scale(k, Uw);
        pf = pf + mulHT(H, ccw) + mul(M, ccv) + scale(k, Ul);
      }
    } else if (c.parent >= 0) {                              // fixed joint: nothing is removed (c = 0)
      pn = pn + mul(A, ccw) + mulH(H, ccv);
      pf = pf + mulHT(H, ccw) + mul(M, ccv);
    }
    if (c.parent < 0) continue;
    // X^T I^a X and X^T p^a into the parent's rows: rotate, translate
    Joint J;
    joint_of(c, q, B, e, J);
    const Sym3 A1 = rot_sym(J.R, A), M1 = rot_sym(J.R, M);
    float H1[9], Hp[9];
    rot_gen(J.R, H, H1);
    const float Mf[9] = {M1.xx, M1.xy, M1.xz, M1.xy, M1.yy, M1.yz, M1.xz, M1.yz, M1.zz};
#pragma unroll
    for (int j = 0; j < 3; ++j) {                            // H_p[:, j] = H'[:, j] + t x M'[:, j]
      const V3f cj = cross(J.t, V3f{Mf[j], Mf[3 + j], Mf[6 + j]});
      Hp[j] = H1[j] + cj.x; Hp[3 + j] = H1[3 + j] + cj.y; Hp[6 + j] = H1[6 + j] + cj.z;
    }
    V3f uu[3], wwv[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      uu[k] = cross(J.t, V3f{H1[3 * k], H1[3 * k + 1], H1[3 * k + 2]});       // (-H' [t]x)[k, :]
      wwv[k] = cross(J.t, V3f{Hp[3 * k], Hp[3 * k + 1], Hp[3 * k + 2]});      // ([t]x H_p^T)[:, k]
    }
    const float u0[3] = {uu[0].x, uu[0].y, uu[0].z}, u1[3] = {uu[1].x, uu[1].y, uu[1].z}, u2[3] = {uu[2].x, uu[2].y, uu[2].z};
    const float w0[3] = {wwv[0].x, wwv[0].y, wwv[0].z}, w1[3] = {wwv[1].x, wwv[1].y, wwv[1].z}, w2[3] = {wwv[2].x, wwv[2].y, wwv[2].z};
    const float Ap[6] = {A1.xx + u0[0] + w0[0], A1.xy + u0[1] + w1[0], A1.xz + u0[2] + w2[0], A1.yy + u1[1] + w1[1], A1.yz + u1[2] + w2[1],
                         A1.zz + u2[2] + w2[2]};
    const V3f fp = mulR(J.R, pf), np_ = mulR(J.R, pn) + cross(J.t, fp);
    const int p = c.parent;
#pragma unroll
    for (int k = 0; k < 6; ++k) W(p, 12 + k) += Ap[k];
#pragma unroll
    for (int k = 0; k < 9; ++k) W(p, 18 + k) += Hp[k];
    W(p, 27) += M1.xx; W(p, 28) += M1.xy; W(p, 29) += M1.xz; W(p, 30) += M1.yy; W(p, 31) += M1.yz; W(p, 32) += M1.zz;
    W(p, 33) += np_.x; W(p, 34) += np_.y; W(p, 35) += np_.z; W(p, 36) += fp.x; W(p, 37) += fp.y; W(p, 38) += fp.z;
  }

  // ---- pass 3
  V3f aw_ = {0, 0, 0}, av_ = {0, 0, 0};
  const V3f ag = {-Hd->g[0], -Hd->g[1], -Hd->g[2]};
  for (int pos = 0; pos < nb; ++pos) {
    const int i = tab.order[pos];
    const BodyConst& c = BC[i];
    V3f pw = {0, 0, 0}, pv = ag;
    const int ld = tab.load[pos];
    if (ld == -1) { pw = aw_; pv = av_; }
    else if (ld >= 0) { pw = {slot(ld, 0), slot(ld, 1), slot(ld, 2)}; pv = {slot(ld, 3), slot(ld, 4), slot(ld, 5)}; }
    Joint J;
    joint_of(c, q, B, e, J);
    V3f aw = mulT(J.R, pw) + V3f{W(i, 6), W(i, 7), W(i, 8)}, av = mulT(J.R, pv + cross(pw, J.t)) + V3f{W(i, 9), W(i, 10), W(i, 11)};   // a' = X a_p + c
    if (c.type == BARD_JOINT_FREE) {
      const V3f bw = {W(i, 39), W(i, 40), W(i, 41)}, bv = {W(i, 42), W(i, 43), W(i, 44)};
      const uint32_t vo = c.v_off * B + e;
      qdd[vo] = bv.x - av.x; qdd[vo + B] = bv.y - av.y; qdd[vo + 2 * B] = bv.z - av.z;                  // API order [linear; angular]
      qdd[vo + 3 * B] = bw.x - aw.x; qdd[vo + 4 * B] = bw.y - aw.y; qdd[vo + 5 * B] = bw.z - aw.z;
      aw = bw; av = bv;
    } else if (c.type != BARD_JOINT_FIXED) {
      const V3f Uw = {W(i, 39), W(i, 40), W(i, 41)}, Ul = {W(i, 42), W(i, 43), W(i, 44)};
      const float a = W(i, 45) * (W(i, 46) - dot(Uw, aw) - dot(Ul, av));
      qdd[c.v_off * B + e] = a;
      aw = aw + scale(a, V3f{c.Sw[0], c.Sw[1], c.Sw[2]});
      av = av + scale(a, V3f{c.Sl[0], c.Sl[1], c.Sl[2]});
    }
    const int sv = tab.save[pos];
    if (sv >= 0) { slot(sv, 0) = aw.x; slot(sv, 1) = aw.y; slot(sv, 2) = aw.z; slot(sv, 3) = av.x; slot(sv, 4) = av.y; slot(sv, 5) = av.z; }
    aw_ = aw; av_ = av;
  }
}

constexpr size_t kSmemCapA = 227 * 1024;

}  // namespace

size_t aba_generic_workspace_floats(const Model& M, int64_t B) { return B > 0 ? (size_t)kRows * (size_t)M.nb * (size_t)B : 0; }

bard_status launch_aba_generic(const Model& M, int64_t B, const float* q, const float* qd, const float* tau, float* qdd, float* ws, void* stream) {
  if ((int64_t)kRows * M.nb * B >= ((int64_t)1 << 32) || (int64_t)std::max(M.nq, M.nv) * B >= ((int64_t)1 << 32)) {
    set_error("bard_aba: an array (the workspace: 48 nb B floats) has 2^32 elements or more");
    return BARD_ERR_UNSUPPORTED;
  }
  const DfsPlan P = dfs_plan(M);
  const uint32_t cwords = (uint32_t)((sizeof(BlobHeader) + sizeof(BodyConst) * (size_t)M.nb) / 4);
  const int block = 128;
  const size_t smem = (size_t)cwords * 4 + (size_t)P.nslots * 6 * block * 4;
  if (smem > kSmemCapA) { set_error("bard_aba: per-environment state does not fit in shared memory"); return BARD_ERR_UNSUPPORTED; }
  static thread_local int done_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  if (done_dev != dev) {
    cudaError_t e = cudaFuncSetAttribute(aba_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemCapA);
    if (e != cudaSuccess) { set_error(std::string("bard_aba: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
    done_dev = dev;
  }
  aba_generic_kernel<<<(unsigned)((B + block - 1) / block), block, smem, (cudaStream_t)stream>>>((const unsigned char*)M.d_blob, cwords, M.nb, P.tab,
                                                                                                (uint32_t)B, q, qd, tau, qdd, ws);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_error(std::string("bard_aba: ") + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
  g_launches.fetch_add(1);
  return BARD_OK;
}

}  // namespace bard
