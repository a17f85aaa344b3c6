// What the table-driven one-thread-per-environment kernels share (vjp.cu, aba_generic.cu): the depth-first preorder
// walk of the tree with its parent-state slots, 3-vector helpers, the kernels' sincos and the joint transform read from
// the BodyConst table (eq. (4)-(5)).
//
// Walk: bodies in depth-first preorder, so a body's parent is either the body the thread processed just before (state
// still in registers) or a branching ancestor whose state was saved to a slot indexed by the number of branching
// ancestors above it (stack discipline).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <vector>

#include "bard_internal.h"

namespace bard {
namespace {

struct DfsTab {
  uint8_t order[BARD_MAX_BODIES];     // depth-first preorder
  int8_t load[BARD_MAX_BODIES];       // per position: -2 world, -1 registers (parent = previous position), >= 0 slot
  int8_t save[BARD_MAX_BODIES];       // per position: slot to save (v, a, lambda) to, -1 none
};

struct V3f { float x, y, z; };
__device__ __forceinline__ V3f operator+(V3f a, V3f b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ V3f cross(V3f a, V3f b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
__device__ __forceinline__ float dot(V3f a, V3f b) { return fmaf(a.z, b.z, fmaf(a.y, b.y, a.x * b.x)); }
__device__ __forceinline__ V3f scale(float s, V3f a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ V3f mulT(const float* R, V3f v) {        // R^T v
  return {fmaf(R[6], v.z, fmaf(R[3], v.y, R[0] * v.x)), fmaf(R[7], v.z, fmaf(R[4], v.y, R[1] * v.x)), fmaf(R[8], v.z, fmaf(R[5], v.y, R[2] * v.x))};
}

// same reduction and polynomials as kernels.cu / the generated kernels (reading 16)
__device__ __forceinline__ void sincos_fast(float x, float& s, float& c) {
  const float kb = fmaf(x, 0.636619772367581343f, 12582912.0f);
  const float k = kb - 12582912.0f;
  const int qd = __float_as_int(kb);
  float r = fmaf(k, -1.57079637050628662109375f, x);
  r = fmaf(k, 4.371138828673793e-8f, r);
  r = fmaf(k, 1.7151245100058819e-15f, r);
  const float r2 = r * r;
  float ps = fmaf(r2, -1.9515295891e-4f, 8.3321608736e-3f);
  ps = fmaf(ps, r2, -1.6666654611e-1f);
  ps = fmaf(ps * r2, r, r);
  float pc = fmaf(r2, 2.443315711809948e-5f, -1.388731625493765e-3f);
  pc = fmaf(pc, r2, 4.166664568298827e-2f);
  pc = fmaf(pc * r2, r2, fmaf(r2, -0.5f, 1.0f));
  const float ss = (qd & 1) ? pc : ps;
  const float cc = (qd & 1) ? ps : pc;
  s = __int_as_float(__float_as_int(ss) ^ ((qd & 2) << 30));
  c = __int_as_float(__float_as_int(cc) ^ (((qd + 1) & 2) << 30));
}


// R_pc, t_pc of a one-DOF or fixed joint from the joint scalars (u, w) = (sin q, 1 - cos q) / (q, 0) / (0, 0)
__device__ __forceinline__ void joint_Rt_uw(const BodyConst& c, float u, float w, float* R, V3f& t) {
#pragma unroll
  for (int k = 0; k < 9; ++k) R[k] = fmaf(w, c.Bm[k], fmaf(u, c.A[k], c.R0[k]));
  t = {fmaf(w, c.b[0], fmaf(u, c.a[0], c.t0[0])), fmaf(w, c.b[1], fmaf(u, c.a[1], c.t0[1])), fmaf(w, c.b[2], fmaf(u, c.a[2], c.t0[2]))};
}
// free joint: q = [p, quat xyzw] (normalised here); R_pc = R0 R(quat), t_pc = R0 p + t0
__device__ __forceinline__ void free_Rt(const BodyConst& c, const float* __restrict__ q, uint32_t qo, uint32_t B, float* R, V3f& t) {
  const V3f p = {q[qo], q[qo + B], q[qo + 2 * B]};
  float x = q[qo + 3 * B], y = q[qo + 4 * B], z = q[qo + 5 * B], s = q[qo + 6 * B];
  const float n = rsqrtf(fmaf(x, x, fmaf(y, y, fmaf(z, z, s * s))));
  x *= n; y *= n; z *= n; s *= n;
  const float Rq[9] = {1.f - 2.f * (y * y + z * z), 2.f * (x * y - z * s), 2.f * (x * z + y * s),
                       2.f * (x * y + z * s), 1.f - 2.f * (x * x + z * z), 2.f * (y * z - x * s),
                       2.f * (x * z - y * s), 2.f * (y * z + x * s), 1.f - 2.f * (x * x + y * y)};
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) R[3 * a + b] = fmaf(c.R0[3 * a + 2], Rq[6 + b], fmaf(c.R0[3 * a + 1], Rq[3 + b], c.R0[3 * a] * Rq[b]));
  t = {fmaf(c.R0[2], p.z, fmaf(c.R0[1], p.y, fmaf(c.R0[0], p.x, c.t0[0]))), fmaf(c.R0[5], p.z, fmaf(c.R0[4], p.y, fmaf(c.R0[3], p.x, c.t0[1]))),
       fmaf(c.R0[8], p.z, fmaf(c.R0[7], p.y, fmaf(c.R0[6], p.x, c.t0[2])))};
}
__device__ __forceinline__ V3f mulR(const float* R, V3f v) {         // R v
  return {fmaf(R[2], v.z, fmaf(R[1], v.y, R[0] * v.x)), fmaf(R[5], v.z, fmaf(R[4], v.y, R[3] * v.x)), fmaf(R[8], v.z, fmaf(R[7], v.y, R[6] * v.x))};
}
__device__ __forceinline__ V3f operator-(V3f a, V3f b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }

struct DfsPlan { DfsTab tab; int nslots; };

inline DfsPlan dfs_plan(const Model& M) {
  DfsPlan P = {};
  std::vector<std::vector<int>> ch(M.nb);
  for (int i = 0; i < M.nb; ++i)
    if (M.parent[i] >= 0) ch[M.parent[i]].push_back(i);
  std::vector<int> slot_of(M.nb, -1);
  int pos = 0, prev = -1, maxslot = 0;
  // iterative preorder; `depth` = number of branching proper ancestors
  struct Item { int body, depth; };
  std::vector<Item> stack;
  for (int r = M.nb - 1; r >= 0; --r)
    if (M.parent[r] < 0) stack.push_back({r, 0});
  while (!stack.empty()) {
    const Item it = stack.back();
    stack.pop_back();
    const int i = it.body, p = M.parent[i];
    P.tab.order[pos] = (uint8_t)i;
    P.tab.load[pos] = (int8_t)(p < 0 ? -2 : (p == prev ? -1 : slot_of[p]));
    const bool branching = ch[i].size() >= 2;
    P.tab.save[pos] = -1;
    if (branching) { slot_of[i] = it.depth; P.tab.save[pos] = (int8_t)it.depth; maxslot = std::max(maxslot, it.depth + 1); }
    for (int k = (int)ch[i].size() - 1; k >= 0; --k) stack.push_back({ch[i][k], it.depth + (branching ? 1 : 0)});
    prev = i;
    ++pos;
  }
  P.nslots = maxslot;
  return P;
}


}  // namespace
}  // namespace bard
