// bard_rnea_vjp_params: reverse-mode derivative of RNEA with respect to the inertial parameters of every link
// (the paper's differentiability claim, "functional mode", and its use: link
// masses identified through RNEA).
//
// tau is linear in theta_i = (m, h = m c, Io) of every link i (I_i = [[Io, [h]x], [-[h]x, m 1]] is), so with the loss
// cotangent dtau the gradient is  dtheta_i = d/dtheta_i ( lambda_i^T f_i ),  f_i = I_i a_i + v_i x* I_i v_i , where
//   lambda_i = X_up lambda_parent + S_i dtau_i          (lambda_world = 0)
// is dtau pushed OUTWARD like a velocity: tau_j = S_j^T sum_{i in subtree(j)} X^T f_i, so the weight of f_i in
// sum_j dtau_j tau_j is the sum over the ancestors-or-self j of S_j dtau_j, transformed into frame i.  With
// lambda^T (v x* f) = -(v x lambda)^T f :
//   lambda^T f = B_I(lambda, a) - B_I(v x lambda, v),   B_I(x, y) = x^T I y
//   dB/dm = x_v . y_v ;  dB/dh = y_v x x_w + x_v x y_w ;  dB/dIo_ab = x_w,a y_w,b (+ b,a off the diagonal).
// Everything is local to the body once (v, a, lambda) are known: ONE outward pass (eq. (6)), no inward pass.
//
// Mapping: one thread = one environment, bodies in depth-first preorder, so a body's parent is either the body the
// thread processed just before (state still in registers) or a branching ancestor whose (v, a, lambda) were saved
// to a shared-memory slot indexed by the number of branching ancestors above it (stack discipline, [slot][18][thread]).
// Table-driven: any model, no NVRTC.  The batch reduction is deterministic: xor-butterfly over the warp, one
// shared accumulator row per warp (lane 0 adds, fixed tile order), the CTA's warps summed in ascending order into
// partials[cta][nb*10], and a second launch that sums the CTAs in ascending order in fp64.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdint>
#include <string>

#include "bard_internal.h"
#include "dfs.h"

namespace bard {
extern std::atomic<int64_t> g_launches;

namespace {

struct State { V3f vw, vv, aw, av, lw, lv; };    // velocity, acceleration, pushed cotangent: [angular; linear]

extern __shared__ __align__(16) float vsm[];

__global__ void __launch_bounds__(128) rnea_vjp_kernel(const unsigned char* __restrict__ blob, uint32_t cwords, int nb, DfsTab tab,
                                                       int nslots, uint32_t B, const float* __restrict__ q, const float* __restrict__ qd,
                                                       const float* __restrict__ qdd, const float* __restrict__ dtau,
                                                       float* __restrict__ partials) {
  // shared: [COMMON (BlobHeader | BodyConst[nb])][acc: warps x nb*10][slots: nslots x 18 x blockDim]
  float* cst = vsm;
  const int nw = blockDim.x >> 5, np = nb * 10;
  float* acc = vsm + cwords;
  float* slots = acc + nw * np;
  for (uint32_t i = threadIdx.x; i < cwords; i += blockDim.x) cst[i] = reinterpret_cast<const float*>(blob)[i];
  for (int i = threadIdx.x; i < nw * np; i += blockDim.x) acc[i] = 0.f;
  __syncthreads();
  const BlobHeader* H = reinterpret_cast<const BlobHeader*>(cst);
  const BodyConst* BC = reinterpret_cast<const BodyConst*>(cst + sizeof(BlobHeader) / 4);
  const V3f ag = {-H->g[0], -H->g[1], -H->g[2]};
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t ntiles = (B + blockDim.x - 1) / blockDim.x;
  for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const uint32_t e0 = tile * blockDim.x + threadIdx.x;
    const bool valid = e0 < B;
    const uint32_t e = valid ? e0 : B - 1;
    State cur = {};
    // the four input scalars of a one-DOF joint are loaded one body ahead of their use (the walk is one dependent chain)
    float nq = 0.f, nqd = 0.f, nqdd = 0.f, ndt = 0.f;
    auto fetch = [&](int pos) {
      if (pos >= nb) return;
      const BodyConst& n = BC[tab.order[pos]];
      if (n.type == BARD_JOINT_REVOLUTE || n.type == BARD_JOINT_PRISMATIC) {
        nq = __ldg(q + (n.q_off * B + e)); nqd = __ldg(qd + (n.v_off * B + e)); nqdd = __ldg(qdd + (n.v_off * B + e)); ndt = __ldg(dtau + (n.v_off * B + e));
      }
    };
    fetch(0);
    for (int pos = 0; pos < nb; ++pos) {
      const int i = tab.order[pos];
      const BodyConst& c = BC[i];
      const float cq = nq, cqd = nqd, cqdd = nqdd, cdt = ndt;
      fetch(pos + 1);
      const int ld = tab.load[pos];
      State P;
      if (ld == -1) P = cur;
      else if (ld == -2) { P = State{}; P.av = ag; }
      else {
        const float* s = slots + (size_t)ld * 18 * blockDim.x + threadIdx.x;
        float t[18];
#pragma unroll
        for (int k = 0; k < 18; ++k) t[k] = s[k * blockDim.x];
        P = {{t[0], t[1], t[2]}, {t[3], t[4], t[5]}, {t[6], t[7], t[8]}, {t[9], t[10], t[11]}, {t[12], t[13], t[14]}, {t[15], t[16], t[17]}};
      }
      // joint transform (eq. (4)-(5)) and the joint's own motion
      float R[9];
      V3f t;
      V3f jw = {0, 0, 0}, jv = {0, 0, 0}, bw = {0, 0, 0}, bv = {0, 0, 0}, dw = {0, 0, 0}, dv = {0, 0, 0};   // S qd, S qdd, S dtau
      if (c.type == BARD_JOINT_FREE) {
        const uint32_t qo = c.q_off * B + e, vo = c.v_off * B + e;
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
        jv = {qd[vo], qd[vo + B], qd[vo + 2 * B]};      jw = {qd[vo + 3 * B], qd[vo + 4 * B], qd[vo + 5 * B]};      // API order [linear; angular]
        bv = {qdd[vo], qdd[vo + B], qdd[vo + 2 * B]};   bw = {qdd[vo + 3 * B], qdd[vo + 4 * B], qdd[vo + 5 * B]};
        dv = {dtau[vo], dtau[vo + B], dtau[vo + 2 * B]}; dw = {dtau[vo + 3 * B], dtau[vo + 4 * B], dtau[vo + 5 * B]};
      } else {
        float u = 0.f, w = 0.f;
        if (c.type == BARD_JOINT_REVOLUTE) {
          float s, co;
          sincos_fast(cq, s, co);
          u = s; w = 1.f - co;
        } else if (c.type == BARD_JOINT_PRISMATIC) {
          u = cq;
        }
#pragma unroll
        for (int k = 0; k < 9; ++k) R[k] = fmaf(w, c.Bm[k], fmaf(u, c.A[k], c.R0[k]));
        t = {fmaf(w, c.b[0], fmaf(u, c.a[0], c.t0[0])), fmaf(w, c.b[1], fmaf(u, c.a[1], c.t0[1])), fmaf(w, c.b[2], fmaf(u, c.a[2], c.t0[2]))};
        if (c.type != BARD_JOINT_FIXED) {
          const float x = cqd, y = cqdd, z = cdt;
          const V3f Sw = {c.Sw[0], c.Sw[1], c.Sw[2]}, Sl = {c.Sl[0], c.Sl[1], c.Sl[2]};
          jw = scale(x, Sw); jv = scale(x, Sl); bw = scale(y, Sw); bv = scale(y, Sl); dw = scale(z, Sw); dv = scale(z, Sl);
        }
      }
      // X_up [w; v] = [R^T w ; R^T (v + w x t)]   (motion transform parent -> child)
      cur.vw = mulT(R, P.vw) + jw;
      cur.vv = mulT(R, P.vv + cross(P.vw, t)) + jv;
      cur.aw = mulT(R, P.aw) + bw + cross(cur.vw, jw);
      cur.av = mulT(R, P.av + cross(P.aw, t)) + bv + cross(cur.vw, jv) + cross(cur.vv, jw);
      cur.lw = mulT(R, P.lw) + dw;
      cur.lv = mulT(R, P.lv + cross(P.lw, t)) + dv;
      const int sv = tab.save[pos];
      if (sv >= 0) {
        float* s = slots + (size_t)sv * 18 * blockDim.x + threadIdx.x;
        const float tt[18] = {cur.vw.x, cur.vw.y, cur.vw.z, cur.vv.x, cur.vv.y, cur.vv.z, cur.aw.x, cur.aw.y, cur.aw.z,
                              cur.av.x, cur.av.y, cur.av.z, cur.lw.x, cur.lw.y, cur.lw.z, cur.lv.x, cur.lv.y, cur.lv.z};
#pragma unroll
        for (int k = 0; k < 18; ++k) s[k * blockDim.x] = tt[k];
      }
      // g = dB(lambda, a) - dB(u, v),  u = v x lambda (motion cross product)
      const V3f uw = cross(cur.vw, cur.lw), uv = cross(cur.vw, cur.lv) + cross(cur.vv, cur.lw);
      const V3f h1 = cross(cur.av, cur.lw) + cross(cur.lv, cur.aw), h2 = cross(cur.vv, uw) + cross(uv, cur.vw);
      float g[10];
      g[0] = dot(cur.lv, cur.av) - dot(uv, cur.vv);
      g[1] = h1.x - h2.x; g[2] = h1.y - h2.y; g[3] = h1.z - h2.z;
      const V3f xw = cur.lw, yw = cur.aw, zw = cur.vw;
      g[4] = xw.x * yw.x - uw.x * zw.x;
      g[5] = (xw.x * yw.y + xw.y * yw.x) - (uw.x * zw.y + uw.y * zw.x);
      g[6] = (xw.x * yw.z + xw.z * yw.x) - (uw.x * zw.z + uw.z * zw.x);
      g[7] = xw.y * yw.y - uw.y * zw.y;
      g[8] = (xw.y * yw.z + xw.z * yw.y) - (uw.y * zw.z + uw.z * zw.y);
      g[9] = xw.z * yw.z - uw.z * zw.z;
#pragma unroll
      for (int k = 0; k < 10; ++k) {
        float r = valid ? g[k] : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
        if (lane == 0) acc[warp * np + i * 10 + k] += r;
      }
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < np; k += blockDim.x) {
    float s = 0.f;
    for (int w = 0; w < nw; ++w) s += acc[w * np + k];
    partials[(size_t)blockIdx.x * np + k] = s;
  }
}

__global__ void vjp_reduce_kernel(const float* __restrict__ partials, int nparts, int np, float* __restrict__ out) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= np) return;
  double s = 0.0;
  for (int c = 0; c < nparts; ++c) s += (double)partials[(size_t)c * np + k];     // ascending CTA order, fp64
  out[k] = (float)s;
}

// partials[np][ncta] (the generated kernel's layout): one warp per output, lanes over the CTAs in fp64, fixed order
__global__ void vjp_reduce_columns_kernel(const float* __restrict__ partials, int ncta, int np, float* __restrict__ out) {
  const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= np) return;
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const float* p = partials + (size_t)k * ncta;
  double s = 0.0;
  for (int c = lane; c < ncta; c += 32) s += (double)p[c];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) out[k] = (float)s;
}

constexpr size_t kSmemCap = 227 * 1024;

int vjp_grid(const Model& M, int64_t B, int block) {
  const int64_t tiles = (B + block - 1) / block;
  return (int)std::min<int64_t>(tiles, (int64_t)M.sm_count * 4);
}
int vjp_block(const Model& M, int nslots) {
  const size_t cbytes = sizeof(BlobHeader) + sizeof(BodyConst) * (size_t)M.nb;
  for (int block : {128, 64, 32}) {
    const size_t smem = cbytes + (size_t)(block / 32) * M.nb * 10 * 4 + (size_t)nslots * 18 * block * 4;
    if (smem * (block >= 128 ? 2 : 1) <= kSmemCap) return block;     // two CTAs per SM where possible
  }
  return 0;
}

}  // namespace

// nb * 10 partial sums per CTA; neither kernel (this file's, the generated one of specialize.cu) runs more than
// min(tiles of 32 environments, 4 CTAs per SM) CTAs, so the size does not depend on which of them serves the call
size_t rnea_vjp_workspace_floats(const Model& M, int64_t B) {
  if (B <= 0) return 0;
  return (size_t)vjp_grid(M, B, 32) * (size_t)M.nb * 10;
}

bard_status launch_vjp_reduce_columns(const float* partials, int ncta, int np, float* dparams, void* stream) {
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)((np + 3) / 4));
  lc.blockDim = dim3(128);
  lc.stream = (cudaStream_t)stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = attr;
  lc.numAttrs = 1;
  const cudaError_t e = cudaLaunchKernelEx(&lc, vjp_reduce_columns_kernel, partials, ncta, np, dparams);
  if (e != cudaSuccess) { set_error(std::string("bard_rnea_vjp_params: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
  g_launches.fetch_add(1);
  return BARD_OK;
}

bard_status launch_rnea_vjp(const Model& M, int64_t B, const float* q, const float* qd, const float* qdd, const float* dtau,
                            float* dparams, float* ws, void* stream) {
  if ((int64_t)std::max(M.nq, M.nv) * B >= ((int64_t)1 << 32)) { set_error("bard_rnea_vjp_params: an input array has 2^32 elements or more"); return BARD_ERR_UNSUPPORTED; }
  bard_status st = BARD_OK;
  if (launch_vjp_specialized(M, B, q, qd, qdd, dtau, dparams, ws, stream, st)) return st;
  const DfsPlan P = dfs_plan(M);
  const int block = vjp_block(M, P.nslots);
  if (!block) { set_error("bard_rnea_vjp_params: per-environment state does not fit in shared memory"); return BARD_ERR_UNSUPPORTED; }
  const int grid = vjp_grid(M, B, block), np = M.nb * 10;
  const uint32_t cwords = (uint32_t)((sizeof(BlobHeader) + sizeof(BodyConst) * (size_t)M.nb) / 4);
  const size_t smem = (size_t)cwords * 4 + (size_t)(block / 32) * np * 4 + (size_t)P.nslots * 18 * block * 4;
  static thread_local int done_dev = -1;
  int dev = 0;
  cudaGetDevice(&dev);
  if (done_dev != dev) {
    cudaError_t e = cudaFuncSetAttribute(rnea_vjp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemCap);
    if (e != cudaSuccess) { set_error(std::string("bard_rnea_vjp_params: ") + cudaGetErrorString(e)); cudaGetLastError(); return BARD_ERR_CUDA; }
    done_dev = dev;
  }
  rnea_vjp_kernel<<<grid, block, smem, (cudaStream_t)stream>>>((const unsigned char*)M.d_blob, cwords, M.nb, P.tab, P.nslots, (uint32_t)B, q, qd,
                                                               qdd, dtau, ws);
  vjp_reduce_kernel<<<(np + 127) / 128, 128, 0, (cudaStream_t)stream>>>(ws, grid, np, dparams);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_error(std::string("bard_rnea_vjp_params: ") + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
  g_launches.fetch_add(2);
  return BARD_OK;
}

}  // namespace bard
