// sm_100a kernels for the four operators -- level-parallel team schedule, N environments per lane.
//
// Mapping.  A TEAM of L warps evaluates one TILE of 32 N environments (N = 1 or 2): lane l owns the N adjacent
// environments e0 + N l ... so the 32 lanes of every warp touch 32 N adjacent floats of one SoA row (batch
// fastest): every global or shared load/store instruction moves one or two full 128-byte lines, and with
// N = 2 every memory instruction, every address computation, every constant load and every piece of control
// flow is shared by two environments (the kernels are bound by instruction issue, not by DRAM).
// The bodies of one tree level (eq. (6)) are spread over the team's L warps by the host
// schedule (model.cu); whole warps work on different bodies of the same environments, so there is no
// divergence and an idle warp costs no issue slots.  Warps of a team meet at a named barrier (bar.sync id,
// 32 L) between levels and exchange per-environment state through shared-memory rows state[row][32 N]
// (bank-conflict free); a body that continues on its parent's warp reads it from registers.
// A CTA holds TEAMS teams that share one copy of the model constants.
//
// Staging.  The model constant sections (a few KB, identical for all environments) are copied into shared
// memory once per CTA with TMA bulk copies (cp.async.bulk + mbarrier) and read with warp-uniform (broadcast)
// 16-byte loads.  The team's input rows (q, and qd / qdd for RNEA) are staged with cp.async (LDGSTS) so that
// all input lines are in flight at once instead of one DRAM round trip per body.
//
// Stores.  Output rows are B floats apart (B is a run-time value).  Element indices row * B + e are kept in
// 32 bits (the C ABI refuses outputs of 2^32 elements or more), so a store address costs one IMAD and one
// IMAD.WIDE; structurally zero rows of J and M are written by a separate pass with 16-byte stores.
//
// Every kernel is instantiated for SIMPLE models (every joint is a revolute joint with T_post = I or a free
// joint -- all BASELINE configs) and for general ones (prismatic / fixed joints, T_post != I).
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <type_traits>

#include "bard_internal.h"

namespace bard {

extern std::atomic<int64_t> g_launches;

namespace {

// ----------------------------------------------------------------------------- scalar packs
// f2: the same quantity for the lane's two environments, kept in one aligned 64-bit register pair so that the
// arithmetic maps onto Blackwell's packed FP32 instructions (PTX add / mul / fma .f32x2 -> SASS FADD2 / FMUL2 /
// FFMA2): one issue slot does the work of two, and the kernels are bound by instruction issue.  A plain float
// converts to an f2 with both halves equal (a model constant: FFMA2 reads it as a broadcast `.F32` operand, no
// extra instruction), so mixed expressions need no extra overloads.
struct f2 {
  unsigned long long v;
  __device__ __forceinline__ f2() {}
  __device__ __forceinline__ f2(float x, float y) { asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(x), "f"(y)); }
  __device__ __forceinline__ f2(float s) : f2(s, s) {}
  __device__ __forceinline__ float lo() const { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
  __device__ __forceinline__ float hi() const { return __uint_as_float((unsigned)(v >> 32)); }
};
__device__ __forceinline__ f2 operator-(f2 x) { return {-x.lo(), -x.hi()}; }     // folds into an operand modifier
__device__ __forceinline__ f2 operator+(f2 x, f2 y) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(x.v), "l"(y.v)); return r; }
__device__ __forceinline__ f2 operator-(f2 x, f2 y) { return x + (-y); }
__device__ __forceinline__ f2 operator*(f2 x, f2 y) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(x.v), "l"(y.v)); return r; }
__device__ __forceinline__ float fm(float x, float y, float z) { return fmaf(x, y, z); }
__device__ __forceinline__ f2 fm(f2 x, f2 y, f2 z) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(x.v), "l"(y.v), "l"(z.v)); return r; }
__device__ __forceinline__ float rsq(float x) { return rsqrtf(x); }
__device__ __forceinline__ f2 rsq(f2 x) { return {rsqrtf(x.lo()), rsqrtf(x.hi())}; }

template <int N> struct Pack { using T = float; };
template <> struct Pack<2> { using T = f2; };

// ----------------------------------------------------------------------------- small vector algebra
// Written as fused multiply-add chains: acc + R v, acc + a x b, ... so that almost every FP instruction
// is an FFMA.  Operands may be per-environment (T) or warp-uniform model constants (float).
template <class T> struct V3 { T x, y, z; };
template <class T> struct M3 { T m[9]; };   // row-major
template <class A, class B> using Mix = typename std::conditional<std::is_same<A, f2>::value || std::is_same<B, f2>::value, f2, float>::type;

template <class A, class B>
__device__ __forceinline__ V3<Mix<A, B>> operator+(V3<A> a, V3<B> b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
template <class S, class A>
__device__ __forceinline__ V3<Mix<S, A>> scale(S s, V3<A> a) { return {s * a.x, s * a.y, s * a.z}; }
template <class S, class A, class C>
__device__ __forceinline__ V3<Mix<Mix<S, A>, C>> axpy(S s, V3<A> a, V3<C> acc) {      // acc + s a
  return {fm(s, a.x, acc.x), fm(s, a.y, acc.y), fm(s, a.z, acc.z)};
}
template <class A, class B>
__device__ __forceinline__ V3<Mix<A, B>> cross(V3<A> a, V3<B> b) {
  return {fm(a.y, b.z, -(a.z * b.y)), fm(a.z, b.x, -(a.x * b.z)), fm(a.x, b.y, -(a.y * b.x))};
}
template <class A, class B, class C>
__device__ __forceinline__ V3<Mix<Mix<A, B>, C>> cross_acc(V3<A> a, V3<B> b, V3<C> acc) {    // acc + a x b
  return {fm(-a.z, b.y, fm(a.y, b.z, acc.x)), fm(-a.x, b.z, fm(a.z, b.x, acc.y)), fm(-a.y, b.x, fm(a.x, b.y, acc.z))};
}
template <class A, class B>
__device__ __forceinline__ Mix<A, B> dot(V3<A> a, V3<B> b) { return fm(a.z, b.z, fm(a.y, b.y, a.x * b.x)); }
template <class A, class B, class C>
__device__ __forceinline__ Mix<Mix<A, B>, C> dot_acc(V3<A> a, V3<B> b, C acc) {
  return fm(a.z, b.z, fm(a.y, b.y, fm(a.x, b.x, acc)));
}
template <class A, class B>
__device__ __forceinline__ V3<Mix<A, B>> mul(const M3<A>& R, V3<B> v) {           // R v
  return {fm(R.m[2], v.z, fm(R.m[1], v.y, R.m[0] * v.x)), fm(R.m[5], v.z, fm(R.m[4], v.y, R.m[3] * v.x)),
          fm(R.m[8], v.z, fm(R.m[7], v.y, R.m[6] * v.x))};
}
template <class A, class B, class C>
__device__ __forceinline__ V3<Mix<Mix<A, B>, C>> mul_acc(const M3<A>& R, V3<B> v, V3<C> acc) {   // acc + R v
  return {fm(R.m[2], v.z, fm(R.m[1], v.y, fm(R.m[0], v.x, acc.x))), fm(R.m[5], v.z, fm(R.m[4], v.y, fm(R.m[3], v.x, acc.y))),
          fm(R.m[8], v.z, fm(R.m[7], v.y, fm(R.m[6], v.x, acc.z)))};
}
template <class A, class B>
__device__ __forceinline__ V3<Mix<A, B>> mulT(const M3<A>& R, V3<B> v) {          // R^T v
  return {fm(R.m[6], v.z, fm(R.m[3], v.y, R.m[0] * v.x)), fm(R.m[7], v.z, fm(R.m[4], v.y, R.m[1] * v.x)),
          fm(R.m[8], v.z, fm(R.m[5], v.y, R.m[2] * v.x))};
}
template <class A, class B, class C>
__device__ __forceinline__ V3<Mix<Mix<A, B>, C>> mulT_acc(const M3<A>& R, V3<B> v, V3<C> acc) {  // acc + R^T v
  return {fm(R.m[6], v.z, fm(R.m[3], v.y, fm(R.m[0], v.x, acc.x))), fm(R.m[7], v.z, fm(R.m[4], v.y, fm(R.m[1], v.x, acc.y))),
          fm(R.m[8], v.z, fm(R.m[5], v.y, fm(R.m[2], v.x, acc.z)))};
}
template <class A, class B>
__device__ __forceinline__ M3<Mix<A, B>> mul(const M3<A>& a, const M3<B>& b) {
  M3<Mix<A, B>> c;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      c.m[3 * i + j] = fm(a.m[3 * i + 2], b.m[6 + j], fm(a.m[3 * i + 1], b.m[3 + j], a.m[3 * i] * b.m[j]));
  return c;
}
// symmetric 3x3 (xx,xy,xz,yy,yz,zz) times vector
template <class A, class B>
__device__ __forceinline__ V3<Mix<A, B>> symmul(const A* I, V3<B> v) {
  return {fm(I[2], v.z, fm(I[1], v.y, I[0] * v.x)), fm(I[4], v.z, fm(I[3], v.y, I[1] * v.x)),
          fm(I[5], v.z, fm(I[4], v.y, I[2] * v.x))};
}

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
__device__ __forceinline__ void sincos_fast(f2 x, f2& s, f2& c) {
  // same arithmetic as the scalar version, the FP part in packed form; the quadrant logic stays per half
  const f2 kb = fm(x, f2(0.636619772367581343f), f2(12582912.0f));
  const f2 k = kb + f2(-12582912.0f);
  const int q0 = __float_as_int(kb.lo()), q1 = __float_as_int(kb.hi());
  f2 r = fm(k, f2(-1.57079637050628662109375f), x);
  r = fm(k, f2(4.371138828673793e-8f), r);
  r = fm(k, f2(1.7151245100058819e-15f), r);
  const f2 r2 = r * r;
  f2 ps = fm(r2, f2(-1.9515295891e-4f), f2(8.3321608736e-3f));
  ps = fm(ps, r2, f2(-1.6666654611e-1f));
  ps = fm(ps * r2, r, r);
  f2 pc = fm(r2, f2(2.443315711809948e-5f), f2(-1.388731625493765e-3f));
  pc = fm(pc, r2, f2(4.166664568298827e-2f));
  pc = fm(pc * r2, r2, fm(r2, f2(-0.5f), f2(1.0f)));
  const float ss0 = (q0 & 1) ? pc.lo() : ps.lo(), cc0 = (q0 & 1) ? ps.lo() : pc.lo();
  const float ss1 = (q1 & 1) ? pc.hi() : ps.hi(), cc1 = (q1 & 1) ? ps.hi() : pc.hi();
  s = {__int_as_float(__float_as_int(ss0) ^ ((q0 & 2) << 30)), __int_as_float(__float_as_int(ss1) ^ ((q1 & 2) << 30))};
  c = {__int_as_float(__float_as_int(cc0) ^ (((q0 + 1) & 2) << 30)), __int_as_float(__float_as_int(cc1) ^ (((q1 + 1) & 2) << 30))};
}

// ----------------------------------------------------------------------------- shared memory, staging, addressing
// All shared-memory accesses index this one array with 32-bit float indices.
// Layout: [4 floats: mbarrier][COMMON][extra section: M or J tables, or nothing][team 0 rows][team 1 rows]...
// A state row holds one float per environment of the tile (32 N floats); lane l owns floats N l .. N l + N - 1.
extern __shared__ __align__(16) float smf[];

template <class T> __device__ __forceinline__ T lds(int idx);
template <> __device__ __forceinline__ float lds<float>(int idx) { return smf[idx]; }
template <> __device__ __forceinline__ f2 lds<f2>(int idx) {
  f2 r;
  r.v = *reinterpret_cast<const unsigned long long*>(smf + idx);
  return r;
}
__device__ __forceinline__ void sts(int idx, float v) { smf[idx] = v; }
__device__ __forceinline__ void sts(int idx, f2 v) { *reinterpret_cast<unsigned long long*>(smf + idx) = v.v; }
// three consecutive state rows (RW floats apart) starting at idx
template <class T, int RW> __device__ __forceinline__ V3<T> ldrow3(int idx) {
  return {lds<T>(idx), lds<T>(idx + RW), lds<T>(idx + 2 * RW)};
}
template <int RW, class T> __device__ __forceinline__ void strow3(int idx, V3<T> v) {
  sts(idx, v.x); sts(idx + RW, v.y); sts(idx + 2 * RW, v.z);
}
// model constants: 16-byte and 4-byte warp-uniform loads at a float index
__device__ __forceinline__ float4 ldc4(int idx) { return *reinterpret_cast<const float4*>(smf + idx); }
__device__ __forceinline__ int4 ldc4i(int idx) { return *reinterpret_cast<const int4*>(smf + idx); }
__device__ __forceinline__ float ldc(int idx) { return smf[idx]; }
__device__ __forceinline__ int ldci(int idx) { return __float_as_int(smf[idx]); }
__device__ __forceinline__ uint32_t ldc_u16(int byte_off) { return reinterpret_cast<const uint16_t*>(smf)[byte_off >> 1]; }
__device__ __forceinline__ uint32_t ldc_u8(int byte_off) { return reinterpret_cast<const uint8_t*>(smf)[byte_off]; }

// global stores of a pack at a 32-bit element index (streaming: outputs are never re-read by the kernels)
__device__ __forceinline__ void stg(float* out, uint32_t idx, float v) { __stcs(out + idx, v); }
__device__ __forceinline__ void stg(float* out, uint32_t idx, f2 v) {
  __stcs(reinterpret_cast<unsigned long long*>(out + idx), v.v);
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void bulk_g2s(uint32_t sdst, const void* gsrc, uint32_t bytes, uint32_t bar_a) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(sdst),
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
template <int N> __device__ __forceinline__ void cp_async_row(uint32_t sdst, const float* gsrc) {
  if (N == 1) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sdst), "l"(gsrc) : "memory");
  else        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sdst), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

// Per-thread view of the CTA.  All positions are float indices into smf.
struct Ctx {
  int common;        // BlobHeader
  int extra;         // MHeader... or JHeader...
  int bodies;        // BodyConst[0]; body i is at bodies + 64 i
  int tasks_b;       // BYTE offset of this warp's task list
  int st;            // this team's state rows, already offset to the lane's first float
  uint32_t e;        // first environment of this lane (>= B in the ragged tail: stores are skipped)
  uint32_t bar_id, bar_cnt;
  int w, L, lane;
  bool valid;
};

__device__ __forceinline__ void team_sync(const Ctx& c) {
  if (c.L > 1) asm volatile("bar.sync %0, %1;" ::"r"(c.bar_id), "r"(c.bar_cnt) : "memory");
}

// Where each staged input row lands among the team's state rows (RNEA parks q / qd / qdd of a body in the rows
// that later hold that body's force and joint scalars, so the inputs cost no shared memory of their own).
struct RowMap { uint16_t q[128], qd[64], qdd[64]; };

// `rcpL` = ceil(65536 / L): warp / L as a multiply and a shift (exact for warp < 64).
// map == nullptr: input row r of array k lands in state row (rows of the arrays before it) + r.
template <int N>
__device__ __forceinline__ Ctx setup(const void* gcommon, uint32_t cbytes, const void* gextra, uint32_t xbytes, int L,
                                     uint32_t rcpL, int team_rows, uint32_t B, const float* in0, int n0, const float* in1,
                                     int n1, const float* in2, int n2, const RowMap* map = nullptr) {
  constexpr int RW = 32 * N;
  const uint32_t bar_a = smem_u32(smf);
  Ctx c;
  const int warp = threadIdx.x >> 5;
  c.lane = threadIdx.x & 31;
  c.L = L;
  const int team = (warp * rcpL) >> 16;
  c.w = warp - team * L;
  const int teams = ((blockDim.x >> 5) * rcpL) >> 16;
  c.bar_id = team + 1;
  c.bar_cnt = L * 32;
  c.e = ((blockIdx.x * teams + team) * 32 + c.lane) * N;
  c.valid = c.e < B;
  const uint32_t el = c.valid ? c.e : B - N;                 // clamped environment for loads
  c.common = 4;
  c.extra = 4 + (cbytes >> 2);
  c.st = c.extra + (xbytes >> 2) + team * team_rows * RW + c.lane * N;
  // Programmatic dependent launch: let the next kernel in the stream start its own prologue while this grid
  // drains; our constants are immutable, so only the batched inputs wait for the previous grid (below).
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(cbytes + xbytes) : "memory");
    bulk_g2s(bar_a + 16, gcommon, cbytes, bar_a);
    if (xbytes) bulk_g2s(bar_a + 16 + cbytes, gextra, xbytes, bar_a);
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");           // previous grid complete, its writes visible
  // stage the team's input rows; warp w takes rows w, w + L, ...
  const uint32_t st_a = bar_a + 4u * c.st;
  if (map) {
    for (int r = c.w; r < n0; r += L) cp_async_row<N>(st_a + 4u * (map->q[r] * RW), in0 + ((uint32_t)r * B + el));
    for (int r = c.w; r < n1; r += L) cp_async_row<N>(st_a + 4u * (map->qd[r] * RW), in1 + ((uint32_t)r * B + el));
    for (int r = c.w; r < n2; r += L) cp_async_row<N>(st_a + 4u * (map->qdd[r] * RW), in2 + ((uint32_t)r * B + el));
  } else {
    for (int r = c.w; r < n0; r += L) cp_async_row<N>(st_a + 4u * (r * RW), in0 + ((uint32_t)r * B + el));
    for (int r = c.w; r < n1; r += L) cp_async_row<N>(st_a + 4u * ((n0 + r) * RW), in1 + ((uint32_t)r * B + el));
    for (int r = c.w; r < n2; r += L) cp_async_row<N>(st_a + 4u * ((n0 + n1 + r) * RW), in2 + ((uint32_t)r * B + el));
  }
  cp_async_wait_all();
  __syncthreads();          // mbarrier init visible to all; staged rows visible to the other warps
  mbar_wait(bar_a);
  c.bodies = c.common + (int)(sizeof(BlobHeader) / 4);
  c.tasks_b = 16 + ldci(c.common + 6) + 2 * c.w * ldci(c.common + 7);   // BlobHeader::off_tasks, task_stride
  return c;
}

// BlobHeader fields by word index (see bard_internal.h)
enum { H_NB = 0, H_NQ = 1, H_NV = 2, H_NSLOTS = 4, H_G = 8, H_OFF_CHILDREN = 11, H_OFF_DOF_BODY = 12 };

// Integer fields of BodyConst i (words 52..63) with three 16-byte broadcast loads.
struct Meta { int type, parent, q_off, v_off, src, save, flags, level; uint32_t anc_lo, anc_hi; int child_begin, child_count; };
__device__ __forceinline__ Meta load_meta(int body) {
  const int4 a = ldc4i(body + 52), b = ldc4i(body + 56), d = ldc4i(body + 60);
  return {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, (uint32_t)d.x, (uint32_t)d.y, d.z, d.w};
}
// words 36..51: Sw Sl mass h Io
struct Inertia { V3<float> Sw, Sl; float mass; V3<float> h; float Io[6]; };
__device__ __forceinline__ Inertia load_inertia(int body) {
  const float4 a = ldc4(body + 36), b = ldc4(body + 40), d = ldc4(body + 44), e = ldc4(body + 48);
  return {{a.x, a.y, a.z}, {a.w, b.x, b.y}, b.z, {b.w, d.x, d.y}, {d.z, d.w, e.x, e.y, e.z, e.w}};
}

// ----------------------------------------------------------------------------- joint transform (a1)
// R_pc = R0 + u A + w B ; t_pc = t0 + u a + w b   (eq. (4)-(5)), constants read with
// 16-byte broadcast loads.  (u, w): revolute (sin q, 1 - cos q); prismatic (q, 0); fixed (0, 0).
// With T_post = I (always so in SIMPLE kernels) t_pc = t0 is a model constant: `tc`; otherwise `tv`.
template <bool SIMPLE, class T>
__device__ __forceinline__ void joint_Rt(int body, int flags, T u, T w, M3<T>& R, V3<float>& tc, V3<T>& tv) {
  float k[36];
#pragma unroll
  for (int i = 0; i < (SIMPLE ? 8 : 9); ++i) {
    const float4 v = ldc4(body + 4 * i);
    k[4 * i] = v.x; k[4 * i + 1] = v.y; k[4 * i + 2] = v.z; k[4 * i + 3] = v.w;
  }
#pragma unroll
  for (int i = 0; i < 9; ++i) R.m[i] = fm(w, k[18 + i], fm(u, k[9 + i], k[i]));
  tc = {k[27], k[28], k[29]};
  if (!SIMPLE) {
    if (flags & 1) tv = {T(k[27]), T(k[28]), T(k[29])};
    else tv = {fm(w, k[33], fm(u, k[30], k[27])), fm(w, k[34], fm(u, k[31], k[28])), fm(w, k[35], fm(u, k[32], k[29]))};
  }
}
// free joint: q = [p, quat xyzw]; R_pc = R0 R(quat/|quat|), t_pc = R0 p + t0.  qrow = first staged q row of the joint.
template <class T, int RW>
__device__ __forceinline__ void free_Rt(int body, int qrow, M3<T>& R, V3<T>& t) {
  const V3<T> p = ldrow3<T, RW>(qrow);
  T x = lds<T>(qrow + 3 * RW), y = lds<T>(qrow + 4 * RW), z = lds<T>(qrow + 5 * RW), s = lds<T>(qrow + 6 * RW);
  const T n = rsq(fm(x, x, fm(y, y, fm(z, z, s * s))));
  x = x * n; y = y * n; z = z * n; s = s * n;
  const T one = 1.f, two = 2.f;
  const M3<T> Rq = {{one - two * (y * y + z * z), two * (x * y - z * s), two * (x * z + y * s),
                     two * (x * y + z * s), one - two * (x * x + z * z), two * (y * z - x * s),
                     two * (x * z - y * s), two * (y * z + x * s), one - two * (x * x + y * y)}};
  M3<float> R0;
  const float4 a = ldc4(body), b = ldc4(body + 4);
  R0.m[0] = a.x; R0.m[1] = a.y; R0.m[2] = a.z; R0.m[3] = a.w; R0.m[4] = b.x; R0.m[5] = b.y; R0.m[6] = b.z; R0.m[7] = b.w;
  R0.m[8] = ldc(body + 8);
  const V3<float> t0 = {ldc(body + 27), ldc(body + 28), ldc(body + 29)};
  R = mul(R0, Rq);
  t = mul_acc(R0, p, t0);
}
// Local transform of a body from its staged q row(s) (qrow = float index of the body's first q row for this lane).
// Returns true when the translation is the per-environment tv, false when it is the constant tc.
template <bool SIMPLE, class T, int RW>
__device__ __forceinline__ bool local_Rt(int body, const Meta& m, int qrow, M3<T>& R, V3<float>& tc, V3<T>& tv, T& u, T& w) {
  if (m.type == BARD_JOINT_FREE) {
    u = 0.f; w = 0.f;
    free_Rt<T, RW>(body, qrow, R, tv);
    return true;
  }
  if (SIMPLE || m.type == BARD_JOINT_REVOLUTE) {
    T s, co;
    sincos_fast(lds<T>(qrow), s, co);
    u = s; w = T(1.0f) - co;
  } else if (m.type == BARD_JOINT_PRISMATIC) {
    u = lds<T>(qrow); w = 0.f;
  } else {
    u = 0.f; w = 0.f;
  }
  joint_Rt<SIMPLE, T>(body, m.flags, u, w, R, tc, tv);
  return !SIMPLE;
}

// World pose of a body from its parent's -- a2.  `cur` holds the pose of this warp's previous task; a parent
// on another warp is first fetched from its slot into `cur`, then cur <- cur * (R, t).
template <class T> struct Pose { M3<T> R; V3<T> p; };

template <class T, int RW>
__device__ __forceinline__ void fetch_parent(int src, Pose<T>& cur, int slots) {
  if (src >= 0) {
    const int s = slots + src * 12 * RW;
#pragma unroll
    for (int k = 0; k < 9; ++k) cur.R.m[k] = lds<T>(s + k * RW);
    cur.p = ldrow3<T, RW>(s + 9 * RW);
  }
}
template <class T, class TT>
__device__ __forceinline__ void compose(int src, Pose<T>& cur, const M3<T>& R, V3<TT> t) {
  if (src == -1) {
    cur.R = R;
    cur.p = {T(t.x), T(t.y), T(t.z)};
  } else {
    cur.p = mul_acc(cur.R, t, cur.p);
    cur.R = mul(cur.R, R);
  }
}
template <class T, int RW>
__device__ __forceinline__ void save_pose(int save, const Pose<T>& P, int slots) {
  if (save >= 0) {
    const int s = slots + save * 12 * RW;
#pragma unroll
    for (int k = 0; k < 9; ++k) sts(s + k * RW, P.R.m[k]);
    strow3<RW>(s + 9 * RW, P.p);
  }
}
// FK of one body: local transform, parent fetch, compose, save.
template <bool SIMPLE, class T, int RW>
__device__ __forceinline__ void fk_body(int body, const Meta& m, int qs, int slots, Pose<T>& cur, T& u, T& w) {
  M3<T> R; V3<float> tc; V3<T> tv;
  const bool var_t = local_Rt<SIMPLE, T, RW>(body, m, qs + m.q_off * RW, R, tc, tv, u, w);
  fetch_parent<T, RW>(m.src, cur, slots);
  if (var_t) compose(m.src, cur, R, tv);
  else compose(m.src, cur, R, tc);
  save_pose<T, RW>(m.save, cur, slots);
}

// ============================================================================= FK kernel (a1 + a2)
// team rows: q[nq] | pose slots[12 nslots]
template <bool SIMPLE, int N>
__global__ void __launch_bounds__(256) fk_kernel(const void* __restrict__ gcommon, uint32_t cbytes, int L, uint32_t rcpL,
                                                 int team_rows, int nq, uint32_t B, const float* __restrict__ q,
                                                 float* __restrict__ pose) {
  using T = typename Pack<N>::T;
  constexpr int RW = 32 * N;
  const Ctx C = setup<N>(gcommon, cbytes, nullptr, 0, L, rcpL, team_rows, B, q, nq, nullptr, 0, nullptr, 0);
  const int qs = C.st;
  const int slots = C.st + nq * RW;
  Pose<T> cur;
  for (int k = 0;; ++k) {
    const uint32_t tk = ldc_u16(C.tasks_b + 2 * k);
    if (tk == TASK_END) break;
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const int body = C.bodies + 64 * i;
      const Meta m = load_meta(body);
      T u, w;
      fk_body<SIMPLE, T, RW>(body, m, qs, slots, cur, u, w);
      if (C.valid) {
        const uint32_t o = (uint32_t)(i * 12) * B + C.e;
#pragma unroll
        for (int j = 0; j < 9; ++j) stg(pose, o + j * B, cur.R.m[j]);
        stg(pose, o + 9 * B, cur.p.x); stg(pose, o + 10 * B, cur.p.y); stg(pose, o + 11 * B, cur.p.z);
      }
    }
    if (tk & TASK_BAR) team_sync(C);
  }
}

// World-origin screws of a body's DOFs, s = [omega; v0] with v0 = R l + p x omega: for a revolute joint
// with T_post = I this is exactly the column [p_k x (R_k a'_k); R_k a'_k] of eq. (7).
// Stored as 6 rows per DOF at dof + (v * 6 + k) * RW.
template <bool SIMPLE, class T, int RW>
__device__ __forceinline__ void store_screws(int body, const Meta& m, const Pose<T>& P, int dof) {
  if (!SIMPLE && m.type == BARD_JOINT_FIXED) return;
  const int d = dof + m.v_off * 6 * RW;
  if (m.type == BARD_JOINT_FREE) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const V3<T> col = {P.R.m[k], P.R.m[3 + k], P.R.m[6 + k]};   // R e_k
      const int dl = d + k * 6 * RW;                              // linear DOF k: omega = 0, v0 = R e_k
      strow3<RW>(dl, V3<T>{T(0.f), T(0.f), T(0.f)});
      strow3<RW>(dl + 3 * RW, col);
      const int da = d + (3 + k) * 6 * RW;                        // angular DOF k: omega = R e_k, v0 = p x omega
      strow3<RW>(da, col);
      strow3<RW>(da + 3 * RW, cross(P.p, col));
    }
    return;
  }
  const float4 a = ldc4(body + 36);                               // Sw, Sl.x
  const V3<T> om = mul(P.R, V3<float>{a.x, a.y, a.z});
  V3<T> v0 = cross(P.p, om);
  if (!SIMPLE && (!(m.flags & 1) || m.type == BARD_JOINT_PRISMATIC)) {
    const float4 b = ldc4(body + 40);
    v0 = mul_acc(P.R, V3<float>{a.w, b.x, b.y}, v0);
  }
  strow3<RW>(d, om);
  strow3<RW>(d + 3 * RW, v0);
}

// Structurally zero output rows (flat row indices, list padded to a multiple of 4 with 0xffff): 8 N lanes x
// 16 bytes cover the 32 N environments of one row, so one store instruction clears 4 / N rows.  Needs
// B % 4 == 0 and a 16-byte aligned output (else one row per instruction).
template <int N>
__device__ __forceinline__ void zero_rows(const Ctx& C, int zr_b, int nz, float* out, uint32_t B, bool vec_ok) {
  if (vec_ok) {
    constexpr int LPR = 8 * N, RPI = 4 / N;                       // lanes per row, rows per instruction
    const int sub = C.lane / LPR;
    const uint32_t ev = C.e - C.lane * N + (C.lane % LPR) * 4;
    const bool ok = ev < B;
    for (int g = C.w * RPI; g < nz; g += C.L * RPI) {
      const uint32_t row = ldc_u16(zr_b + 2 * (g + sub));
      if (ok && row != 0xffffu) __stcs(reinterpret_cast<float4*>(out + (row * B + ev)), make_float4(0.f, 0.f, 0.f, 0.f));
    }
  } else {
    using T = typename Pack<N>::T;
    for (int g = C.w; g < nz; g += C.L) {
      const uint32_t row = ldc_u16(zr_b + 2 * g);
      if (C.valid && row != 0xffffu) stg(out, row * B + C.e, T(0.f));
    }
  }
}

// ============================================================================= Jacobian kernel (a3)
// team rows: q[nq] | pose slots[12 nslots] | screws[6 nv] | frame origins[3 nframes]
// Phase 1: level-parallel FK over the union of the frames' ancestor paths, screws and frame origins to smem.
// Phase 2: the non-zero columns (frame, dof) are dealt round-robin to the team's warps; each writes its 6 rows.
// Phase 3: the zero rows.
template <bool SIMPLE, int N>
__global__ void __launch_bounds__(256) jacobian_kernel(const void* __restrict__ gcommon, uint32_t cbytes,
                                                       const void* __restrict__ gj, uint32_t jbytes, int L, uint32_t rcpL,
                                                       int team_rows, int nq, int nv, int nslots, uint32_t B,
                                                       const float* __restrict__ q, float* __restrict__ J, int vec_ok) {
  using T = typename Pack<N>::T;
  constexpr int RW = 32 * N;
  const Ctx C = setup<N>(gcommon, cbytes, gj, jbytes, L, rcpL, team_rows, B, q, nq, nullptr, 0, nullptr, 0);
  const int xb = 4 * C.extra;                                    // byte offset of the J section
  const int frames = C.extra + 8;                                // FrameConst[0] (8 words each)
  const int qs = C.st;
  const int slots = C.st + nq * RW;
  const int dof = slots + nslots * 12 * RW;
  const int pe = dof + nv * 6 * RW;
  const uint32_t jm_lo = (uint32_t)ldci(C.extra + 1), jm_hi = (uint32_t)ldci(C.extra + 2);
  const int bframes_b = xb + ldci(C.extra + 7);
  Pose<T> cur;
  for (int k = 0;; ++k) {
    const uint32_t tk = ldc_u16(C.tasks_b + 2 * k);
    if (tk == TASK_END) break;
    const int i = tk & TASK_BODY_MASK;
    if (!(tk & TASK_NOOP) && (((i < 32 ? jm_lo : jm_hi) >> (i & 31)) & 1)) {
      const int body = C.bodies + 64 * i;
      const Meta m = load_meta(body);
      T u, w;
      fk_body<SIMPLE, T, RW>(body, m, qs, slots, cur, u, w);
      store_screws<SIMPLE, T, RW>(body, m, cur, dof);
      uint32_t fm_ = ldc_u16(bframes_b + 2 * i);                 // frames attached to this body
      while (fm_) {
        const int f = __ffs(fm_) - 1;
        fm_ &= fm_ - 1;
        const float4 fr = ldc4(frames + 8 * f);                  // body, off[3]
        strow3<RW>(pe + 3 * f * RW, mul_acc(cur.R, V3<float>{fr.y, fr.z, fr.w}, cur.p));
      }
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  const int cols_b = xb + ldci(C.extra + 3);
  const int ncols = ldci(C.extra + 4);
  const uint32_t nvu = nv;
  for (int idx = C.w; idx < ncols; idx += L) {
    const uint32_t cj = ldc_u16(cols_b + 2 * idx);
    const uint32_t f = cj >> 8, j = cj & 255u;
    const int d = dof + j * 6 * RW;
    const V3<T> ang = ldrow3<T, RW>(d);
    const V3<T> lin = cross_acc(ang, ldrow3<T, RW>(pe + 3 * f * RW), ldrow3<T, RW>(d + 3 * RW));   // shift to the frame origin
    if (C.valid) {
      const uint32_t o = (f * 6 * nvu + j) * B + C.e;
      const uint32_t rs = nvu * B;
      stg(J, o, lin.x); stg(J, o + rs, lin.y); stg(J, o + 2 * rs, lin.z);
      stg(J, o + 3 * rs, ang.x); stg(J, o + 4 * rs, ang.y); stg(J, o + 5 * rs, ang.z);
    }
  }
  zero_rows<N>(C, xb + ldci(C.extra + 5), ldci(C.extra + 6), J, B, vec_ok != 0);
}

// ============================================================================= RNEA kernel (a4 + a5)
// Body-frame recursion, internal order [angular; linear].
// team rows: motion slots[12 nslots] (v.w v.v a.w a.v) | body regions[8 nb] (n(3) f(3) u w) | free-joint inputs[19 nfree]
// The staged inputs of a 1-DOF body are parked in its own region until its outward task has read them
// (qd -> row 0, qdd -> row 1, q -> row 6); a free joint's q(7) qd(6) qdd(6) get 19 rows of their own (q is
// read again by the inward pass).
// Outward (level-parallel, eq. (6)): v, a of the parent come from the registers of this warp's
// previous task, a shared-memory slot, or the world (v = 0, a = -g: gravity trick); the net body force f_i and
// the joint scalars (u, w) are parked in shared memory.
// Inward (PAPER.md:91 keeps this pass sequential because siblings collide on the parent; here it is
// level-parallel too): a body first adds the forces its children left -- already expressed in ITS frame -- in
// ascending child order (deterministic, no atomics), emits tau_i = S_i^T f_i, then overwrites its own force
// rows with X_up^T f_i for its parent, rebuilding T_pc from (u, w) with eq. (4)-(5).
template <class T> struct Motion { V3<T> vw, vv, aw, av; };

// v, a of a body from its parent's (already in `cur`): X_up [w; v] = [R^T w ; R^T (v + w x t)]
template <class T, class TT>
__device__ __forceinline__ void rnea_outward(Motion<T>& cur, const M3<T>& R, V3<TT> t, bool haslin, V3<T> vJw, V3<T> vJv,
                                             V3<T> aJw, V3<T> aJv) {
  const V3<T> vw = mulT_acc(R, cur.vw, vJw);
  const V3<T> tv = cross_acc(cur.vw, t, cur.vv);
  const V3<T> ta = cross_acc(cur.aw, t, cur.av);
  const V3<T> aw = cross_acc(vw, vJw, mulT_acc(R, cur.aw, aJw));
  V3<T> vv, av;
  if (haslin) {
    vv = mulT_acc(R, tv, vJv);
    av = cross_acc(vw, vJv, cross_acc(vv, vJw, mulT_acc(R, ta, aJv)));
  } else {
    vv = mulT(R, tv);
    av = cross_acc(vv, vJw, mulT(R, ta));
  }
  cur.vw = vw; cur.vv = vv; cur.aw = aw; cur.av = av;
}

template <bool SIMPLE, int N>
__global__ void __launch_bounds__(256) rnea_kernel(const void* __restrict__ gcommon, uint32_t cbytes, int L, uint32_t rcpL,
                                                   int team_rows, int nq, int nv, int nb, int nslots, uint32_t B,
                                                   const float* __restrict__ q, const float* __restrict__ qd,
                                                   const float* __restrict__ qdd, float* __restrict__ tau,
                                                   const __grid_constant__ RowMap map) {
  using T = typename Pack<N>::T;
  constexpr int RW = 32 * N;
  const Ctx C = setup<N>(gcommon, cbytes, nullptr, 0, L, rcpL, team_rows, B, q, nq, qd, nv, qdd, nv, &map);
  const int children_b = 16 + ldci(C.common + H_OFF_CHILDREN);
  const int slots = C.st;
  const int bst = slots + nslots * 12 * RW;                    // 8 rows per body
  const int fin = bst + nb * 8 * RW;                           // 19 rows per free-joint body
  const V3<float> ng = {-ldc(C.common + H_G), -ldc(C.common + H_G + 1), -ldc(C.common + H_G + 2)};
  Motion<T> cur;                                               // this warp's previous body: v and a
  int ntask = 0;
  for (int k = 0;; ++k) {
    const uint32_t tk = ldc_u16(C.tasks_b + 2 * k);
    if (tk == TASK_END) { ntask = k; break; }
    if (!(tk & TASK_NOOP)) {
      const int i = tk & TASK_BODY_MASK;
      const int body = C.bodies + 64 * i;
      const Meta m = load_meta(body);
      const Inertia in = load_inertia(body);
      M3<T> R; V3<float> tc; V3<T> tv; T u, w;
      const bool is_free = m.type == BARD_JOINT_FREE;
      const int b = bst + i * 8 * RW;
      const int fi = fin + ((m.flags >> 8) & 0xff) * 19 * RW;
      const bool var_t = local_Rt<SIMPLE, T, RW>(body, m, is_free ? fi : b + 6 * RW, R, tc, tv, u, w);
      // joint velocity / acceleration in the body frame: S qd, S qdd
      const bool haslin = is_free || !SIMPLE;
      const V3<T> zero = {T(0.f), T(0.f), T(0.f)};
      V3<T> vJw = zero, vJv = zero, aJw = zero, aJv = zero;
      if (is_free) {
        const int d1 = fi + 7 * RW, d2 = fi + 13 * RW;
        vJw = ldrow3<T, RW>(d1 + 3 * RW); vJv = ldrow3<T, RW>(d1);
        aJw = ldrow3<T, RW>(d2 + 3 * RW); aJv = ldrow3<T, RW>(d2);
      } else if (SIMPLE || m.type != BARD_JOINT_FIXED) {
        const T qd_i = lds<T>(b), qdd_i = lds<T>(b + RW);
        vJw = scale(qd_i, in.Sw); aJw = scale(qdd_i, in.Sw);
        if (!SIMPLE) { vJv = scale(qd_i, in.Sl); aJv = scale(qdd_i, in.Sl); }
      }
      if (m.src == -1) {                                       // world parent: v_p = 0, a_p = [0; -g]; v x vJ = 0
        cur.vw = vJw; cur.vv = vJv; cur.aw = aJw;
        if (haslin) cur.av = mulT_acc(R, ng, aJv);
        else cur.av = mulT(R, ng);
      } else {
        if (m.src >= 0) {
          const int s = slots + m.src * 12 * RW;
          cur.vw = ldrow3<T, RW>(s); cur.vv = ldrow3<T, RW>(s + 3 * RW);
          cur.aw = ldrow3<T, RW>(s + 6 * RW); cur.av = ldrow3<T, RW>(s + 9 * RW);
        }
        if (var_t) rnea_outward(cur, R, tv, haslin, vJw, vJv, aJw, aJv);
        else rnea_outward(cur, R, tc, haslin, vJw, vJv, aJw, aJv);
      }
      // f = I a + v x* (I v),  I = (m, h, Io) about the body origin
      const V3<T> n1 = cross_acc(in.h, cur.vv, symmul(in.Io, cur.vw));
      const V3<T> f1 = cross_acc(cur.vw, in.h, scale(in.mass, cur.vv));
      const V3<T> n2 = cross_acc(in.h, cur.av, symmul(in.Io, cur.aw));
      const V3<T> f2_ = cross_acc(cur.aw, in.h, scale(in.mass, cur.av));
      const V3<T> n = cross_acc(cur.vv, f1, cross_acc(cur.vw, n1, n2));
      const V3<T> f = cross_acc(cur.vw, f1, f2_);
      strow3<RW>(b, n); strow3<RW>(b + 3 * RW, f);
      sts(b + 6 * RW, u); sts(b + 7 * RW, w);
      if (m.save >= 0) {
        const int s = slots + m.save * 12 * RW;
        strow3<RW>(s, cur.vw); strow3<RW>(s + 3 * RW, cur.vv); strow3<RW>(s + 6 * RW, cur.aw); strow3<RW>(s + 9 * RW, cur.av);
      }
    }
    if (tk & TASK_BAR) team_sync(C);
  }
  // inward pass, deepest level first: the same task list walked backwards
  for (int k = ntask - 1; k >= 0; --k) {
    const uint32_t tk = ldc_u16(C.tasks_b + 2 * k);
    if ((tk & TASK_BAR) && k != ntask - 1) team_sync(C);
    if (tk & TASK_NOOP) continue;
    const int i = tk & TASK_BODY_MASK;
    const int body = C.bodies + 64 * i;
    const Meta m = load_meta(body);
    const int b = bst + i * 8 * RW;
    V3<T> n = ldrow3<T, RW>(b), f = ldrow3<T, RW>(b + 3 * RW);
    for (int cc = 0; cc < m.child_count; ++cc) {
      const int cb = bst + (int)ldc_u8(children_b + m.child_begin + cc) * 8 * RW;
      n = n + ldrow3<T, RW>(cb); f = f + ldrow3<T, RW>(cb + 3 * RW);
    }
    if (C.valid) {
      const uint32_t o = (uint32_t)m.v_off * B + C.e;
      if (m.type == BARD_JOINT_FREE) {
        stg(tau, o, f.x); stg(tau, o + B, f.y); stg(tau, o + 2 * B, f.z);
        stg(tau, o + 3 * B, n.x); stg(tau, o + 4 * B, n.y); stg(tau, o + 5 * B, n.z);
      } else if (SIMPLE || m.type != BARD_JOINT_FIXED) {
        const float4 a4 = ldc4(body + 36);
        T tv = dot(V3<float>{a4.x, a4.y, a4.z}, n);
        if (!SIMPLE) { const float4 b4 = ldc4(body + 40); tv = dot_acc(V3<float>{a4.w, b4.x, b4.y}, f, tv); }
        stg(tau, o, tv);
      }
    }
    if (m.parent >= 0) {
      M3<T> R; V3<float> tc; V3<T> tv;
      bool var_t = true;
      if (m.type == BARD_JOINT_FREE) free_Rt<T, RW>(body, fin + ((m.flags >> 8) & 0xff) * 19 * RW, R, tv);
      else { joint_Rt<SIMPLE, T>(body, m.flags, lds<T>(b + 6 * RW), lds<T>(b + 7 * RW), R, tc, tv); var_t = !SIMPLE; }
      const V3<T> fp = mul(R, f);
      if (var_t) strow3<RW>(b, cross_acc(tv, fp, mul(R, n)));
      else strow3<RW>(b, cross_acc(tc, fp, mul(R, n)));
      strow3<RW>(b + 3 * RW, fp);
    }
  }
}

// ============================================================================= CRBA kernel (a6 + a7)
// World-frame formulation: every composite inertia is expressed about the WORLD origin in world axes
// (m, h, I: 10 floats), so the backward sweep  I^c_parent += X^T I^c_child X degenerates to
// ten additions (X = identity between world-frame quantities), and M_ij = s_j . (I^c_i s_i) for every
// ancestor DOF j needs no transform along the walk.  The screws s are the eq. (7) columns (store_screws).
// team rows: q[nq] | pose slots[12 nslots] | screws[6 nv] | inertia[10 nb] | poses of free-joint bodies[12 nfree]
// Phase 1 (outward, level-parallel): FK, screws, world-frame body inertias.
// Phase 2 (inward, level-parallel): a body adds its children's composites in ascending child order.
// Phase 3: the rows of M are dealt to the team's warps (host LPT schedule); the warp that owns row i walks
//          the host-built list of DOFs j <= i on ancestor bodies and writes M[i][j] and M[j][i]; the six
//          entries against a free-joint ancestor (floating base) come from ONE force transform into that
//          body's frame, [R^T f ; R^T (n + f x p)], instead of six 6-term dot products.
// Phase 4: the structurally zero entries.  Every element of M is written exactly once.
template <bool SIMPLE, int N>
__global__ void __launch_bounds__(256) crba_kernel(const void* __restrict__ gcommon, uint32_t cbytes, uint32_t mbytes, int L,
                                                   uint32_t rcpL, int team_rows, int nq, int nv, int nslots, uint32_t B,
                                                   const float* __restrict__ q, float* __restrict__ Mout, int vec_ok) {
  using T = typename Pack<N>::T;
  constexpr int RW = 32 * N;
  const Ctx C = setup<N>(gcommon, cbytes, static_cast<const unsigned char*>(gcommon) + cbytes, mbytes, L, rcpL, team_rows, B,
                         q, nq, nullptr, 0, nullptr, 0);
  const int children_b = 16 + ldci(C.common + H_OFF_CHILDREN);
  const int xb = 4 * C.extra;                                  // byte offset of the M section
  const int qs = C.st;
  const int slots = C.st + nq * RW;
  const int dof = slots + nslots * 12 * RW;                    // 6 rows per DOF
  const int ic = dof + nv * 6 * RW;                            // 10 rows per body: m h(3) I(6)
  const int fpose = ic + ldci(C.common + H_NB) * 10 * RW;      // 12 rows per free-joint body: R p
  if (C.w >= ldci(C.common + 5)) {
    // helper warp (w >= L): no body of its own in the level sweeps, only the team barriers -- nlevels in the
    // outward sweep, nlevels - 1 in the inward one -- then its share of the fill
    const int nl = ldci(C.common + 3);
    for (int l = 0; l < 2 * nl - 1; ++l) team_sync(C);
  } else {
    Pose<T> cur;
    int ntask = 0;
    for (int k = 0;; ++k) {
      const uint32_t tk = ldc_u16(C.tasks_b + 2 * k);
      if (tk == TASK_END) { ntask = k; break; }
      if (!(tk & TASK_NOOP)) {
        const int i = tk & TASK_BODY_MASK;
        const int body = C.bodies + 64 * i;
        const Meta m = load_meta(body);
        T u, w;
        fk_body<SIMPLE, T, RW>(body, m, qs, slots, cur, u, w);
        store_screws<SIMPLE, T, RW>(body, m, cur, dof);
        if (m.type == BARD_JOINT_FREE) {
          const int fp = fpose + ((m.flags >> 8) & 0xff) * 12 * RW;
  #pragma unroll
          for (int j = 0; j < 9; ++j) sts(fp + j * RW, cur.R.m[j]);
          strow3<RW>(fp + 9 * RW, cur.p);
        }
        // body inertia about the world origin: h' = R h + m p ; with h'' = R h + m p / 2:
        // I' = R Io R^T + 2 (p . h'') 1 - (h'' p^T + p h''^T)
        const Inertia in = load_inertia(body);
        const float ms = in.mass;
        const V3<T> p = cur.p;
        const V3<T> hr = mul(cur.R, in.h);
        const V3<T> hh = axpy(0.5f * ms, p, hr);
        const V3<T> r0 = {cur.R.m[0], cur.R.m[1], cur.R.m[2]}, r1 = {cur.R.m[3], cur.R.m[4], cur.R.m[5]},
                    r2 = {cur.R.m[6], cur.R.m[7], cur.R.m[8]};
        const V3<T> a0 = symmul(in.Io, r0), a1 = symmul(in.Io, r1), a2 = symmul(in.Io, r2);
        const T d = T(2.f) * dot(p, hh);
        const int o = ic + i * 10 * RW;
        sts(o, T(ms));
        strow3<RW>(o + RW, axpy(ms, p, hr));
        sts(o + 4 * RW, fm(T(-2.f) * hh.x, p.x, dot_acc(r0, a0, d)));           // xx
        sts(o + 5 * RW, fm(-hh.x, p.y, fm(-p.x, hh.y, dot(r0, a1))));           // xy
        sts(o + 6 * RW, fm(-hh.x, p.z, fm(-p.x, hh.z, dot(r0, a2))));           // xz
        sts(o + 7 * RW, fm(T(-2.f) * hh.y, p.y, dot_acc(r1, a1, d)));           // yy
        sts(o + 8 * RW, fm(-hh.y, p.z, fm(-p.y, hh.z, dot(r1, a2))));           // yz
        sts(o + 9 * RW, fm(T(-2.f) * hh.z, p.z, dot_acc(r2, a2, d)));           // zz
      }
      if (tk & TASK_BAR) team_sync(C);
    }
    // composite sweep, deepest level first
    for (int k = ntask - 1; k >= 0; --k) {
      const uint32_t tk = ldc_u16(C.tasks_b + 2 * k);
      if ((tk & TASK_BAR) && k != ntask - 1) team_sync(C);
      if (tk & TASK_NOOP) continue;
      const int i = tk & TASK_BODY_MASK;
      const int cbeg = ldci(C.bodies + 64 * i + 62), ccnt = ldci(C.bodies + 64 * i + 63);
      if (ccnt == 0) continue;
      const int d = ic + i * 10 * RW;
      T acc[10];
  #pragma unroll
      for (int j = 0; j < 10; ++j) acc[j] = lds<T>(d + j * RW);
      for (int cc = 0; cc < ccnt; ++cc) {
        const int s = ic + (int)ldc_u8(children_b + cbeg + cc) * 10 * RW;
  #pragma unroll
        for (int j = 0; j < 10; ++j) acc[j] = acc[j] + lds<T>(s + j * RW);
      }
  #pragma unroll
      for (int j = 0; j < 10; ++j) sts(d + j * RW, acc[j]);
    }
  }
  team_sync(C);
  // fill
  const int dof_body_b = 16 + ldci(C.common + H_OFF_DOF_BODY);
  const int rows_b = xb + ldci(C.extra + 0) + C.w * ldci(C.extra + 1);
  const int pairs_b = xb + ldci(C.extra + 5);
  const int pptr_b = xb + ldci(C.extra + 6);
  const int fanc_b = xb + ldci(C.extra + 7);
  const int fptr_b = xb + ldci(C.extra + 8);
  const uint32_t nvu = nv;
  for (int k = 0;; ++k) {
    const uint32_t i = ldc_u8(rows_b + k);
    if (i == 0xffu) break;
    const int I = ic + (int)ldc_u8(dof_body_b + i) * 10 * RW;
    const T ms = lds<T>(I);
    const V3<T> h = ldrow3<T, RW>(I + RW);
    const T Iw[6] = {lds<T>(I + 4 * RW), lds<T>(I + 5 * RW), lds<T>(I + 6 * RW), lds<T>(I + 7 * RW), lds<T>(I + 8 * RW),
                     lds<T>(I + 9 * RW)};
    const int si = dof + i * 6 * RW;
    const V3<T> om = ldrow3<T, RW>(si), v0 = ldrow3<T, RW>(si + 3 * RW);
    const V3<T> Fn = cross_acc(h, v0, symmul(Iw, om));       // F = I^c_i s_i  (moment about the world origin)
    const V3<T> Ff = cross_acc(om, h, scale(ms, v0));        //               (force)  m v0 - h x om
    const uint32_t rowo = i * nvu * B + C.e;                 // M[i][.]
    const uint32_t colo = i * B + C.e;                       // M[.][i]
    const int pe_ = pairs_b + ldc_u16(pptr_b + 2 * i + 2);
    int pp = pairs_b + ldc_u16(pptr_b + 2 * i);
    for (; pp + 1 < pe_; pp += 2) {                          // two pairs per trip: two independent FMA chains
      const uint32_t j0 = ldc_u8(pp), j1 = ldc_u8(pp + 1);
      const int s0 = dof + j0 * 6 * RW, s1 = dof + j1 * 6 * RW;
      const V3<T> a0 = ldrow3<T, RW>(s0), b0 = ldrow3<T, RW>(s0 + 3 * RW);
      const V3<T> a1 = ldrow3<T, RW>(s1), b1 = ldrow3<T, RW>(s1 + 3 * RW);
      const T v0_ = dot_acc(b0, Ff, dot(a0, Fn));
      const T v1_ = dot_acc(b1, Ff, dot(a1, Fn));
      if (C.valid) {
        stg(Mout, rowo + j0 * B, v0_);
        stg(Mout, colo + j0 * nvu * B, v0_);                 // j0 < j1 <= i: never the diagonal
        stg(Mout, rowo + j1 * B, v1_);
        if (j1 != i) stg(Mout, colo + j1 * nvu * B, v1_);
      }
    }
    if (pp < pe_) {
      const uint32_t j = ldc_u8(pp);
      const int sj = dof + j * 6 * RW;
      const T val = dot_acc(ldrow3<T, RW>(sj + 3 * RW), Ff, dot(ldrow3<T, RW>(sj), Fn));
      if (C.valid) {
        stg(Mout, rowo + j * B, val);
        if (j != i) stg(Mout, colo + j * nvu * B, val);
      }
    }
    // free-joint ancestors: M[i][v .. v+5] = [R^T Ff ; R^T (Fn + Ff x p)]  (linear block, angular block)
    const int fe_ = fanc_b + ldc_u16(fptr_b + 2 * i + 2);
    for (int fq = fanc_b + ldc_u16(fptr_b + 2 * i); fq < fe_; ++fq) {
      const int fbody = C.bodies + 64 * (int)ldc_u8(fq);
      const uint32_t vo = (uint32_t)ldci(fbody + 55);
      const int fp = fpose + ((ldci(fbody + 58) >> 8) & 0xff) * 12 * RW;
      M3<T> R;
#pragma unroll
      for (int j = 0; j < 9; ++j) R.m[j] = lds<T>(fp + j * RW);
      const V3<T> p = ldrow3<T, RW>(fp + 9 * RW);
      const V3<T> fl = mulT(R, Ff);
      const V3<T> nn = mulT(R, cross_acc(Ff, p, Fn));
      if (C.valid) {
        const uint32_t ro = rowo + vo * B, co = colo + vo * nvu * B, cs = nvu * B;
        stg(Mout, ro, fl.x); stg(Mout, ro + B, fl.y); stg(Mout, ro + 2 * B, fl.z);
        stg(Mout, ro + 3 * B, nn.x); stg(Mout, ro + 4 * B, nn.y); stg(Mout, ro + 5 * B, nn.z);
        stg(Mout, co, fl.x); stg(Mout, co + cs, fl.y); stg(Mout, co + 2 * cs, fl.z);
        stg(Mout, co + 3 * cs, nn.x); stg(Mout, co + 4 * cs, nn.y); stg(Mout, co + 5 * cs, nn.z);
      }
    }
  }
  zero_rows<N>(C, xb + ldci(C.extra + 3), ldci(C.extra + 4), Mout, B, vec_ok != 0);
}

// ============================================================================= explicit Euler step (config 2)
// qd += dt qdd ; q (+)= dt qd, in place (readings 1 and 15).  One thread per environment, the joint
// table (type, q_off, v_off of every body) read from the constant blob in global memory (warp-uniform, cached).
// Free joint: p += dt R(quat) v ; quat += dt/2 quat (x) (omega, 0) ; renormalised.  HBM-bound: 2 nv + nq rows in,
// nv + nq rows out, every access one full line per warp.
// qi / qdi: state in; qo_ / qdo: state out (the same pointers for the in-place step; no __restrict__ on them)
__global__ void __launch_bounds__(256) euler_kernel(const unsigned char* __restrict__ blob, int nb, uint32_t B, float dt,
                                                    const float* qi, const float* qdi, const float* __restrict__ qdd,
                                                    float* qo_, float* qdo) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (e >= B) return;
  const BodyConst* bc = reinterpret_cast<const BodyConst*>(blob + sizeof(BlobHeader));
  for (int i = 0; i < nb; ++i) {
    const int t = bc[i].type;
    const uint32_t qo = (uint32_t)bc[i].q_off * B + e, vo = (uint32_t)bc[i].v_off * B + e;
    if (t == BARD_JOINT_REVOLUTE || t == BARD_JOINT_PRISMATIC) {
      const float v = fmaf(dt, qdd[vo], qdi[vo]);
      qdo[vo] = v;
      qo_[qo] = fmaf(dt, v, qi[qo]);
    } else if (t == BARD_JOINT_FREE) {
      float tw[6];
#pragma unroll
      for (int k = 0; k < 6; ++k) { tw[k] = fmaf(dt, qdd[vo + k * B], qdi[vo + k * B]); qdo[vo + k * B] = tw[k]; }
      float x = qi[qo + 3 * B], y = qi[qo + 4 * B], z = qi[qo + 5 * B], w = qi[qo + 6 * B];
      const float n = rsqrtf(fmaf(x, x, fmaf(y, y, fmaf(z, z, w * w))));
      x *= n; y *= n; z *= n; w *= n;
      const float R[9] = {1.f - 2.f * (y * y + z * z), 2.f * (x * y - z * w), 2.f * (x * z + y * w),
                          2.f * (x * y + z * w), 1.f - 2.f * (x * x + z * z), 2.f * (y * z - x * w),
                          2.f * (x * z - y * w), 2.f * (y * z + x * w), 1.f - 2.f * (x * x + y * y)};
#pragma unroll
      for (int r = 0; r < 3; ++r)
        qo_[qo + r * B] = fmaf(dt, fmaf(R[3 * r + 2], tw[2], fmaf(R[3 * r + 1], tw[1], R[3 * r] * tw[0])), qi[qo + r * B]);
      const float h = 0.5f * dt, ox = tw[3], oy = tw[4], oz = tw[5];
      const float ex = fmaf(h, fmaf(w, ox, fmaf(y, oz, -z * oy)), x), ey = fmaf(h, fmaf(w, oy, fmaf(z, ox, -x * oz)), y),
                  ez = fmaf(h, fmaf(w, oz, fmaf(x, oy, -y * ox)), z), ew = fmaf(h, -fmaf(x, ox, fmaf(y, oy, z * oz)), w);
      const float m = rsqrtf(fmaf(ex, ex, fmaf(ey, ey, fmaf(ez, ez, ew * ew))));
      qo_[qo + 3 * B] = ex * m; qo_[qo + 4 * B] = ey * m; qo_[qo + 5 * B] = ez * m; qo_[qo + 6 * B] = ew * m;
    }
  }
}

// ----------------------------------------------------------------------------- launchers
struct LaunchCfg { int teams, threads, team_rows, pack; size_t smem; unsigned grid; uint32_t rcpL; bool pdl = true; };

constexpr size_t kSmemMax = 227 * 1024;

bool aligned(const void* p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

// N (environments per lane): 2 when the batch is even, every pointer is 8-byte aligned, there are enough
// tiles to fill the machine and the doubled tile state still leaves three CTAs per SM; else 1.  TEAMS per CTA: two tiles share one copy of the constants when the team
// is narrow; fewer if the state does not fit.  Small CTAs keep the last wave short.
bool pick_cfg(const Options& o, int L, int64_t B, size_t const_bytes, int team_rows, bool can_pack2, int64_t max_rows,
              LaunchCfg& cfg, std::string& why) {
  const int want_teams = (int)o.teams;                         // tuning / test knobs: fields of the model (bard_model_set_option)
  const int want_pack = (int)o.pack;
  const int64_t pack2_min_b = o.pack2_min_b;
  cfg.pdl = o.pdl != 0;
  const size_t fixed = 16 + const_bytes;
  // two environments per lane halve the non-FP instructions per environment but double the tile's shared
  // memory: taken only when at least three such CTAs still fit on an SM (measured: DESIGN.md "Tuning")
  const size_t tile2 = (size_t)team_rows * 64 * sizeof(float);
  int N = (can_pack2 && B >= pack2_min_b && (fixed + tile2 + 1024) * 3 <= kSmemMax) ? 2 : 1;
  if (want_pack == 1) N = 1;
  if (want_pack == 2 && can_pack2) N = 2;
  int teams = want_teams > 0 ? want_teams : (L <= 4 ? 2 : 1);
  teams = std::max(1, std::min(teams, 8 / L));
  size_t per_team = (size_t)team_rows * 32 * N * sizeof(float);
  if (N == 2 && fixed + per_team > kSmemMax) { N = 1; per_team /= 2; }
  while (teams > 1 && (fixed + per_team * teams) * 2 + 2048 > kSmemMax) --teams;   // keep >= 2 CTAs per SM
  cfg.teams = teams;
  cfg.pack = N;
  cfg.threads = teams * L * 32;
  cfg.team_rows = team_rows;
  cfg.smem = fixed + per_team * teams;
  const int64_t per_cta = (int64_t)teams * 32 * N;
  cfg.grid = (unsigned)((B + per_cta - 1) / per_cta);
  cfg.rcpL = (65536u + L - 1) / L;
  if (cfg.smem > kSmemMax) { why = "per-environment state does not fit in shared memory"; return false; }
  if (max_rows * B >= ((int64_t)1 << 32)) { why = "an input or output array has 2^32 elements or more"; return false; }
  return true;
}

template <int ID, typename K>   // ID: one static per kernel instantiation (several kernels share a signature)
bard_status prep(K kernel, const char* name) {
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
bard_status refuse(const char* name, const std::string& why) {
  set_error(std::string(name) + ": " + why);
  return BARD_ERR_UNSUPPORTED;
}
template <int V> using IC = std::integral_constant<int, V>;

// Launch with programmatic stream serialization (PDL): see setup().
template <typename K, typename... Args>
void launch(K kernel, const LaunchCfg& cfg, void* stream, Args... args) {
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3(cfg.grid);
  lc.blockDim = dim3(cfg.threads);
  lc.dynamicSmemBytes = cfg.smem;
  lc.stream = (cudaStream_t)stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = attr;
  lc.numAttrs = cfg.pdl ? 1 : 0;
  cudaLaunchKernelEx(&lc, kernel, args...);
}

// Calls go(kernel<SIMPLE, N>, id) for the run-time (simple, pack) pair.
#define BARD_DISPATCH(KERNEL, BASE, simple, pack, go)                                           \
  ((simple) ? ((pack) == 2 ? go(KERNEL<true, 2>, IC<BASE + 0>()) : go(KERNEL<true, 1>, IC<BASE + 1>()))   \
            : ((pack) == 2 ? go(KERNEL<false, 2>, IC<BASE + 2>()) : go(KERNEL<false, 1>, IC<BASE + 3>())))

}  // namespace

bard_status launch_euler(const Model& m, int64_t B, float dt, const float* q, const float* qd, const float* qdd, float* q_out, float* qd_out,
                         void* stream) {
  if ((int64_t)std::max(m.nq, m.nv) * B >= ((int64_t)1 << 32)) return refuse("bard_euler_step", "an input array has 2^32 elements or more");
  LaunchCfg cfg = {};
  cfg.pdl = m.opt.pdl != 0;
  cfg.threads = 256;
  cfg.grid = (unsigned)((B + 255) / 256);
  cfg.smem = 0;
  launch(euler_kernel, cfg, stream, (const unsigned char*)m.d_blob, (int)m.nb, (uint32_t)B, dt, q, qd, qdd, q_out, qd_out);
  return finish("bard_euler_step");
}
bard_status launch_fk(const Model& m, int64_t B, const float* q, float* pose, void* stream) {
  LaunchCfg cfg;
  std::string why;
  const bool p2 = B % 2 == 0 && aligned(q, 8) && aligned(pose, 8);
  if (!pick_cfg(m.opt, m.team_warps, B, m.common_bytes, m.nq + 12 * m.nslots, p2, std::max(12 * m.nb, m.nq), cfg, why)) return refuse("bard_fk", why);
  cfg.smem = solo_smem(m, cfg.grid, cfg.smem);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_fk");
    if (s != BARD_OK) return s;
    launch(kernel, cfg, stream, (const void*)m.d_blob, (uint32_t)m.common_bytes, (int)m.team_warps, cfg.rcpL, cfg.team_rows,
           (int)m.nq, (uint32_t)B, q, pose);
    return finish("bard_fk");
  };
  return BARD_DISPATCH(fk_kernel, 0, m.simple, cfg.pack, go);
}
bard_status launch_jacobian(const Model& m, int64_t B, const float* q, float* J, void* stream) {
  LaunchCfg cfg;
  std::string why;
  const bool p2 = B % 2 == 0 && aligned(q, 8) && aligned(J, 8);
  if (!pick_cfg(m.opt, m.team_warps, B, m.common_bytes + m.j_bytes, m.nq + 12 * m.nslots + 6 * m.nv + 3 * m.nframes, p2,
                std::max(6 * m.nframes * m.nv, m.nq), cfg, why))
    return refuse("bard_jacobian", why);
  const int vec_ok = (B % 4 == 0) && aligned(J, 16);
  cfg.smem = solo_smem(m, cfg.grid, cfg.smem);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_jacobian");
    if (s != BARD_OK) return s;
    launch(kernel, cfg, stream, (const void*)m.d_blob, (uint32_t)m.common_bytes, (const void*)m.d_jblob, (uint32_t)m.j_bytes,
           (int)m.team_warps, cfg.rcpL, cfg.team_rows, (int)m.nq, (int)m.nv, (int)m.nslots, (uint32_t)B, q, J, vec_ok);
    return finish("bard_jacobian");
  };
  return BARD_DISPATCH(jacobian_kernel, 4, m.simple, cfg.pack, go);
}
bard_status launch_rnea(const Model& m, int64_t B, const float* q, const float* qd, const float* qdd, float* tau,
                        void* stream) {
  LaunchCfg cfg;
  std::string why;
  const bool p2 = B % 2 == 0 && aligned(q, 8) && aligned(qd, 8) && aligned(qdd, 8) && aligned(tau, 8);
  if (!pick_cfg(m.opt, m.team_warps, B, m.common_bytes, 12 * m.nslots + 8 * m.nb + 19 * m.nfree, p2, std::max(m.nq, m.nv), cfg, why))
    return refuse("bard_rnea", why);
  RowMap map;                                                  // where the staged input rows land: built once with the model
  static_assert(sizeof(map.q) == sizeof(m.rowmap_q) && sizeof(map.qd) == sizeof(m.rowmap_qd) && sizeof(map.qdd) == sizeof(m.rowmap_qdd), "RowMap");
  std::memcpy(map.q, m.rowmap_q, sizeof(map.q));
  std::memcpy(map.qd, m.rowmap_qd, sizeof(map.qd));
  std::memcpy(map.qdd, m.rowmap_qdd, sizeof(map.qdd));
  cfg.smem = solo_smem(m, cfg.grid, cfg.smem);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_rnea");
    if (s != BARD_OK) return s;
    launch(kernel, cfg, stream, (const void*)m.d_blob, (uint32_t)m.common_bytes, (int)m.team_warps, cfg.rcpL, cfg.team_rows,
           (int)m.nq, (int)m.nv, (int)m.nb, (int)m.nslots, (uint32_t)B, q, qd, qdd, tau, map);
    return finish("bard_rnea");
  };
  return BARD_DISPATCH(rnea_kernel, 8, m.simple, cfg.pack, go);
}
bard_status launch_crba(const Model& m, int64_t B, const float* q, float* M, void* stream) {
  LaunchCfg cfg;
  std::string why;
  const bool p2 = B % 2 == 0 && aligned(q, 8) && aligned(M, 8);
  if (!pick_cfg(m.opt, m.crba_warps, B, m.common_bytes + m.m_bytes, m.nq + 12 * m.nslots + 6 * m.nv + 10 * m.nb + 12 * m.nfree, p2,
                std::max(m.nv * m.nv, m.nq), cfg, why))
    return refuse("bard_crba", why);
  const int vec_ok = (B % 4 == 0) && aligned(M, 16);
  cfg.smem = solo_smem(m, cfg.grid, cfg.smem);
  auto go = [&](auto kernel, auto id) {
    bard_status s = prep<decltype(id)::value>(kernel, "bard_crba");
    if (s != BARD_OK) return s;
    launch(kernel, cfg, stream, (const void*)m.d_blob, (uint32_t)m.common_bytes, (uint32_t)m.m_bytes, (int)m.crba_warps, cfg.rcpL,
           cfg.team_rows, (int)m.nq, (int)m.nv, (int)m.nslots, (uint32_t)B, q, M, vec_ok);
    return finish("bard_crba");
  };
  return BARD_DISPATCH(crba_kernel, 12, m.simple, cfg.pack, go);
}

}  // namespace bard
