// Host-side model builder: validation, offsets, level schedule, ancestor masks, Rodrigues
// constants (eq. (2)-(3)), motion subspaces, compact inertias, slot allocation for the
// outward sweeps, and the single upload of the constant blob.  All precompute is fp64, rounded once to fp32.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "bard_internal.h"

namespace bard {

namespace {

struct M3 { double m[9]; };
struct V3 { double v[3]; };

M3 mul(const M3& a, const M3& b) {
  M3 c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double s = 0;
      for (int k = 0; k < 3; ++k) s += a.m[3 * i + k] * b.m[3 * k + j];
      c.m[3 * i + j] = s;
    }
  return c;
}
V3 mul(const M3& a, const V3& x) {
  V3 y;
  for (int i = 0; i < 3; ++i) y.v[i] = a.m[3 * i] * x.v[0] + a.m[3 * i + 1] * x.v[1] + a.m[3 * i + 2] * x.v[2];
  return y;
}
M3 transpose(const M3& a) {
  M3 c;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) c.m[3 * i + j] = a.m[3 * j + i];
  return c;
}
M3 hat(const V3& k) {  // [k]x
  M3 c = {{0, -k.v[2], k.v[1], k.v[2], 0, -k.v[0], -k.v[1], k.v[0], 0}};
  return c;
}
V3 cross(const V3& a, const V3& b) {
  V3 c = {{a.v[1] * b.v[2] - a.v[2] * b.v[1], a.v[2] * b.v[0] - a.v[0] * b.v[2], a.v[0] * b.v[1] - a.v[1] * b.v[0]}};
  return c;
}
void split12(const double* T, M3& R, V3& t) {
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) R.m[3 * i + j] = T[4 * i + j];
    t.v[i] = T[4 * i + 3];
  }
}
bool is_identity12(const double* T) {
  static const double I[12] = {1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0};
  for (int k = 0; k < 12; ++k)
    if (std::fabs(T[k] - I[k]) > 1e-12) return false;
  return true;
}
void put(float* dst, const double* src, int n) {
  for (int k = 0; k < n; ++k) dst[k] = (float)src[k];
}

}  // namespace

bard_status set_frames(Model& M, int32_t nframes, const int32_t* body, const double* offset);

bard_status build_model(const bard_model_desc* d, int device, Model& M) {
  if (!d || d->nb < 1 || !d->parent || !d->joint_type || !d->T_pre || !d->mass || !d->com || !d->inertia) {
    set_error("bard_model_create: NULL pointer in description or nb < 1");
    return BARD_ERR_INVALID_ARG;
  }
  const int nb = d->nb;
  if (nb > BARD_MAX_BODIES) {
    set_error("bard_model_create: nb exceeds BARD_MAX_BODIES");
    return BARD_ERR_UNSUPPORTED;
  }
  for (int i = 0; i < nb; ++i) {
    int t = d->joint_type[i];
    if (t < 0 || t > 3) { set_error("bard_model_create: unknown joint type"); return BARD_ERR_INVALID_ARG; }
    if (d->parent[i] >= i || d->parent[i] < -1) {
      set_error("bard_model_create: parent[i] must be in {-1, 0..i-1}");
      return BARD_ERR_TOPOLOGY;
    }
    // mass >= 0: massless links (URDF base / tool / sensor frames behind fixed joints) are legal for FK, Jacobian,
    // RNEA and CRBA; only ABA needs a positive-definite articulated inertia under every DOF (checked there)
    if (!(d->mass[i] >= 0.0)) { set_error("bard_model_create: mass must be >= 0"); return BARD_ERR_INVALID_ARG; }
    if ((t == BARD_JOINT_REVOLUTE || t == BARD_JOINT_PRISMATIC)) {
      if (!d->axis) { set_error("bard_model_create: axis is NULL"); return BARD_ERR_INVALID_ARG; }
      const double* a = d->axis + 3 * i;
      if (std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]) < 1e-12) {
        set_error("bard_model_create: zero-length joint axis");
        return BARD_ERR_INVALID_ARG;
      }
    }
    if (t == BARD_JOINT_FREE && d->T_post && !is_identity12(d->T_post + 12 * i)) {
      set_error("bard_model_create: T_post must be identity on a free joint");
      return BARD_ERR_INVALID_ARG;
    }
  }
  M.device = device;
  options_from_env(M.opt);
  M.nb = nb;
  M.parent.assign(d->parent, d->parent + nb);
  M.jtype.assign(d->joint_type, d->joint_type + nb);

  // offsets
  static const int NQ[4] = {1, 1, 0, 7}, NV[4] = {1, 1, 0, 6};
  M.q_off.assign(nb + 1, 0);
  M.v_off.assign(nb + 1, 0);
  for (int i = 0; i < nb; ++i) {
    M.q_off[i + 1] = M.q_off[i] + NQ[M.jtype[i]];
    M.v_off[i + 1] = M.v_off[i] + NV[M.jtype[i]];
  }
  M.nq = M.q_off[nb];
  M.nv = M.v_off[nb];
  if (M.nv > BARD_MAX_DOF) { set_error("bard_model_create: nv exceeds BARD_MAX_DOF"); return BARD_ERR_UNSUPPORTED; }
  M.dof_body.clear();
  for (int i = 0; i < nb; ++i)
    for (int k = 0; k < NV[M.jtype[i]]; ++k) M.dof_body.push_back(i);

  // level schedule: level 0 = attached to world; inside a level ascending body index
  M.body_level.assign(nb, 0);
  int nl = 0;
  for (int i = 0; i < nb; ++i) {
    M.body_level[i] = M.parent[i] < 0 ? 0 : M.body_level[M.parent[i]] + 1;
    if (M.body_level[i] + 1 > nl) nl = M.body_level[i] + 1;
  }
  M.nlevels = nl;
  M.level_ptr.assign(nl + 1, 0);
  for (int i = 0; i < nb; ++i) M.level_ptr[M.body_level[i] + 1]++;
  for (int l = 0; l < nl; ++l) M.level_ptr[l + 1] += M.level_ptr[l];
  M.level_body.assign(nb, 0);
  std::vector<int32_t> slot_of(nb, -1), cursor(M.level_ptr.begin(), M.level_ptr.end() - 1);
  for (int i = 0; i < nb; ++i) {
    int s = cursor[M.body_level[i]]++;
    M.level_body[s] = i;
    slot_of[i] = s;
  }
  M.parent_slot.assign(nb, -1);
  for (int s = 0; s < nb; ++s) {
    int p = M.parent[M.level_body[s]];
    M.parent_slot[s] = p < 0 ? -1 : slot_of[p];
  }
  M.anc_mask.assign(nb, 0);
  for (int i = 0; i < nb; ++i) M.anc_mask[i] = (1ull << i) | (M.parent[i] < 0 ? 0ull : M.anc_mask[M.parent[i]]);

  // ---- level-parallel team schedule: L warps share one 32-environment tile.
  std::vector<std::vector<int32_t>> children(nb);
  for (int i = 0; i < nb; ++i)
    if (M.parent[i] >= 0) children[M.parent[i]].push_back(i);
  int maxw = 1;
  for (int l = 0; l < nl; ++l) maxw = std::max(maxw, (int)(M.level_ptr[l + 1] - M.level_ptr[l]));
  int L = std::min(maxw, 8);
  if (const char* ev = std::getenv("BARD_TEAM_WARPS")) {   // tuning knob for experiments
    int v = std::atoi(ev);
    if (v >= 1 && v <= 8) L = v;
  }
  M.team_warps = L;
  // Bodies of a level go to warps: a body continues on its parent's warp when the parent was that warp's
  // last task (its state is then still in registers); the others go to the least loaded warp.
  M.warp_of.assign(nb, 0);
  std::vector<std::vector<uint16_t>> tasks(L);
  std::vector<int32_t> last_task(L, -1), total(L, 0), src(nb, -1), save(nb, -1);
  std::vector<char> reg_fed(nb, 0);
  for (int l = 0; l < nl; ++l) {
    std::vector<std::vector<int32_t>> mine(L);
    std::vector<int32_t> load(L, 0);
    std::vector<char> claimed(L, 0), placed(nb, 0);
    for (int s = M.level_ptr[l]; s < M.level_ptr[l + 1]; ++s) {
      const int b = M.level_body[s], p = M.parent[b];
      if (p < 0) continue;
      const int w = M.warp_of[p];
      if (last_task[w] == p && !claimed[w]) {
        claimed[w] = 1; placed[b] = 1; reg_fed[b] = 1;
        M.warp_of[b] = w; mine[w].push_back(b); load[w]++;
      }
    }
    for (int s = M.level_ptr[l]; s < M.level_ptr[l + 1]; ++s) {
      const int b = M.level_body[s];
      if (placed[b]) continue;
      int best = 0;
      for (int w = 1; w < L; ++w)
        if (load[w] < load[best] || (load[w] == load[best] && total[w] < total[best])) best = w;
      M.warp_of[b] = best; mine[best].push_back(b); load[best]++;
    }
    for (int w = 0; w < L; ++w) {
      if (mine[w].empty()) {
        tasks[w].push_back((uint16_t)(TASK_NOOP | TASK_BAR));
      } else {
        for (size_t k = 0; k < mine[w].size(); ++k)
          tasks[w].push_back((uint16_t)(mine[w][k] | (k + 1 == mine[w].size() ? TASK_BAR : 0)));
        last_task[w] = mine[w].back();
        total[w] += (int)mine[w].size();
      }
    }
  }
  int nslots = 0;
  for (int i = 0; i < nb; ++i) {
    bool need = false;
    for (int c : children[i]) need = need || !reg_fed[c];
    if (need) save[i] = nslots++;
  }
  for (int i = 0; i < nb; ++i) src[i] = M.parent[i] < 0 ? -1 : (reg_fed[i] ? -2 : save[M.parent[i]]);
  M.nslots = nslots;
  // CRBA runs with Lc >= L warps per team: the extra warps idle through the level sweeps (barrier-only task
  // lists) and share the fill of M, which parallelises over rows, not over tree levels.
  int Lc = std::min(8, std::max(L, (M.nv + 3) / 4));
  if (const char* ev = std::getenv("BARD_CRBA_WARPS")) {   // tuning knob for experiments
    int v = std::atoi(ev);
    if (v >= L && v <= 8) Lc = v;
  }
  M.crba_warps = Lc;
  tasks.resize(Lc);
  for (int w = L; w < Lc; ++w)
    for (int l = 0; l < nl; ++l) tasks[w].push_back((uint16_t)(TASK_NOOP | TASK_BAR));
  size_t task_stride = 0;
  for (int w = 0; w < Lc; ++w) task_stride = std::max(task_stride, tasks[w].size() + 1);
  task_stride = (task_stride + 7) & ~(size_t)7;
  // ---- CRBA fill tables.  rel[i]: DOFs j <= i on ancestor-or-self bodies of DOF i (the non-zero part of
  // row i of the lower triangle).  Rows go to warps by longest-processing-time greedy on popcount(rel).
  std::vector<uint64_t> rel(M.nv, 0);
  for (int i = 0; i < M.nv; ++i)
    for (int j = 0; j <= i; ++j)
      if ((M.anc_mask[M.dof_body[i]] >> M.dof_body[j]) & 1) rel[i] |= 1ull << j;
  std::vector<std::vector<uint8_t>> fill(Lc);
  {
    std::vector<int> order(M.nv);
    for (int i = 0; i < M.nv; ++i) order[i] = i;
    auto pc = [&](int i) { return __builtin_popcountll(rel[i]); };
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return pc(x) > pc(y); });
    std::vector<int64_t> work(Lc, 0);
    for (int i : order) {
      int best = 0;
      for (int w = 1; w < Lc; ++w)
        if (work[w] < work[best]) best = w;
      fill[best].push_back((uint8_t)i);
      work[best] += pc(i) + 2;
    }
  }
  size_t fill_stride = 0;
  for (int w = 0; w < Lc; ++w) fill_stride = std::max(fill_stride, fill[w].size() + 1);
  fill_stride = (fill_stride + 15) & ~(size_t)15;
  std::vector<uint16_t> zrows;   // structurally zero entries of M, both triangles
  for (int i = 0; i < M.nv; ++i)
    for (int j = 0; j < M.nv; ++j) {
      const int hi = std::max(i, j), lo = std::min(i, j);
      if (!((rel[hi] >> lo) & 1)) zrows.push_back((uint16_t)(i * M.nv + j));
    }
  while (zrows.size() % 4) zrows.push_back(0xffff);

  M.simple = true;
  for (int i = 0; i < nb; ++i) {
    const int t = M.jtype[i];
    const bool post_id = !d->T_post || is_identity12(d->T_post + 12 * i);
    if (!(t == BARD_JOINT_FREE || (t == BARD_JOINT_REVOLUTE && post_id))) M.simple = false;
  }
  if (const char* ev = std::getenv("BARD_FORCE_GENERAL"))   // test knob: run the general kernels on simple models
    if (std::atoi(ev)) M.simple = false;

  // ---- constant sections COMMON | M
  auto align16 = [](size_t x) { return (x + 15) & ~(size_t)15; };
  const size_t off_bodies = sizeof(BlobHeader);
  const size_t off_tasks = off_bodies + sizeof(BodyConst) * nb;
  const size_t off_children = align16(off_tasks + sizeof(uint16_t) * Lc * task_stride);
  const size_t off_dof_body = align16(off_children + (size_t)nb);
  M.common_bytes = align16(off_dof_body + (size_t)M.nv);
  const size_t m_off_fill = sizeof(MHeader);
  const size_t m_off_rel = align16(m_off_fill + (size_t)Lc * fill_stride);
  const size_t m_off_zrows = align16(m_off_rel + sizeof(uint64_t) * M.nv);
  std::vector<uint8_t> pairs, fanc;
  std::vector<uint16_t> pair_ptr(M.nv + 1, 0), fanc_ptr(M.nv + 1, 0);
  for (int i = 0; i < M.nv; ++i) {
    const int bi = M.dof_body[i];
    for (int j = 0; j <= i; ++j) {
      const int bj = M.dof_body[j];
      if (((rel[i] >> j) & 1) && !(M.jtype[bj] == BARD_JOINT_FREE && bj != bi)) pairs.push_back((uint8_t)j);
    }
    pair_ptr[i + 1] = (uint16_t)pairs.size();
    for (int b = 0; b < bi; ++b)
      if (M.jtype[b] == BARD_JOINT_FREE && ((M.anc_mask[bi] >> b) & 1)) fanc.push_back((uint8_t)b);
    fanc_ptr[i + 1] = (uint16_t)fanc.size();
  }
  const size_t m_off_pairs = align16(m_off_zrows + sizeof(uint16_t) * zrows.size());
  const size_t m_off_pair_ptr = align16(m_off_pairs + pairs.size());
  const size_t m_off_fanc = align16(m_off_pair_ptr + sizeof(uint16_t) * pair_ptr.size());
  const size_t m_off_fanc_ptr = align16(m_off_fanc + fanc.size());
  M.m_bytes = align16(m_off_fanc_ptr + sizeof(uint16_t) * fanc_ptr.size());
  M.blob.assign(M.common_bytes + M.m_bytes, 0);
  BlobHeader* H = reinterpret_cast<BlobHeader*>(M.blob.data());
  H->nb = nb; H->nq = M.nq; H->nv = M.nv; H->nlevels = nl; H->nslots = nslots;
  for (int k = 0; k < 3; ++k) H->g[k] = (float)d->gravity[k];
  H->team_warps = L;
  H->off_tasks = (int32_t)off_tasks; H->task_stride = (int32_t)task_stride;
  H->off_children = (int32_t)off_children;
  H->off_dof_body = (int32_t)off_dof_body;
  H->simple = M.simple ? 1 : 0;
  {
    uint16_t* T = reinterpret_cast<uint16_t*>(M.blob.data() + off_tasks);
    for (int w = 0; w < Lc; ++w) {
      for (size_t k = 0; k < task_stride; ++k) T[w * task_stride + k] = TASK_END;
      for (size_t k = 0; k < tasks[w].size(); ++k) T[w * task_stride + k] = tasks[w][k];
    }
    uint8_t* D = M.blob.data() + off_dof_body;
    for (int j = 0; j < M.nv; ++j) D[j] = (uint8_t)M.dof_body[j];
    unsigned char* MS = M.blob.data() + M.common_bytes;
    MHeader* MH = reinterpret_cast<MHeader*>(MS);
    MH->off_fill = (int32_t)m_off_fill; MH->fill_stride = (int32_t)fill_stride;
    MH->off_rel = (int32_t)m_off_rel; MH->off_zrows = (int32_t)m_off_zrows; MH->nzrows = (int32_t)zrows.size();
    uint8_t* F = MS + m_off_fill;
    for (int w = 0; w < Lc; ++w) {
      for (size_t k = 0; k < fill_stride; ++k) F[w * fill_stride + k] = 0xff;
      for (size_t k = 0; k < fill[w].size(); ++k) F[w * fill_stride + k] = fill[w][k];
    }
    if (M.nv) std::memcpy(MS + m_off_rel, rel.data(), sizeof(uint64_t) * M.nv);
    if (!zrows.empty()) std::memcpy(MS + m_off_zrows, zrows.data(), sizeof(uint16_t) * zrows.size());
    MH->off_pairs = (int32_t)m_off_pairs; MH->off_pair_ptr = (int32_t)m_off_pair_ptr;
    if (!pairs.empty()) std::memcpy(MS + m_off_pairs, pairs.data(), pairs.size());
    std::memcpy(MS + m_off_pair_ptr, pair_ptr.data(), sizeof(uint16_t) * pair_ptr.size());
    MH->off_fanc = (int32_t)m_off_fanc; MH->off_fanc_ptr = (int32_t)m_off_fanc_ptr;
    if (!fanc.empty()) std::memcpy(MS + m_off_fanc, fanc.data(), fanc.size());
    std::memcpy(MS + m_off_fanc_ptr, fanc_ptr.data(), sizeof(uint16_t) * fanc_ptr.size());
  }
  std::vector<int32_t> child_begin(nb, 0);
  {
    uint8_t* C = M.blob.data() + off_children;
    int pos = 0;
    for (int i = 0; i < nb; ++i) {
      child_begin[i] = pos;
      for (int c : children[i]) C[pos++] = (uint8_t)c;
    }
  }
  BodyConst* BC = reinterpret_cast<BodyConst*>(M.blob.data() + sizeof(BlobHeader));
  M.rodrigues.assign((size_t)nb * 36, 0.f);
  M.bc64.assign((size_t)nb * kBc64, 0.0);
  for (int k = 0; k < 3; ++k) M.g64[k] = d->gravity[k];
  M.free_index.assign(nb, -1);
  for (int i = 0; i < nb; ++i) {
    BodyConst& c = BC[i];
    const int t = M.jtype[i];
    M3 Rpre, Rpost = {{1, 0, 0, 0, 1, 0, 0, 0, 1}};
    V3 tpre, tpost = {{0, 0, 0}};
    split12(d->T_pre + 12 * i, Rpre, tpre);
    bool post_id = true;
    if (d->T_post) { split12(d->T_post + 12 * i, Rpost, tpost); post_id = is_identity12(d->T_post + 12 * i); }
    V3 ax = {{0, 0, 0}};
    if (t == BARD_JOINT_REVOLUTE || t == BARD_JOINT_PRISMATIC) {
      const double* a = d->axis + 3 * i;
      double n = std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
      for (int k = 0; k < 3; ++k) ax.v[k] = a[k] / n;
    }
    double rod[36];
    std::memset(rod, 0, sizeof(rod));
    M3 R0 = mul(Rpre, Rpost);
    V3 t0 = mul(Rpre, tpost);
    for (int k = 0; k < 3; ++k) t0.v[k] += tpre.v[k];
    std::memcpy(rod, R0.m, sizeof(R0.m));
    std::memcpy(rod + 27, t0.v, sizeof(t0.v));
    double Sw[3] = {0, 0, 0}, Sl[3] = {0, 0, 0};
    if (t == BARD_JOINT_REVOLUTE) {
      M3 K = hat(ax), K2 = mul(K, K);
      M3 RK = mul(Rpre, K), RK2 = mul(Rpre, K2);
      M3 A = mul(RK, Rpost), Bm = mul(RK2, Rpost);
      V3 a = mul(RK, tpost), b = mul(RK2, tpost);
      std::memcpy(rod + 9, A.m, sizeof(A.m));
      std::memcpy(rod + 18, Bm.m, sizeof(Bm.m));
      std::memcpy(rod + 30, a.v, sizeof(a.v));
      std::memcpy(rod + 33, b.v, sizeof(b.v));
      // S = X_post^{-1} [axis; 0] in the body frame: w = Rpost^T axis, l = Rpost^T (axis x tpost)
      M3 Rt = transpose(Rpost);
      V3 w = mul(Rt, ax), l = mul(Rt, cross(ax, tpost));
      for (int k = 0; k < 3; ++k) { Sw[k] = w.v[k]; Sl[k] = l.v[k]; }
    } else if (t == BARD_JOINT_PRISMATIC) {
      V3 a = mul(Rpre, ax);
      std::memcpy(rod + 30, a.v, sizeof(a.v));
      V3 l = mul(transpose(Rpost), ax);
      for (int k = 0; k < 3; ++k) Sl[k] = l.v[k];
    } else if (t == BARD_JOINT_FREE) {
      std::memcpy(rod, Rpre.m, sizeof(Rpre.m));
      std::memcpy(rod + 27, tpre.v, sizeof(tpre.v));
    }
    put(c.R0, rod, 36);
    put(&M.rodrigues[(size_t)36 * i], rod, 36);
    put(c.Sw, Sw, 3);
    put(c.Sl, Sl, 3);
    double* c64 = &M.bc64[(size_t)kBc64 * i];
    std::memcpy(c64, rod, sizeof(rod));
    std::memcpy(c64 + 36, Sw, sizeof(Sw));
    std::memcpy(c64 + 39, Sl, sizeof(Sl));
    // compact spatial inertia about the body origin: m, h = m c, Io = Ic + m (|c|^2 1 - c c^T)
    const double m = d->mass[i];
    const double* cm = d->com + 3 * i;
    const double* Ic = d->inertia + 6 * i;
    const double c2 = cm[0] * cm[0] + cm[1] * cm[1] + cm[2] * cm[2];
    double Io[6] = {Ic[0] + m * (c2 - cm[0] * cm[0]), Ic[1] - m * cm[0] * cm[1], Ic[2] - m * cm[0] * cm[2],
                    Ic[3] + m * (c2 - cm[1] * cm[1]), Ic[4] - m * cm[1] * cm[2], Ic[5] + m * (c2 - cm[2] * cm[2])};
    double h[3] = {m * cm[0], m * cm[1], m * cm[2]};
    c.mass = (float)m;
    put(c.h, h, 3);
    put(c.Io, Io, 6);
    c64[42] = m;
    std::memcpy(c64 + 43, h, sizeof(h));
    std::memcpy(c64 + 46, Io, sizeof(Io));
    c.type = t; c.parent = M.parent[i]; c.q_off = M.q_off[i]; c.v_off = M.v_off[i];
    c.src = src[i]; c.save = save[i]; c.flags = post_id ? 1 : 0; c.level = M.body_level[i];
    if (t == BARD_JOINT_FREE) { M.free_index[i] = M.nfree; c.flags |= (M.nfree++) << 8; }
    c.anc_lo = (uint32_t)M.anc_mask[i]; c.anc_hi = (uint32_t)(M.anc_mask[i] >> 32);
    c.child_begin = child_begin[i]; c.child_count = (int32_t)children[i].size();
  }

  // where rnea_kernel parks the staged input rows: in the rows that later hold the body's force (see rnea_kernel)
  for (int i = 0; i < nb; ++i) {
    const int reg = 12 * nslots + 8 * i, qo = M.q_off[i], vo = M.v_off[i];
    if (M.jtype[i] == BARD_JOINT_FREE) {
      const int fi = 12 * nslots + 8 * nb + 19 * M.free_index[i];
      for (int k = 0; k < 7 && qo + k < 128; ++k) M.rowmap_q[qo + k] = (uint16_t)(fi + k);
      for (int k = 0; k < 6; ++k) { M.rowmap_qd[vo + k] = (uint16_t)(fi + 7 + k); M.rowmap_qdd[vo + k] = (uint16_t)(fi + 13 + k); }
    } else if (M.jtype[i] != BARD_JOINT_FIXED) {
      M.rowmap_q[qo] = (uint16_t)(reg + 6); M.rowmap_qd[vo] = (uint16_t)reg; M.rowmap_qdd[vo] = (uint16_t)(reg + 1);
    }
  }
  set_frames(M, 0, nullptr, nullptr);   // empty J section (host side; the device copy follows below)
  if (device < 0) return BARD_OK;  // host-only model: tables can be queried, operators refuse to run
  int dev_count = 0;
  cudaError_t e = cudaGetDeviceCount(&dev_count);
  if (e != cudaSuccess || device >= dev_count) {
    set_error(std::string("bard_model_create: no such CUDA device: ") + cudaGetErrorString(e));
    cudaGetLastError();
    return BARD_ERR_CUDA;
  }
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(device);
  cudaDeviceGetAttribute(&M.sm_count, cudaDevAttrMultiProcessorCount, device);
  e = cudaMalloc(&M.d_blob, M.blob.size());
  if (e == cudaSuccess) e = cudaMalloc(&M.d_jblob, kJBlobMax);
  if (e == cudaSuccess) e = cudaMemcpy(M.d_blob, M.blob.data(), M.blob.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(M.d_jblob, M.jblob.data(), M.jblob.size(), cudaMemcpyHostToDevice);
  cudaSetDevice(prev);
  if (e != cudaSuccess) {
    set_error(std::string("bard_model_create: ") + cudaGetErrorString(e));
    if (M.d_blob) cudaFree(M.d_blob);
    if (M.d_jblob) cudaFree(M.d_jblob);
    M.d_blob = M.d_jblob = nullptr;
    return e == cudaErrorMemoryAllocation ? BARD_ERR_ALLOC : BARD_ERR_CUDA;
  }
  return BARD_OK;
}

// J section: frames, the non-zero columns (frame, dof) and the flat indices of the zero rows of J.
bard_status set_frames(Model& M, int32_t nframes, const int32_t* body, const double* offset) {
  if (nframes < 0 || (nframes > 0 && !body)) { set_error("bard_model_set_frames: bad arguments"); return BARD_ERR_INVALID_ARG; }
  if (nframes > BARD_MAX_FRAMES) { set_error("bard_model_set_frames: too many frames"); return BARD_ERR_UNSUPPORTED; }
  for (int f = 0; f < nframes; ++f)
    if (body[f] < 0 || body[f] >= M.nb) { set_error("bard_model_set_frames: frame body out of range"); return BARD_ERR_INVALID_ARG; }
  auto align16 = [](size_t x) { return (x + 15) & ~(size_t)15; };
  std::vector<uint16_t> cols, zrows;
  uint64_t uni = 0;
  for (int f = 0; f < nframes; ++f) {
    const uint64_t a = M.anc_mask[body[f]];
    uni |= a;
    for (int j = 0; j < M.nv; ++j) {
      if ((a >> M.dof_body[j]) & 1) cols.push_back((uint16_t)((f << 8) | j));
      else
        for (int r = 0; r < 6; ++r) zrows.push_back((uint16_t)((f * 6 + r) * M.nv + j));
    }
  }
  while (zrows.size() % 4) zrows.push_back(0xffff);
  const size_t off_frames = sizeof(JHeader);
  const size_t off_cols = off_frames + sizeof(FrameConst) * BARD_MAX_FRAMES;
  const size_t off_zrows = align16(off_cols + sizeof(uint16_t) * cols.size());
  const size_t off_bframes = align16(off_zrows + sizeof(uint16_t) * zrows.size());
  const size_t bytes = align16(off_bframes + sizeof(uint16_t) * M.nb);
  if (bytes > kJBlobMax) { set_error("bard_model_set_frames: internal: J section too large"); return BARD_ERR_UNSUPPORTED; }
  M.jblob.assign(bytes, 0);
  JHeader* JH = reinterpret_cast<JHeader*>(M.jblob.data());
  JH->nframes = nframes;
  JH->jmask_lo = (uint32_t)uni; JH->jmask_hi = (uint32_t)(uni >> 32);
  JH->off_cols = (int32_t)off_cols; JH->ncols = (int32_t)cols.size();
  JH->off_zrows = (int32_t)off_zrows; JH->nzrows = (int32_t)zrows.size();
  JH->off_bframes = (int32_t)off_bframes;
  {
    uint16_t* BF = reinterpret_cast<uint16_t*>(M.jblob.data() + off_bframes);
    for (int f = 0; f < nframes; ++f) BF[body[f]] |= (uint16_t)(1u << f);
  }
  FrameConst* F = reinterpret_cast<FrameConst*>(M.jblob.data() + off_frames);
  for (int f = 0; f < nframes; ++f) {
    F[f].body = body[f];
    for (int k = 0; k < 3; ++k) F[f].off[k] = offset ? (float)offset[3 * f + k] : 0.f;
    const uint64_t a = M.anc_mask[body[f]];
    F[f].anc_lo = (uint32_t)a; F[f].anc_hi = (uint32_t)(a >> 32);
  }
  if (!cols.empty()) std::memcpy(M.jblob.data() + off_cols, cols.data(), sizeof(uint16_t) * cols.size());
  if (!zrows.empty()) std::memcpy(M.jblob.data() + off_zrows, zrows.data(), sizeof(uint16_t) * zrows.size());
  M.j_bytes = bytes;
  M.nframes = nframes;
  M.frame_off64.assign((size_t)nframes * 3, 0.0);
  for (int k = 0; k < 3 * nframes && offset; ++k) M.frame_off64[k] = offset[k];
  if (!M.d_jblob) return BARD_OK;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(M.device);
  cudaError_t e = cudaMemcpy(M.d_jblob, M.jblob.data(), bytes, cudaMemcpyHostToDevice);
  cudaSetDevice(prev);
  if (e != cudaSuccess) { set_error(std::string("bard_model_set_frames: ") + cudaGetErrorString(e)); return BARD_ERR_CUDA; }
  return BARD_OK;
}

}  // namespace bard
