/*
 * bard_oracle.c -- fp64 CPU oracle (TEST INFRASTRUCTURE, see bard_oracle.h).
 *
 * Plain dense restatement of Featherstone's recursions, one environment at a time, in body
 * order (no level schedule, no compact 3-vector algebra, no Rodrigues constants on the main
 * path: T_joint * R_axis(q) * T_link is multiplied out as 4x4 matrices, eq. (1)).
 * Spatial vectors are 6-vectors [angular; linear], spatial transforms and inertias are dense
 * 6x6 matrices.  The only parallelism is an OpenMP loop over independent environments.
 *
 * Passages followed: eq. (1)-(5) PAPER.md:59-81; level grouping PAPER.md:87; eq. (6)
 * PAPER.md:89; backward pass PAPER.md:91; eq. (7); X^T M X PAPER.md:103;
 * Featherstone RBDA (ref. [5]) Table 5.1 (RNEA) and Table 6.2 (CRBA) as restated in
 * SURVEY.md section 8(c) items 1-9.
 */
#include "bard_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MAXB 64 /* bodies; matches the 64-bit ancestor mask */

enum { JT_REVOLUTE = 0, JT_PRISMATIC = 1, JT_FIXED = 2, JT_FREE = 3 };

static int g_threads = 0;

void bard_oracle_set_threads(int n) { g_threads = n; }
int bard_oracle_get_threads(void) {
#ifdef _OPENMP
  return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------ small dense algebra */

static void mat_mul(const double* A, const double* B, double* C, int n, int k, int m) {
  /* C[n x m] = A[n x k] * B[k x m], row-major */
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < m; ++j) {
      double s = 0.0;
      for (int l = 0; l < k; ++l) s += A[i * k + l] * B[l * m + j];
      C[i * m + j] = s;
    }
}

static void mat_transpose(const double* A, double* At, int n, int m) {
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < m; ++j) At[j * n + i] = A[i * m + j];
}

static void skew(const double v[3], double K[9]) {
  /* K = [v]x : K w = v x w */
  K[0] = 0.0;   K[1] = -v[2]; K[2] = v[1];
  K[3] = v[2];  K[4] = 0.0;   K[5] = -v[0];
  K[6] = -v[1]; K[7] = v[0];  K[8] = 0.0;
}

static void cross3(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

static void mat4_identity(double T[16]) {
  memset(T, 0, 16 * sizeof(double));
  T[0] = T[5] = T[10] = T[15] = 1.0;
}

static void mat4_from_Rt12(const double* Rt /* rows r0 r1 r2 t */, double T[16]) {
  /* input: 3 rows of 4 (R | t) */
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 4; ++j) T[i * 4 + j] = Rt[i * 4 + j];
  T[12] = T[13] = T[14] = 0.0;
  T[15] = 1.0;
}

static void mat4_get_R(const double T[16], double R[9]) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) R[i * 3 + j] = T[i * 4 + j];
}
static void mat4_get_t(const double T[16], double t[3]) {
  for (int i = 0; i < 3; ++i) t[i] = T[i * 4 + 3];
}

/* ------------------------------------------------------------------ model bookkeeping */

typedef struct {
  int nb, nq, nv;
  int parent[MAXB], jtype[MAXB], qoff[MAXB + 1], voff[MAXB + 1], nvi[MAXB];
  double axis[MAXB][3];
  double Tpre[MAXB][16], Tpost[MAXB][16];
  double S[MAXB][36];   /* 6 x nvi, row-major with row stride nvi, internal order [ang; lin] */
  double I[MAXB][36];   /* spatial inertia, internal order */
  double a_world[6];    /* [0; -g] */
} omodel;

static int joint_nq(int t) { return t == JT_REVOLUTE || t == JT_PRISMATIC ? 1 : (t == JT_FREE ? 7 : 0); }
static int joint_nv(int t) { return t == JT_REVOLUTE || t == JT_PRISMATIC ? 1 : (t == JT_FREE ? 6 : 0); }

static int build_model(const bard_oracle_desc* d, omodel* m) {
  if (!d || d->nb < 1 || d->nb > MAXB || !d->parent || !d->joint_type || !d->T_pre) return 1;
  m->nb = d->nb;
  m->qoff[0] = m->voff[0] = 0;
  for (int i = 0; i < d->nb; ++i) {
    int p = d->parent[i], t = d->joint_type[i];
    if (p < -1 || p >= i) return 2;
    if (t < 0 || t > 3) return 3;
    m->parent[i] = p;
    m->jtype[i] = t;
    m->nvi[i] = joint_nv(t);
    m->qoff[i + 1] = m->qoff[i] + joint_nq(t);
    m->voff[i + 1] = m->voff[i] + joint_nv(t);

    /* normalised axis ("normalised axis") */
    double ax[3] = {0, 0, 0};
    if (t == JT_REVOLUTE || t == JT_PRISMATIC) {
      if (!d->axis) return 4;
      double n = sqrt(d->axis[3 * i] * d->axis[3 * i] + d->axis[3 * i + 1] * d->axis[3 * i + 1] +
                      d->axis[3 * i + 2] * d->axis[3 * i + 2]);
      if (!(n > 1e-12)) return 4;
      for (int k = 0; k < 3; ++k) ax[k] = d->axis[3 * i + k] / n;
    }
    for (int k = 0; k < 3; ++k) m->axis[i][k] = ax[k];

    mat4_from_Rt12(d->T_pre + 12 * i, m->Tpre[i]);
    if (d->T_post) mat4_from_Rt12(d->T_post + 12 * i, m->Tpost[i]);
    else mat4_identity(m->Tpost[i]);

    /* motion subspace in the body frame, internal order [ang; lin] */
    double Rpost[9], tpost[3], RpostT[9];
    mat4_get_R(m->Tpost[i], Rpost);
    mat4_get_t(m->Tpost[i], tpost);
    mat_transpose(Rpost, RpostT, 3, 3);
    memset(m->S[i], 0, sizeof(m->S[i]));
    if (t == JT_REVOLUTE) {
      double w[3], axt[3], l[3];
      mat_mul(RpostT, ax, w, 3, 3, 1);
      cross3(ax, tpost, axt);
      mat_mul(RpostT, axt, l, 3, 3, 1);
      for (int k = 0; k < 3; ++k) { m->S[i][k] = w[k]; m->S[i][3 + k] = l[k]; }
    } else if (t == JT_PRISMATIC) {
      double l[3];
      mat_mul(RpostT, ax, l, 3, 3, 1);
      for (int k = 0; k < 3; ++k) m->S[i][3 + k] = l[k];
    } else if (t == JT_FREE) {
      /* API qd = [v_lin; omega] (body frame) -> internal [omega; v]: 6x6 permutation */
      for (int k = 0; k < 3; ++k) {
        m->S[i][(3 + k) * 6 + k] = 1.0;      /* linear rows <- API cols 0..2 */
        m->S[i][k * 6 + (3 + k)] = 1.0;      /* angular rows <- API cols 3..5 */
      }
    }

    /* spatial inertia about the body origin:
       I = [[Ic + m cx cx^T, m cx], [m cx^T, m 1]] */
    double mass = d->mass ? d->mass[i] : 0.0;
    double c[3] = {0, 0, 0};
    if (d->com) for (int k = 0; k < 3; ++k) c[k] = d->com[3 * i + k];
    double Ic[9] = {0};
    if (d->inertia) {
      const double* in = d->inertia + 6 * i;
      Ic[0] = in[0]; Ic[1] = in[1]; Ic[2] = in[2];
      Ic[3] = in[1]; Ic[4] = in[3]; Ic[5] = in[4];
      Ic[6] = in[2]; Ic[7] = in[4]; Ic[8] = in[5];
    }
    double cx[9], cxT[9], cxcxT[9];
    skew(c, cx);
    mat_transpose(cx, cxT, 3, 3);
    mat_mul(cx, cxT, cxcxT, 3, 3, 3);
    double* I = m->I[i];
    for (int r = 0; r < 3; ++r)
      for (int s = 0; s < 3; ++s) {
        I[r * 6 + s] = Ic[r * 3 + s] + mass * cxcxT[r * 3 + s];
        I[r * 6 + 3 + s] = mass * cx[r * 3 + s];
        I[(3 + r) * 6 + s] = mass * cxT[r * 3 + s];
        I[(3 + r) * 6 + 3 + s] = (r == s) ? mass : 0.0;
      }
  }
  m->nq = m->qoff[d->nb];
  m->nv = m->voff[d->nb];
  if (m->nv > MAXB) return 6; /* dense M scratch is MAXB x MAXB */
  for (int k = 0; k < 3; ++k) { m->a_world[k] = 0.0; m->a_world[3 + k] = -d->gravity[k]; }
  return 0;
}

/* joint transform T_J(q) as a 4x4 */
static void joint_T(const omodel* m, int i, const double* qi, double TJ[16]) {
  mat4_identity(TJ);
  int t = m->jtype[i];
  if (t == JT_REVOLUTE) {
    /* Rodrigues: R = I + sin q K + (1 - cos q) K^2 */
    double K[9], K2[9];
    skew(m->axis[i], K);
    mat_mul(K, K, K2, 3, 3, 3);
    double s = sin(qi[0]), c = cos(qi[0]);
    for (int r = 0; r < 3; ++r)
      for (int cc = 0; cc < 3; ++cc)
        TJ[r * 4 + cc] = (r == cc ? 1.0 : 0.0) + s * K[r * 3 + cc] + (1.0 - c) * K2[r * 3 + cc];
  } else if (t == JT_PRISMATIC) {
    for (int k = 0; k < 3; ++k) TJ[k * 4 + 3] = m->axis[i][k] * qi[0];
  } else if (t == JT_FREE) {
    double x = qi[3], y = qi[4], z = qi[5], w = qi[6];
    double n = sqrt(x * x + y * y + z * z + w * w);
    x /= n; y /= n; z /= n; w /= n;
    TJ[0] = 1 - 2 * (y * y + z * z); TJ[1] = 2 * (x * y - z * w);     TJ[2] = 2 * (x * z + y * w);
    TJ[4] = 2 * (x * y + z * w);     TJ[5] = 1 - 2 * (x * x + z * z); TJ[6] = 2 * (y * z - x * w);
    TJ[8] = 2 * (x * z - y * w);     TJ[9] = 2 * (y * z + x * w);     TJ[10] = 1 - 2 * (x * x + y * y);
    TJ[3] = qi[0]; TJ[7] = qi[1]; TJ[11] = qi[2];
  }
}

/* T_pc = T_pre * T_J(q) * T_post, eq. (1) */
static void parent_child_T(const omodel* m, int i, const double* qi, double Tpc[16]) {
  double TJ[16], tmp[16];
  joint_T(m, i, qi, TJ);
  mat_mul(m->Tpre[i], TJ, tmp, 4, 4, 4);
  mat_mul(tmp, m->Tpost[i], Tpc, 4, 4, 4);
}

/* Pluecker motion transform parent -> child from T_pc = (R, t):
   X = [[R^T, 0], [-R^T [t]x, R^T]] */
static void plucker_X(const double Tpc[16], double X[36]) {
  double R[9], t[3], RT[9], tx[9], RTtx[9];
  mat4_get_R(Tpc, R);
  mat4_get_t(Tpc, t);
  mat_transpose(R, RT, 3, 3);
  skew(t, tx);
  mat_mul(RT, tx, RTtx, 3, 3, 3);
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) {
      X[r * 6 + c] = RT[r * 3 + c];
      X[r * 6 + 3 + c] = 0.0;
      X[(3 + r) * 6 + c] = -RTtx[r * 3 + c];
      X[(3 + r) * 6 + 3 + c] = RT[r * 3 + c];
    }
}

/* crm(v) m = v x m (motion cross), crf(v) f = v x* f (force cross) for v = [w; u] */
static void crm(const double v[6], double C[36]) {
  double wx[9], ux[9];
  skew(v, wx);
  skew(v + 3, ux);
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) {
      C[r * 6 + c] = wx[r * 3 + c];
      C[r * 6 + 3 + c] = 0.0;
      C[(3 + r) * 6 + c] = ux[r * 3 + c];
      C[(3 + r) * 6 + 3 + c] = wx[r * 3 + c];
    }
}
static void crf(const double v[6], double C[36]) {
  /* crf(v) = -crm(v)^T */
  double M[36];
  crm(v, M);
  for (int r = 0; r < 6; ++r)
    for (int c = 0; c < 6; ++c) C[r * 6 + c] = -M[c * 6 + r];
}

static void gather_q(const omodel* m, int i, const double* q, int64_t B, int64_t b, double qi[7]) {
  int n = m->qoff[i + 1] - m->qoff[i];
  for (int k = 0; k < n; ++k) qi[k] = q[(int64_t)(m->qoff[i] + k) * B + b];
}

/* ------------------------------------------------------------------ tables (item 9) */

static int body_level_by_walk(const omodel* m, int i) {
  /* explicit walk to the root (a different route than level[parent]+1) */
  int l = 0;
  for (int j = m->parent[i]; j >= 0; j = m->parent[j]) ++l;
  return l;
}

int bard_oracle_dims(const bard_oracle_desc* d, int32_t* nq, int32_t* nv, int32_t* nlevels) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (!rc) {
    int lmax = 0;
    for (int i = 0; i < m->nb; ++i) { int l = body_level_by_walk(m, i); if (l > lmax) lmax = l; }
    if (nq) *nq = m->nq;
    if (nv) *nv = m->nv;
    if (nlevels) *nlevels = lmax + 1;
  }
  free(m);
  return rc;
}

int bard_oracle_table(const bard_oracle_desc* d, int table_id, int64_t* out, int64_t cap) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  if (build_model(d, m)) { free(m); return -1; }
  int nb = m->nb, n = -2;
  int level[MAXB], lmax = 0;
  for (int i = 0; i < nb; ++i) { level[i] = body_level_by_walk(m, i); if (level[i] > lmax) lmax = level[i]; }
  int nlev = lmax + 1;
  /* stable counting sort of bodies by level */
  int count[MAXB + 1] = {0}, ptr[MAXB + 2] = {0}, order[MAXB], fill[MAXB + 1];
  for (int i = 0; i < nb; ++i) count[level[i]]++;
  for (int l = 0; l < nlev; ++l) ptr[l + 1] = ptr[l] + count[l];
  for (int l = 0; l < nlev; ++l) fill[l] = ptr[l];
  for (int i = 0; i < nb; ++i) order[fill[level[i]]++] = i;

  switch (table_id) {
    case BARD_ORACLE_TAB_LEVEL_PTR:
      n = nlev + 1;
      if (n <= cap) for (int l = 0; l <= nlev; ++l) out[l] = ptr[l];
      break;
    case BARD_ORACLE_TAB_LEVEL_BODY:
      n = nb;
      if (n <= cap) for (int s = 0; s < nb; ++s) out[s] = order[s];
      break;
    case BARD_ORACLE_TAB_BODY_LEVEL:
      n = nb;
      if (n <= cap) for (int i = 0; i < nb; ++i) out[i] = level[i];
      break;
    case BARD_ORACLE_TAB_PARENT_SLOT:
      n = nb;
      if (n <= cap)
        for (int s = 0; s < nb; ++s) {
          int p = m->parent[order[s]];
          int64_t slot = -1;
          if (p >= 0) for (int r = 0; r < nb; ++r) if (order[r] == p) slot = r; /* linear search */
          out[s] = slot;
        }
      break;
    case BARD_ORACLE_TAB_Q_OFF:
      n = nb + 1;
      if (n <= cap) for (int i = 0; i <= nb; ++i) out[i] = m->qoff[i];
      break;
    case BARD_ORACLE_TAB_V_OFF:
      n = nb + 1;
      if (n <= cap) for (int i = 0; i <= nb; ++i) out[i] = m->voff[i];
      break;
    case BARD_ORACLE_TAB_DOF_BODY:
      n = m->nv;
      if (n <= cap)
        for (int i = 0; i < nb; ++i)
          for (int k = m->voff[i]; k < m->voff[i + 1]; ++k) out[k] = i;
      break;
    case BARD_ORACLE_TAB_ANC_MASK:
      n = nb;
      if (n <= cap)
        for (int i = 0; i < nb; ++i) {
          uint64_t mask = 0;
          for (int j = i; j >= 0; j = m->parent[j]) mask |= (uint64_t)1 << j;
          out[i] = (int64_t)mask;
        }
      break;
    default: n = -3;
  }
  free(m);
  return n;
}

/* ------------------------------------------------------------------ FK (item 5) */

static void fk_one(const omodel* m, const double* q, int64_t B, int64_t b, double T0[][16]) {
  for (int i = 0; i < m->nb; ++i) {
    double qi[7], Tpc[16];
    gather_q(m, i, q, B, b, qi);
    parent_child_T(m, i, qi, Tpc);
    if (m->parent[i] < 0) memcpy(T0[i], Tpc, sizeof(Tpc));
    else mat_mul(T0[m->parent[i]], Tpc, T0[i], 4, 4, 4);
  }
}

int bard_oracle_fk(const bard_oracle_desc* d, int64_t B, const double* q, double* pose) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
#pragma omp parallel for schedule(static) num_threads(bard_oracle_get_threads())
  for (int64_t b = 0; b < B; ++b) {
    double T0[MAXB][16];
    fk_one(m, q, B, b, T0);
    for (int i = 0; i < m->nb; ++i) {
      for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) pose[((int64_t)i * 12 + r * 3 + c) * B + b] = T0[i][r * 4 + c];
      for (int r = 0; r < 3; ++r) pose[((int64_t)i * 12 + 9 + r) * B + b] = T0[i][r * 4 + 3];
    }
  }
  free(m);
  return 0;
}

/* ------------------------------------------------------------------ Rodrigues constants, eq. (2)-(5) */

static void rodrigues_constants(const omodel* m, int i, double out[36]) {
  /* R0 = Rpre Rpost ; A = Rpre K Rpost ; B = Rpre K^2 Rpost
     t0 = Rpre tpost + tpre ; a = Rpre K tpost ; b = Rpre K^2 tpost          (eq. (2)-(3))
     prismatic ("handled analogously"): R0, t0 as above, A = B = 0, a = Rpre axis
     (t_pc = t0 + q a), b = 0 ; fixed: R0, t0 only ; free: R0 = Rpre, t0 = tpre, rest 0 (T_post = I). */
  double Rpre[9], tpre[3], Rpost[9], tpost[3], K[9], K2[9], tmp[9];
  mat4_get_R(m->Tpre[i], Rpre); mat4_get_t(m->Tpre[i], tpre);
  mat4_get_R(m->Tpost[i], Rpost); mat4_get_t(m->Tpost[i], tpost);
  skew(m->axis[i], K);
  mat_mul(K, K, K2, 3, 3, 3);
  memset(out, 0, 36 * sizeof(double));
  double* R0 = out; double* A = out + 9; double* Bm = out + 18;
  double* t0 = out + 27; double* a = out + 30; double* bb = out + 33;
  mat_mul(Rpre, Rpost, R0, 3, 3, 3);
  mat_mul(Rpre, tpost, t0, 3, 3, 1);
  for (int k = 0; k < 3; ++k) t0[k] += tpre[k];
  if (m->jtype[i] == JT_REVOLUTE) {
    mat_mul(Rpre, K, tmp, 3, 3, 3);  mat_mul(tmp, Rpost, A, 3, 3, 3);
    mat_mul(tmp, tpost, a, 3, 3, 1);
    mat_mul(Rpre, K2, tmp, 3, 3, 3); mat_mul(tmp, Rpost, Bm, 3, 3, 3);
    mat_mul(tmp, tpost, bb, 3, 3, 1);
  } else if (m->jtype[i] == JT_PRISMATIC) {
    mat_mul(Rpre, m->axis[i], a, 3, 3, 1);
  }
}

int bard_oracle_rodrigues(const bard_oracle_desc* d, double* out) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (!rc) for (int i = 0; i < m->nb; ++i) rodrigues_constants(m, i, out + 36 * i);
  free(m);
  return rc;
}

int bard_oracle_fk_rodrigues(const bard_oracle_desc* d, int64_t B, const double* q, double* pose) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  double (*C)[36] = (double (*)[36])malloc(sizeof(double) * 36 * m->nb);
  for (int i = 0; i < m->nb; ++i) rodrigues_constants(m, i, C[i]);
  for (int64_t b = 0; b < B; ++b) {
    double R0w[MAXB][9], p0w[MAXB][3];
    for (int i = 0; i < m->nb; ++i) {
      double qi[7], Rpc[9], tpc[3];
      gather_q(m, i, q, B, b, qi);
      const double* c = C[i];
      if (m->jtype[i] == JT_REVOLUTE) {
        double s = sin(qi[0]), omc = 1.0 - cos(qi[0]);
        for (int k = 0; k < 9; ++k) Rpc[k] = c[k] + s * c[9 + k] + omc * c[18 + k];      /* eq. (4) */
        for (int k = 0; k < 3; ++k) tpc[k] = c[27 + k] + s * c[30 + k] + omc * c[33 + k]; /* eq. (5) */
      } else if (m->jtype[i] == JT_PRISMATIC) {
        for (int k = 0; k < 9; ++k) Rpc[k] = c[k];
        for (int k = 0; k < 3; ++k) tpc[k] = c[27 + k] + qi[0] * c[30 + k];
      } else if (m->jtype[i] == JT_FIXED) {
        for (int k = 0; k < 9; ++k) Rpc[k] = c[k];
        for (int k = 0; k < 3; ++k) tpc[k] = c[27 + k];
      } else {
        double TJ[16], RJ[9];
        joint_T(m, i, qi, TJ);
        mat4_get_R(TJ, RJ);
        mat_mul(c, RJ, Rpc, 3, 3, 3);          /* R0 = Rpre */
        mat_mul(c, qi, tpc, 3, 3, 1);          /* Rpre p */
        for (int k = 0; k < 3; ++k) tpc[k] += c[27 + k];
      }
      int p = m->parent[i];
      if (p < 0) { memcpy(R0w[i], Rpc, sizeof(Rpc)); memcpy(p0w[i], tpc, sizeof(tpc)); }
      else {
        mat_mul(R0w[p], Rpc, R0w[i], 3, 3, 3);
        mat_mul(R0w[p], tpc, p0w[i], 3, 3, 1);
        for (int k = 0; k < 3; ++k) p0w[i][k] += p0w[p][k];
      }
      for (int k = 0; k < 9; ++k) pose[((int64_t)i * 12 + k) * B + b] = R0w[i][k];
      for (int k = 0; k < 3; ++k) pose[((int64_t)i * 12 + 9 + k) * B + b] = p0w[i][k];
    }
  }
  free(C);
  free(m);
  return 0;
}

/* ------------------------------------------------------------------ Jacobian (item 6) */

int bard_oracle_jacobian(const bard_oracle_desc* d, int64_t B, const double* q, double* J) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  if (d->nframes < 0 || (d->nframes > 0 && !d->frame_body)) { free(m); return 5; }
  for (int f = 0; f < d->nframes; ++f)
    if (d->frame_body[f] < 0 || d->frame_body[f] >= m->nb) { free(m); return 5; }
  int nv = m->nv;
#pragma omp parallel for schedule(static) num_threads(bard_oracle_get_threads())
  for (int64_t b = 0; b < B; ++b) {
    double T0[MAXB][16];
    fk_one(m, q, B, b, T0);
    for (int f = 0; f < d->nframes; ++f) {
      int kf = d->frame_body[f];
      double o[3] = {0, 0, 0};
      if (d->frame_offset) for (int k = 0; k < 3; ++k) o[k] = d->frame_offset[3 * f + k];
      double Rk[9], pk[3], pe[3];
      mat4_get_R(T0[kf], Rk); mat4_get_t(T0[kf], pk);
      mat_mul(Rk, o, pe, 3, 3, 1);
      for (int k = 0; k < 3; ++k) pe[k] += pk[k];
      /* zero everything, then fill columns of bodies on the path kf -> root */
      for (int r = 0; r < 6; ++r)
        for (int c = 0; c < nv; ++c) J[(((int64_t)f * 6 + r) * nv + c) * B + b] = 0.0;
      for (int k = kf; k >= 0; k = m->parent[k]) {
        double R[9], p[3];
        mat4_get_R(T0[k], R); mat4_get_t(T0[k], p);
        for (int c = 0; c < m->nvi[k]; ++c) {
          double w[3], l[3], om[3], lin[3], arm[3], oxa[3];
          for (int r = 0; r < 3; ++r) { w[r] = m->S[k][r * m->nvi[k] + c]; l[r] = m->S[k][(3 + r) * m->nvi[k] + c]; }
          mat_mul(R, w, om, 3, 3, 1);
          mat_mul(R, l, lin, 3, 3, 1);
          for (int r = 0; r < 3; ++r) arm[r] = pe[r] - p[r];
          cross3(om, arm, oxa);
          int col = m->voff[k] + c;
          for (int r = 0; r < 3; ++r) {
            J[(((int64_t)f * 6 + r) * nv + col) * B + b] = lin[r] + oxa[r];
            J[(((int64_t)f * 6 + 3 + r) * nv + col) * B + b] = om[r];
          }
        }
      }
    }
  }
  free(m);
  return 0;
}

/* ------------------------------------------------------------------ RNEA (item 7) */

static void joint_velocity(const omodel* m, int i, const double* qd, int64_t B, int64_t b, double vJ[6]) {
  /* vJ = S_i * qd_i */
  int n = m->nvi[i];
  for (int r = 0; r < 6; ++r) {
    double s = 0.0;
    for (int c = 0; c < n; ++c) s += m->S[i][r * n + c] * qd[(int64_t)(m->voff[i] + c) * B + b];
    vJ[r] = s;
  }
}

int bard_oracle_rnea(const bard_oracle_desc* d, int64_t B, const double* q, const double* qd,
                     const double* qdd, double* tau) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
#pragma omp parallel for schedule(static) num_threads(bard_oracle_get_threads())
  for (int64_t b = 0; b < B; ++b) {
    double X[MAXB][36], v[MAXB][6], a[MAXB][6], f[MAXB][6];
    for (int i = 0; i < m->nb; ++i) {
      double qi[7], Tpc[16], vJ[6], aJ[6], Xv[6], Xa[6], C[36], cv[6];
      gather_q(m, i, q, B, b, qi);
      parent_child_T(m, i, qi, Tpc);
      plucker_X(Tpc, X[i]);
      joint_velocity(m, i, qd, B, b, vJ);
      joint_velocity(m, i, qdd, B, b, aJ); /* S * qdd (S is constant in the body frame, c_J = 0) */
      int p = m->parent[i];
      if (p < 0) {
        for (int k = 0; k < 6; ++k) Xv[k] = 0.0;           /* v_world = 0 */
        mat_mul(X[i], m->a_world, Xa, 6, 6, 1);            /* a_world = [0; -g] */
      } else {
        mat_mul(X[i], v[p], Xv, 6, 6, 1);
        mat_mul(X[i], a[p], Xa, 6, 6, 1);
      }
      for (int k = 0; k < 6; ++k) v[i][k] = Xv[k] + vJ[k];
      crm(v[i], C);
      mat_mul(C, vJ, cv, 6, 6, 1);
      for (int k = 0; k < 6; ++k) a[i][k] = Xa[k] + aJ[k] + cv[k];
      /* f = I a + v x* (I v) */
      double Ia[6], Iv[6], Cf[36], vIv[6];
      mat_mul(m->I[i], a[i], Ia, 6, 6, 1);
      mat_mul(m->I[i], v[i], Iv, 6, 6, 1);
      crf(v[i], Cf);
      mat_mul(Cf, Iv, vIv, 6, 6, 1);
      for (int k = 0; k < 6; ++k) f[i][k] = Ia[k] + vIv[k];
    }
    for (int i = m->nb - 1; i >= 0; --i) {
      int n = m->nvi[i];
      for (int c = 0; c < n; ++c) {
        double s = 0.0;
        for (int r = 0; r < 6; ++r) s += m->S[i][r * n + c] * f[i][r];
        tau[(int64_t)(m->voff[i] + c) * B + b] = s;
      }
      int p = m->parent[i];
      if (p >= 0) {
        double XT[36], XTf[6];
        mat_transpose(X[i], XT, 6, 6);
        mat_mul(XT, f[i], XTf, 6, 6, 1);
        for (int k = 0; k < 6; ++k) f[p][k] += XTf[k];
      }
    }
  }
  free(m);
  return 0;
}

int bard_oracle_body_velocity(const bard_oracle_desc* d, int64_t B, const double* q,
                              const double* qd, double* vel) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  for (int64_t b = 0; b < B; ++b) {
    double v[MAXB][6];
    for (int i = 0; i < m->nb; ++i) {
      double qi[7], Tpc[16], X[36], vJ[6], Xv[6];
      gather_q(m, i, q, B, b, qi);
      parent_child_T(m, i, qi, Tpc);
      plucker_X(Tpc, X);
      joint_velocity(m, i, qd, B, b, vJ);
      int p = m->parent[i];
      if (p < 0) for (int k = 0; k < 6; ++k) Xv[k] = 0.0;
      else mat_mul(X, v[p], Xv, 6, 6, 1);
      for (int k = 0; k < 6; ++k) v[i][k] = Xv[k] + vJ[k];
      for (int k = 0; k < 3; ++k) {
        vel[((int64_t)i * 6 + k) * B + b] = v[i][3 + k];     /* linear first at the API */
        vel[((int64_t)i * 6 + 3 + k) * B + b] = v[i][k];
      }
    }
  }
  free(m);
  return 0;
}

/* Explicit Euler step of config 2 (BASELINE.json; readings 1 and 15), in place:
 *   qd += dt qdd ; q (+)= dt qd
 * revolute / prismatic: q += dt qd.  Free joint (q = [p, quat xyzw], qd = body-frame twist [v; omega]):
 *   p += dt R(quat) v ;  quat += dt/2 quat (x) (omega, 0) ;  quat /= |quat|      (quat normalised first)
 * The rotation is taken from joint_T, the same routine FK uses. */
int bard_oracle_euler_step(const bard_oracle_desc* d, int64_t B, double dt, double* q, double* qd, const double* qdd) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  for (int64_t b = 0; b < B; ++b) {
    for (int j = 0; j < m->nv; ++j) qd[(int64_t)j * B + b] += dt * qdd[(int64_t)j * B + b];
    for (int i = 0; i < m->nb; ++i) {
      const int t = m->jtype[i], qo = m->qoff[i], vo = m->voff[i];
      if (t == JT_REVOLUTE || t == JT_PRISMATIC) {
        q[(int64_t)qo * B + b] += dt * qd[(int64_t)vo * B + b];
      } else if (t == JT_FREE) {
        double qi[7], TJ[16], v[3], w[3];
        gather_q(m, i, q, B, b, qi);
        joint_T(m, i, qi, TJ);
        for (int k = 0; k < 3; ++k) { v[k] = qd[(int64_t)(vo + k) * B + b]; w[k] = qd[(int64_t)(vo + 3 + k) * B + b]; }
        for (int r = 0; r < 3; ++r)
          q[(int64_t)(qo + r) * B + b] = qi[r] + dt * (TJ[r * 4] * v[0] + TJ[r * 4 + 1] * v[1] + TJ[r * 4 + 2] * v[2]);
        double n = sqrt(qi[3] * qi[3] + qi[4] * qi[4] + qi[5] * qi[5] + qi[6] * qi[6]);
        double x = qi[3] / n, y = qi[4] / n, z = qi[5] / n, s = qi[6] / n;
        /* Hamilton product (x, y, z; s) (x) (w; 0) */
        double e[4] = {x + 0.5 * dt * (s * w[0] + y * w[2] - z * w[1]), y + 0.5 * dt * (s * w[1] + z * w[0] - x * w[2]),
                       z + 0.5 * dt * (s * w[2] + x * w[1] - y * w[0]), s + 0.5 * dt * (-x * w[0] - y * w[1] - z * w[2])};
        n = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2] + e[3] * e[3]);
        for (int k = 0; k < 4; ++k) q[(int64_t)(qo + 3 + k) * B + b] = e[k] / n;
      }
    }
  }
  free(m);
  return 0;
}

int bard_oracle_spatial_inertia(const bard_oracle_desc* d, int32_t body, double* I66) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (!rc) {
    if (body < 0 || body >= m->nb) rc = 5;
    else {
      /* permute internal [ang; lin] -> API [lin; ang] on both sides */
      int perm[6] = {3, 4, 5, 0, 1, 2};
      for (int r = 0; r < 6; ++r)
        for (int c = 0; c < 6; ++c) I66[r * 6 + c] = m->I[body][perm[r] * 6 + perm[c]];
    }
  }
  free(m);
  return rc;
}

/* ------------------------------------------------------------------ CRBA (item 8) */

int bard_oracle_crba(const bard_oracle_desc* d, int64_t B, const double* q, double* M) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  int nv = m->nv;
#pragma omp parallel for schedule(static) num_threads(bard_oracle_get_threads())
  for (int64_t b = 0; b < B; ++b) {
    double X[MAXB][36], Ic[MAXB][36];
    double Md[MAXB * MAXB];
    for (int k = 0; k < nv * nv; ++k) Md[k] = 0.0;
    for (int i = 0; i < m->nb; ++i) {
      double qi[7], Tpc[16];
      gather_q(m, i, q, B, b, qi);
      parent_child_T(m, i, qi, Tpc);
      plucker_X(Tpc, X[i]);
      memcpy(Ic[i], m->I[i], sizeof(Ic[i]));
    }
    /* composite inertias: Ic_p += X^T Ic X, deepest bodies first (reverse body order) */
    for (int i = m->nb - 1; i >= 0; --i) {
      int p = m->parent[i];
      if (p < 0) continue;
      double XT[36], tmp[36], XtIX[36];
      mat_transpose(X[i], XT, 6, 6);
      mat_mul(XT, Ic[i], tmp, 6, 6, 6);
      mat_mul(tmp, X[i], XtIX, 6, 6, 6);
      for (int k = 0; k < 36; ++k) Ic[p][k] += XtIX[k];
    }
    /* fill */
    for (int i = 0; i < m->nb; ++i) {
      int ni = m->nvi[i];
      if (ni == 0) continue;
      double F[36], ST[36], blk[36];
      mat_mul(Ic[i], m->S[i], F, 6, 6, ni);               /* F = Ic S_i : 6 x ni */
      mat_transpose(m->S[i], ST, 6, ni);                  /* ni x 6 */
      mat_mul(ST, F, blk, ni, 6, ni);                     /* S_i^T F */
      for (int r = 0; r < ni; ++r)
        for (int c = 0; c < ni; ++c) Md[(m->voff[i] + r) * nv + m->voff[i] + c] = blk[r * ni + c];
      int j = i;
      while (m->parent[j] >= 0) {
        double XT[36], F2[36];
        mat_transpose(X[j], XT, 6, 6);
        mat_mul(XT, F, F2, 6, 6, ni);                     /* F <- X_j^T F */
        memcpy(F, F2, sizeof(double) * 6 * ni);
        j = m->parent[j];
        int nj = m->nvi[j];
        if (nj == 0) continue;
        double FT[36], blk2[36];
        mat_transpose(F, FT, 6, ni);                      /* ni x 6 */
        mat_mul(FT, m->S[j], blk2, ni, 6, nj);            /* M[i,j] = F^T S_j : ni x nj */
        for (int r = 0; r < ni; ++r)
          for (int c = 0; c < nj; ++c) {
            Md[(m->voff[i] + r) * nv + m->voff[j] + c] = blk2[r * nj + c];
            Md[(m->voff[j] + c) * nv + m->voff[i] + r] = blk2[r * nj + c];
          }
      }
    }
    for (int r = 0; r < nv; ++r)
      for (int c = 0; c < nv; ++c) M[((int64_t)r * nv + c) * B + b] = Md[r * nv + c];
  }
  free(m);
  return 0;
}

/* ------------------------------------------------------------------ RNEA as a function of the inertial parameters
 * the paper's differentiability claim is exercised by identifying link masses through
 * RNEA (Section 4.3).  tau is LINEAR in the ten inertial parameters of every link,
 *   theta_i = (m, h = m c (3), Io = Ic + m [c]x [c]x^T : xx, xy, xz, yy, yz, zz about the BODY ORIGIN),
 * because the spatial inertia I_i = [[Io, [h]x], [[h]x^T, m 1]] is, and f_i = I_i a_i + v_i x* I_i v_i with v, a
 * independent of theta (RBDA Table 5.1; gravity enters through a_world, so tau(theta = 0) = 0).
 *
 * bard_oracle_rnea_params: the recursion of bard_oracle_rnea, line for line, with I_i built from params[nb][10]
 * instead of (mass, com, inertia).
 * bard_oracle_rnea_vjp_params: the vector-Jacobian product by its definition,
 *   dparams[k] = sum_b sum_j dtau[j][b] * d tau[j][b] / d theta_k ,  d tau / d theta_k = tau(theta = e_k)  (linearity),
 * i.e. nb * 10 evaluations of bard_oracle_rnea_params with unit parameter vectors.  No reverse sweep, no shortcut. */
static void inertia_from_params(const double* th /* 10 */, double I[36]) {
  const double m = th[0], h[3] = {th[1], th[2], th[3]};
  const double Io[9] = {th[4], th[5], th[6], th[5], th[7], th[8], th[6], th[8], th[9]};
  double hx[9], hxT[9];
  skew(h, hx);
  mat_transpose(hx, hxT, 3, 3);
  for (int r = 0; r < 3; ++r)
    for (int s = 0; s < 3; ++s) {
      I[r * 6 + s] = Io[r * 3 + s];
      I[r * 6 + 3 + s] = hx[r * 3 + s];
      I[(3 + r) * 6 + s] = hxT[r * 3 + s];
      I[(3 + r) * 6 + 3 + s] = (r == s) ? m : 0.0;
    }
}

static void rnea_with_model(const omodel* m, int64_t B, const double* q, const double* qd, const double* qdd, double* tau) {
#pragma omp parallel for schedule(static) num_threads(bard_oracle_get_threads())
  for (int64_t b = 0; b < B; ++b) {
    double X[MAXB][36], v[MAXB][6], a[MAXB][6], f[MAXB][6];
    for (int i = 0; i < m->nb; ++i) {
      double qi[7], Tpc[16], vJ[6], aJ[6], Xv[6], Xa[6], C[36], cv[6];
      gather_q(m, i, q, B, b, qi);
      parent_child_T(m, i, qi, Tpc);
      plucker_X(Tpc, X[i]);
      joint_velocity(m, i, qd, B, b, vJ);
      joint_velocity(m, i, qdd, B, b, aJ);
      int p = m->parent[i];
      if (p < 0) {
        for (int k = 0; k < 6; ++k) Xv[k] = 0.0;
        mat_mul(X[i], m->a_world, Xa, 6, 6, 1);
      } else {
        mat_mul(X[i], v[p], Xv, 6, 6, 1);
        mat_mul(X[i], a[p], Xa, 6, 6, 1);
      }
      for (int k = 0; k < 6; ++k) v[i][k] = Xv[k] + vJ[k];
      crm(v[i], C);
      mat_mul(C, vJ, cv, 6, 6, 1);
      for (int k = 0; k < 6; ++k) a[i][k] = Xa[k] + aJ[k] + cv[k];
      double Ia[6], Iv[6], Cf[36], vIv[6];
      mat_mul(m->I[i], a[i], Ia, 6, 6, 1);
      mat_mul(m->I[i], v[i], Iv, 6, 6, 1);
      crf(v[i], Cf);
      mat_mul(Cf, Iv, vIv, 6, 6, 1);
      for (int k = 0; k < 6; ++k) f[i][k] = Ia[k] + vIv[k];
    }
    for (int i = m->nb - 1; i >= 0; --i) {
      int n = m->nvi[i];
      for (int c = 0; c < n; ++c) {
        double s = 0.0;
        for (int r = 0; r < 6; ++r) s += m->S[i][r * n + c] * f[i][r];
        tau[(int64_t)(m->voff[i] + c) * B + b] = s;
      }
      int p = m->parent[i];
      if (p >= 0) {
        double XT[36], XTf[6];
        mat_transpose(X[i], XT, 6, 6);
        mat_mul(XT, f[i], XTf, 6, 6, 1);
        for (int k = 0; k < 6; ++k) f[p][k] += XTf[k];
      }
    }
  }
}

int bard_oracle_rnea_params(const bard_oracle_desc* d, int64_t B, const double* q, const double* qd, const double* qdd,
                            const double* params, double* tau) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  for (int i = 0; i < m->nb; ++i) inertia_from_params(params + 10 * i, m->I[i]);
  rnea_with_model(m, B, q, qd, qdd, tau);
  free(m);
  return 0;
}

/* the ten parameters of every link of the description: (m, m c, Ic + m [c]x [c]x^T) */
int bard_oracle_inertial_params(const bard_oracle_desc* d, double* params /* [nb*10] */) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  for (int i = 0; i < m->nb; ++i) {
    const double* I = m->I[i];
    double* th = params + 10 * i;
    th[0] = I[3 * 6 + 3];
    th[1] = I[2 * 6 + 4]; th[2] = I[0 * 6 + 5]; th[3] = I[1 * 6 + 3];   /* [h]x: (2,1) = hx, (0,2) = hy, (1,0) = hz */
    th[4] = I[0]; th[5] = I[1]; th[6] = I[2]; th[7] = I[6 + 1]; th[8] = I[6 + 2]; th[9] = I[12 + 2];
  }
  free(m);
  return 0;
}

int bard_oracle_rnea_vjp_params(const bard_oracle_desc* d, int64_t B, const double* q, const double* qd, const double* qdd,
                                const double* dtau, double* dparams) {
  omodel* m = (omodel*)malloc(sizeof(omodel));
  int rc = build_model(d, m);
  if (rc) { free(m); return rc; }
  const int nb = m->nb, nv = m->nv;
  double* tau = (double*)malloc(sizeof(double) * (size_t)(nv > 0 ? nv : 1) * (size_t)(B > 0 ? B : 1));
  double* theta = (double*)calloc((size_t)nb * 10, sizeof(double));
  for (int k = 0; k < nb * 10; ++k) {
    theta[k] = 1.0;                                           /* unit parameter vector e_k */
    for (int i = 0; i < nb; ++i) inertia_from_params(theta + 10 * i, m->I[i]);
    rnea_with_model(m, B, q, qd, qdd, tau);                   /* = d tau / d theta_k for every environment */
    double s = 0.0;
    for (int64_t x = 0; x < (int64_t)nv * B; ++x) s += dtau[x] * tau[x];
    dparams[k] = s;
    theta[k] = 0.0;
  }
  free(theta);
  free(tau);
  free(m);
  return 0;
}
