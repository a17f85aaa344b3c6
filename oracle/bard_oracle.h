/*
 * bard_oracle.h -- fp64 CPU oracle for batched rigid-body operators (TEST INFRASTRUCTURE).
 *
 * This is the plain, slow, "obviously correct" restatement of what the hot path computes:
 * forward kinematics, geometric Jacobians, RNEA inverse dynamics and the CRBA mass matrix
 * (operator list: Section 3), written from Featherstone's recursive definitions
 * that the paper implements (ref. [5] at PAPER.md:190).
 *
 * It is NOT part of the product.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no source, header, table or
 * helper with the CUDA path under paper_2605_31481_b200/ (that is why the model description
 * struct is re-declared here instead of including include/bard.h).
 *
 * Conventions (SURVEY.md section 8 "Notation"; readings listed in DESIGN.md):
 *   - bodies i = 0..nb-1, one joint per body, parent[i] in {-1, 0..i-1}; -1 = world.
 *   - T_pc,i = T_pre,i * T_J(q_i) * T_post,i maps child coordinates to parent coordinates
 *     (eq. (1): T_joint * R_axis(q) * T_link).
 *   - joint types: 0 revolute (nq=nv=1), 1 prismatic (1,1), 2 fixed (0,0), 3 free (nq=7,nv=6).
 *   - free joint: q = [p(3), quat x,y,z,w], quaternion normalised inside; qd = body-frame twist
 *     [v_lin(3); omega(3)]; qdd = its component-wise time derivative; tau = [force(3); moment(3)].
 *   - API spatial order is [linear; angular]; internally Featherstone's [angular; linear].
 *   - all batched arrays are structure-of-arrays, batch fastest: component c of env b is
 *     ptr[c*B + b].  q[nq][B], qd[nv][B], qdd[nv][B], pose[nb][12][B] (R row-major then p),
 *     J[nframes][6][nv][B] (rows 0-2 linear, 3-5 angular), tau[nv][B], M[nv][nv][B].
 *   - all pointers are HOST pointers, all floating point is double.
 *
 * Pins (what ties this oracle to something other than itself) live in tests/test_oracle_*.py:
 * pendulum / double-pendulum / free-body closed forms, finite-difference Jacobians, the
 * unit-acceleration mass matrix, energy and symmetry invariants, brute-force level tables.
 * No function here is "parity unpinned".
 */
#ifndef BARD_ORACLE_H
#define BARD_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t        nb;
  const int32_t* parent;       /* [nb]                                         */
  const int32_t* joint_type;   /* [nb]                                         */
  const double*  axis;         /* [nb*3] joint frame, normalised by the oracle */
  const double*  T_pre;        /* [nb*12] row-major [R|t] rows: r00 r01 r02 t0 ... */
  const double*  T_post;       /* [nb*12] or NULL = identity                   */
  const double*  mass;         /* [nb]                                         */
  const double*  com;          /* [nb*3] body frame                            */
  const double*  inertia;      /* [nb*6] xx,xy,xz,yy,yz,zz about COM, body axes */
  double         gravity[3];   /* world frame                                  */
  int32_t        nframes;      /* Jacobian frames                              */
  const int32_t* frame_body;   /* [nframes]                                    */
  const double*  frame_offset; /* [nframes*3] in body frame, or NULL = zeros   */
} bard_oracle_desc;

enum {
  BARD_ORACLE_TAB_LEVEL_PTR = 0, /* int32 [nlevels+1] */
  BARD_ORACLE_TAB_LEVEL_BODY = 1,/* int32 [nb]  bodies sorted by (level, index) */
  BARD_ORACLE_TAB_BODY_LEVEL = 2,/* int32 [nb]  */
  BARD_ORACLE_TAB_PARENT_SLOT = 3,/* int32 [nb] slot of parent of LEVEL_BODY[s], -1 = world */
  BARD_ORACLE_TAB_Q_OFF = 4,     /* int32 [nb+1] */
  BARD_ORACLE_TAB_V_OFF = 5,     /* int32 [nb+1] */
  BARD_ORACLE_TAB_DOF_BODY = 6,  /* int32 [nv]  */
  BARD_ORACLE_TAB_ANC_MASK = 7   /* uint64 [nb] bit j set <=> j == i or j is an ancestor of i */
};

/* returns 0 on success, non-zero on an invalid description */
int  bard_oracle_dims(const bard_oracle_desc* d, int32_t* nq, int32_t* nv, int32_t* nlevels);
/* writes the table as int64 values (uint64 bit pattern for ANC_MASK); returns element count or <0 */
int  bard_oracle_table(const bard_oracle_desc* d, int table_id, int64_t* out, int64_t cap);

/* Rodrigues constants of eq. (2)-(3): per body 36 doubles
 * R0(9) A(9) B(9) t0(3) a(3) b(3); prismatic/fixed/free use the analogous constants
 * (DESIGN.md "Rodrigues constants for non-revolute joints"). */
int  bard_oracle_rodrigues(const bard_oracle_desc* d, double* out /* [nb*36] */);
/* FK through eq. (4)-(5) with those constants instead of the 4x4 products: second formulation */
int  bard_oracle_fk_rodrigues(const bard_oracle_desc* d, int64_t B, const double* q, double* pose);

int  bard_oracle_fk      (const bard_oracle_desc* d, int64_t B, const double* q, double* pose);
int  bard_oracle_jacobian(const bard_oracle_desc* d, int64_t B, const double* q, double* J);
int  bard_oracle_rnea    (const bard_oracle_desc* d, int64_t B, const double* q, const double* qd,
                          const double* qdd, double* tau);
int  bard_oracle_crba    (const bard_oracle_desc* d, int64_t B, const double* q, double* M);

/* explicit Euler step of the config-2 rollout, in place: qd += dt qdd ; q (+)= dt qd (manifold step for a
 * free joint: p += dt R v, quat += dt/2 quat (x) (omega, 0), renormalised) */
int  bard_oracle_euler_step(const bard_oracle_desc* d, int64_t B, double dt, double* q, double* qd, const double* qdd);

/* spatial velocity of every body, body coordinates, API order [lin; ang]: vel[nb][6][B]
 * (used by the invariants: kinetic energy, frame velocity = J qd) */
int  bard_oracle_body_velocity(const bard_oracle_desc* d, int64_t B, const double* q,
                               const double* qd, double* vel);
/* spatial inertia of body i as a dense 6x6, API order [lin; ang], row-major (free-body pin) */
int  bard_oracle_spatial_inertia(const bard_oracle_desc* d, int32_t body, double* I66);

/* RNEA as a function of the inertial parameters (the paper's system-identification use,
 * PAPER.md:150-158).  params[nb][10] per link: m, h = m c (3), Io = Ic + m [c]x [c]x^T (xx,xy,xz,yy,yz,zz, about the
 * BODY ORIGIN); tau is linear in them.  rnea_params = bard_oracle_rnea with the spatial inertias built from params;
 * inertial_params = the ten parameters of the description's links; rnea_vjp_params = the VJP by its definition:
 * dparams[k] = sum over environments and DOFs of dtau * tau(params = e_k)  (nb*10 RNEA evaluations).
 * Pins (tests/test_rnea_vjp.py): agreement with bard_oracle_rnea at the description's parameters, linearity,
 * pendulum closed form, central finite differences through bard_oracle_rnea with perturbed mass / COM / inertia. */
int  bard_oracle_rnea_params(const bard_oracle_desc* d, int64_t B, const double* q, const double* qd, const double* qdd,
                             const double* params, double* tau);
int  bard_oracle_inertial_params(const bard_oracle_desc* d, double* params);
int  bard_oracle_rnea_vjp_params(const bard_oracle_desc* d, int64_t B, const double* q, const double* qd, const double* qdd,
                                 const double* dtau, double* dparams /* [nb*10] */);

void bard_oracle_set_threads(int n);   /* OpenMP threads over environments; n<=0 -> all cores */
int  bard_oracle_get_threads(void);

#ifdef __cplusplus
}
#endif
#endif
