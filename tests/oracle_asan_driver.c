/* Test helper (tests/test_oracle_pins.py::test_oracle_under_asan_ubsan): every entry point of the fp64 oracle on a small
 * tree with all four joint types, compiled together with oracle/bard_oracle.c under -fsanitize=address,undefined.
 * Prints one checksum; the sanitizers abort with a report on any out-of-bounds access or undefined behaviour. */
#include <stdio.h>
#include <stdlib.h>

#include "../oracle/bard_oracle.h"

int main(void) {
  enum { NB = 6, B = 5 };
  const int32_t parent[NB] = {-1, 0, 1, 1, 0, 4};
  const int32_t jt[NB] = {3, 0, 1, 2, 0, 0};
  double axis[NB * 3], Tpre[NB * 12], Tpost[NB * 12], mass[NB], com[NB * 3], inertia[NB * 6];
  for (int i = 0; i < NB; ++i) {
    axis[3 * i] = 0.3 + i; axis[3 * i + 1] = 1.0; axis[3 * i + 2] = -0.5;
    for (int k = 0; k < 12; ++k) Tpre[12 * i + k] = Tpost[12 * i + k] = (k == 0 || k == 5 || k == 10) ? 1.0 : 0.0;
    if (jt[i] != 3) { Tpre[12 * i + 3] = 0.1 * i; Tpre[12 * i + 7] = -0.05; Tpost[12 * i + 11] = 0.02 * i; }
    mass[i] = 1.0 + 0.1 * i;
    com[3 * i] = 0.01 * i; com[3 * i + 1] = -0.02; com[3 * i + 2] = 0.03;
    inertia[6 * i] = 0.02; inertia[6 * i + 1] = 0.001; inertia[6 * i + 2] = 0.0; inertia[6 * i + 3] = 0.03; inertia[6 * i + 4] = 0.0; inertia[6 * i + 5] = 0.015;
  }
  Tpost[0] = 1.0;
  const int32_t fbody[2] = {3, 5};
  const double foff[6] = {0.1, 0, 0, 0, 0.05, -0.1};
  bard_oracle_desc d = {NB, parent, jt, axis, Tpre, Tpost, mass, com, inertia, {0, 0, -9.81}, 2, fbody, foff};
  int32_t nq, nv, nl;
  if (bard_oracle_dims(&d, &nq, &nv, &nl)) return 2;
  double* q = calloc((size_t)nq * B, sizeof(double));
  double* qd = calloc((size_t)nv * B, sizeof(double));
  double* qdd = calloc((size_t)nv * B, sizeof(double));
  double* dtau = calloc((size_t)nv * B, sizeof(double));
  for (int i = 0; i < nq * B; ++i) q[i] = 0.1 * (i % 7) - 0.3;
  for (int b = 0; b < B; ++b) q[6 * B + b] = 1.0;        /* quaternion w */
  for (int i = 0; i < nv * B; ++i) { qd[i] = 0.05 * (i % 11) - 0.2; qdd[i] = 0.03 * (i % 5); dtau[i] = 1.0 - 0.1 * (i % 3); }
  double* pose = calloc((size_t)NB * 12 * B, sizeof(double));
  double* J = calloc((size_t)2 * 6 * nv * B, sizeof(double));
  double* tau = calloc((size_t)nv * B, sizeof(double));
  double* M = calloc((size_t)nv * nv * B, sizeof(double));
  double* vel = calloc((size_t)NB * 6 * B, sizeof(double));
  double rod[NB * 36], I66[36], th[NB * 10], g[NB * 10];
  int64_t tab[NB + 8];
  int rc = 0;
  bard_oracle_set_threads(2);
  for (int t = 0; t < 8; ++t) rc |= bard_oracle_table(&d, t, tab, NB + 8) < 0;
  rc |= bard_oracle_rodrigues(&d, rod);
  rc |= bard_oracle_fk(&d, B, q, pose);
  rc |= bard_oracle_fk_rodrigues(&d, B, q, pose);
  rc |= bard_oracle_jacobian(&d, B, q, J);
  rc |= bard_oracle_rnea(&d, B, q, qd, qdd, tau);
  rc |= bard_oracle_crba(&d, B, q, M);
  rc |= bard_oracle_body_velocity(&d, B, q, qd, vel);
  rc |= bard_oracle_spatial_inertia(&d, 2, I66);
  rc |= bard_oracle_inertial_params(&d, th);
  rc |= bard_oracle_rnea_params(&d, B, q, qd, qdd, th, tau);
  rc |= bard_oracle_rnea_vjp_params(&d, B, q, qd, qdd, dtau, g);
  rc |= bard_oracle_euler_step(&d, B, 0.005, q, qd, qdd);
  double s = 0;
  for (int i = 0; i < nv * B; ++i) s += tau[i];
  for (int i = 0; i < NB * 10; ++i) s += g[i];
  printf("checksum %.6f rc %d\n", s, rc);
  free(q); free(qd); free(qdd); free(dtau); free(pose); free(J); free(tau); free(M); free(vel);
  return rc;
}
