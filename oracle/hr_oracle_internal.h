/* hr_oracle_internal.h -- layout of the oracle's grid object (ORACLE ONLY; see hr_oracle.h). */
#ifndef HR_ORACLE_INTERNAL_H
#define HR_ORACLE_INTERNAL_H

#include "hr_oracle.h"

#define ORC_MAX_NG 6

struct orc_grid {
  orc_params p;
  double* punctures;         /* owned copy, n_punctures x 10                               */
  int32_t ng;                /* C7                                                         */
  int32_t T[3];              /* points per axis incl. ghosts                               */
  int64_t ntot;              /* T0*T1*T2; flat index i0 + T0*(i1 + T1*i2)  (C8)            */
  double dx[3];              /* uniform spacings of x0 in [0,1], x1 in [0,pi], x2 in [-pi,pi] */
  double *x0, *x1, *x2;      /* cell-centred coordinates incl. ghosts (C8)                 */
  double c1[ORC_MAX_NG + 1]; /* first-derivative weights, unit spacing (C11)               */
  double d2[ORC_MAX_NG + 1]; /* second-derivative weights, unit spacing (C11)              */
  /* (i0,i1) planes, index i0 + T0*i1 (nothing in C4/C9 depends on x2) */
  double *g00, *g11, *g22, *g0, *g1; /* Laplacian factors (C4)                             */
  double *c;                 /* wave speed (C9)                                            */
  double *w;                 /* |h0 h1 h2| (C16)                                           */
  double *ds;                /* min_a |h_a| dx^a (C9)                                      */
  /* radiation-BC factors on the same planes (C13): d_r f = r0*d_0 f + r1*d_1 f */
  double *rad0, *rad1, *invr;
  /* C25 (SinhCartesian): the x2-dependent factors, T2 each (see orc_get_axis2), and per axis the Cartesian
   * coordinate X_a(x^a_i) and 1/h_a at every index, for the radiation condition on the six faces   */
  double *z22, *z2, *zds, *zh;
  double *X[3], *ih[3];
  double dsmin, dt;          /* C9                                                         */
  int64_t n_inner, n_outer;
  int32_t *inner_dst, *inner_src, *outer_idx; /* C13, C14; ascending dst / idx             */
  double bc_max_frac_err;
  double *psi, *S;           /* psi_BL (C1) and (1/8) A~_ij A~^ij (C2), ntot each, fp64    */
};

/* C9: wave speed at (plane position q, i2): c_min ds/ds_min with ds = min_a h_a dx^a. */
static inline double orc_c_at(const struct orc_grid* g, size_t q, int i2) {
  if (g->p.coord != ORC_SINHCARTESIAN) return g->c[q];
  const double ds = g->ds[q] < g->zds[i2] ? g->ds[q] : g->zds[i2];
  return g->p.c_min * ds / g->dsmin;
}

static inline int64_t orc_idx(const struct orc_grid* g, int i0, int i1, int i2) {
  return (int64_t)i0 + (int64_t)g->T[0] * ((int64_t)i1 + (int64_t)g->T[1] * (int64_t)i2);
}

#endif
