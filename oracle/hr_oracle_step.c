/*
 * hr_oracle_step.c -- the evolution half of the CPU ORACLE (test infrastructure; see
 * hr_oracle.h).  Compiled twice: -DORC_REAL=double -DORC_SUF=_f64 and
 * -DORC_REAL=float -DORC_SUF=_f32 (reading C19: state, k, psi_BL, S and every factor are
 * held and combined in ORC_REAL; only the residual sums are fp64).
 *
 * Literal Alg. 1 l.12-16: RHS on interior -> BC on k (outer, then inner)
 * -> RK update over all points, for the system of Eq. 5.  Plain triple
 * loops, i0 innermost; no blocking, no fusion.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "hr_oracle_internal.h"

#ifndef ORC_REAL
#error "compile with -DORC_REAL=double|float -DORC_SUF=_f64|_f32"
#endif

#define ORC_CAT_(a, b) a##b
#define ORC_CAT(a, b) ORC_CAT_(a, b)
#define FN(name) ORC_CAT(name, ORC_SUF)

typedef ORC_REAL real;

static real FN(orc_pow_m7)(real x) {
  /* (psi_BL + u)^-7 of Eq. 4/5, by the library power function in the working precision */
  return (sizeof(real) == sizeof(double)) ? (real)pow((double)x, -7.0) : (real)powf((float)x, -7.0f);
}

/* C11/C12: the five centred derivatives of u at one point and the expanded Laplacian of C4. */
static real FN(orc_lap_point)(const orc_grid* g, const real* u, int i0, int i1, int i2) {
  const int n = g->ng;
  const int64_t s0 = 1, s1 = g->T[0], s2 = (int64_t)g->T[0] * g->T[1];
  const int64_t c = orc_idx(g, i0, i1, i2);
  const real idx0 = (real)(1.0 / g->dx[0]), idx1 = (real)(1.0 / g->dx[1]);
  const real idxx0 = (real)(1.0 / (g->dx[0] * g->dx[0]));
  const real idxx1 = (real)(1.0 / (g->dx[1] * g->dx[1]));
  const real idxx2 = (real)(1.0 / (g->dx[2] * g->dx[2]));
  real d0 = 0, d1 = 0;
  real d00 = (real)g->d2[0] * u[c], d11 = (real)g->d2[0] * u[c], d22 = (real)g->d2[0] * u[c];
  for (int k = 1; k <= n; ++k) {
    d0 += (real)g->c1[k] * (u[c + k * s0] - u[c - k * s0]);
    d1 += (real)g->c1[k] * (u[c + k * s1] - u[c - k * s1]);
    d00 += (real)g->d2[k] * (u[c + k * s0] + u[c - k * s0]);
    d11 += (real)g->d2[k] * (u[c + k * s1] + u[c - k * s1]);
    d22 += (real)g->d2[k] * (u[c + k * s2] + u[c - k * s2]);
  }
  d0 *= idx0;
  d1 *= idx1;
  d00 *= idxx0;
  d11 *= idxx1;
  d22 *= idxx2;
  const size_t q = (size_t)i0 + (size_t)g->T[0] * (size_t)i1;
  if (g->p.coord == ORC_SINHCARTESIAN) {
    /* C25: the u_22 factor depends on x2 and there is a u_2 term (sum_a [u_aa/h_a^2 - X_a''/X_a'^3 u_a]) */
    real d2 = 0;
    for (int k = 1; k <= n; ++k) d2 += (real)g->c1[k] * (u[c + k * s2] - u[c - k * s2]);
    d2 *= (real)(1.0 / g->dx[2]);
    return (real)g->g00[q] * d00 + (real)g->g11[q] * d11 + (real)g->z22[i2] * d22 +
           (real)g->g0[q] * d0 + (real)g->g1[q] * d1 + (real)g->z2[i2] * d2;
  }
  return (real)g->g00[q] * d00 + (real)g->g11[q] * d11 + (real)g->g22[q] * d22 +
         (real)g->g0[q] * d0 + (real)g->g1[q] * d1;
}

void FN(orc_laplacian)(const orc_grid* g, const real* u, real* lap) {
  const int ng = g->ng;
  memset(lap, 0, sizeof(real) * (size_t)g->ntot);
#pragma omp parallel for schedule(static)
  for (int i2 = ng; i2 < g->p.n[2] + ng; ++i2)
    for (int i1 = ng; i1 < g->p.n[1] + ng; ++i1)
      for (int i0 = ng; i0 < g->p.n[0] + ng; ++i0)
        lap[orc_idx(g, i0, i1, i2)] = FN(orc_lap_point)(g, u, i0, i1, i2);
}

/* a1, Eq. 5 at interior points:
 *   k_u = v - eta u ;   k_v = c^2 [ lap u + S (psi_BL + u)^-7 ],  S = (1/8) A~_ij A~^ij      */
void FN(orc_rhs_interior)(const orc_grid* g, const real* u, const real* v, real* ku, real* kv) {
  const int ng = g->ng;
  const real eta = (real)g->p.eta;
#pragma omp parallel for schedule(static)
  for (int i2 = ng; i2 < g->p.n[2] + ng; ++i2)
    for (int i1 = ng; i1 < g->p.n[1] + ng; ++i1)
      for (int i0 = ng; i0 < g->p.n[0] + ng; ++i0) {
        const int64_t c = orc_idx(g, i0, i1, i2);
        const real cw = (real)orc_c_at(g, (size_t)i0 + (size_t)g->T[0] * (size_t)i1, i2);
        const real lap = FN(orc_lap_point)(g, u, i0, i1, i2);
        const real src = (real)g->S[c] * FN(orc_pow_m7)((real)g->psi[c] + u[c]);
        ku[c] = v[c] - eta * u[c];
        kv[c] = cw * cw * (lap + src);
      }
}

/* a2, C13: outgoing-radiation (Sommerfeld) condition at the outer points, applied to k:
 *   k_f = -c [ d_r f + (f - f_inf)/r ],  f_inf = 0,  f in {u, v};
 *   d_r f = rad0 d_0 f + rad1 d_1 f,  each derivative 2nd order: one-sided, pointing into the grid,
 *   along an axis in which the point lies beyond the interior (backward on the high side, forward
 *   on the low side), centred otherwise.  SinhSpherical / SinhSymTP outer points lie beyond x0 only
 *   (backward d_0, centred d_1); SinhCylindrical ones (C24) also beyond either end of x1.        */
/* C25 (SinhCartesian): every ghost point is an outer point; r = |X|, d_r f = sum_a (X_a / r) (1/h_a) d_a f
 * over the three axes, the same one-sided / centred rule per axis; c from orc_c_at.                  */
static void FN(orc_bc_outer_cart)(const orc_grid* g, const real* u, const real* v, real* ku, real* kv) {
  const int64_t st[3] = {1, g->T[0], (int64_t)g->T[0] * g->T[1]};
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < g->n_outer; ++m) {
    const int64_t c = g->outer_idx[m];
    int i[3];
    i[0] = (int)(c % g->T[0]);
    i[1] = (int)((c / g->T[0]) % g->T[1]);
    i[2] = (int)(c / ((int64_t)g->T[0] * g->T[1]));
    const double X0 = g->X[0][i[0]], X1 = g->X[1][i[1]], X2 = g->X[2][i[2]];
    const double dist = sqrt(X0 * X0 + X1 * X1 + X2 * X2);
    const real cw = (real)orc_c_at(g, (size_t)i[0] + (size_t)g->T[0] * (size_t)i[1], i[2]);
    const real ir = (real)(1.0 / dist);
    real rad[3], hh[3];
    for (int a = 0; a < 3; ++a) {
      rad[a] = (real)(g->X[a][i[a]] * g->ih[a][i[a]] / dist);
      hh[a] = (real)(1.0 / (2.0 * g->dx[a]));
    }
    const real* f[2] = {u, v};
    real* k[2] = {ku, kv};
    for (int b = 0; b < 2; ++b) {
      real acc = 0;
      for (int a = 0; a < 3; ++a) {
        const int64_t s = st[a];
        real d;
        if (i[a] >= g->p.n[a] + g->ng)
          d = ((real)3 * f[b][c] - (real)4 * f[b][c - s] + f[b][c - 2 * s]) * hh[a];
        else if (i[a] < g->ng)
          d = ((real)4 * f[b][c + s] - (real)3 * f[b][c] - f[b][c + 2 * s]) * hh[a];
        else
          d = (f[b][c + s] - f[b][c - s]) * hh[a];
        acc += rad[a] * d;
      }
      k[b][c] = -cw * (acc + f[b][c] * ir);
    }
  }
}

void FN(orc_bc_outer)(const orc_grid* g, const real* u, const real* v, real* ku, real* kv) {
  if (g->p.coord == ORC_SINHCARTESIAN) {
    FN(orc_bc_outer_cart)(g, u, v, ku, kv);
    return;
  }
  const int64_t s1 = g->T[0];
  const real h0 = (real)(1.0 / (2.0 * g->dx[0])), h1 = (real)(1.0 / (2.0 * g->dx[1]));
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < g->n_outer; ++m) {
    const int64_t c = g->outer_idx[m];
    const size_t q = (size_t)(c % ((int64_t)g->T[0] * g->T[1]));
    const int i0 = (int)(q % (size_t)g->T[0]), i1 = (int)(q / (size_t)g->T[0]);
    const int hi0 = i0 >= g->p.n[0] + g->ng;
    const int hi1 = i1 >= g->p.n[1] + g->ng, lo1 = i1 < g->ng;
    const real cw = (real)g->c[q], r0 = (real)g->rad0[q], r1 = (real)g->rad1[q],
               ir = (real)g->invr[q];
    const real* f[2] = {u, v};
    real* k[2] = {ku, kv};
    for (int a = 0; a < 2; ++a) {
      real d0, d1;
      if (hi0)
        d0 = ((real)3 * f[a][c] - (real)4 * f[a][c - 1] + f[a][c - 2]) * h0;
      else
        d0 = (f[a][c + 1] - f[a][c - 1]) * h0;
      if (hi1)
        d1 = ((real)3 * f[a][c] - (real)4 * f[a][c - s1] + f[a][c - 2 * s1]) * h1;
      else if (lo1)
        d1 = ((real)4 * f[a][c + s1] - (real)3 * f[a][c] - f[a][c + 2 * s1]) * h1;
      else
        d1 = (f[a][c + s1] - f[a][c - s1]) * h1;
      k[a][c] = -cw * (r0 * d0 + r1 * d1 + f[a][c] * ir);
    }
  }
}

/* a3, C14: inner (parity) boundary condition, parity +1 for the scalars u, v. */
void FN(orc_bc_inner)(const orc_grid* g, real* f) {
  for (int64_t m = 0; m < g->n_inner; ++m) f[g->inner_dst[m]] = f[g->inner_src[m]];
}

/* Alg. 1 l.13-14: RHS, then BCs on the freshly computed k (outer first: some inner sources
 * are outer points). */
void FN(orc_rhs)(const orc_grid* g, const real* u, const real* v, real* ku, real* kv) {
  FN(orc_rhs_interior)(g, u, v, ku, kv);
  FN(orc_bc_outer)(g, u, v, ku, kv);
  FN(orc_bc_inner)(g, ku);
  FN(orc_bc_inner)(g, kv);
}

/* a4, C15: classic RK4, update over ALL ntot points:
 *   k1 = F(Y); k2 = F(Y + dt/2 k1); k3 = F(Y + dt/2 k2); k4 = F(Y + dt k3);
 *   Y <- Y + dt/6 (k1 + 2 k2 + 2 k3 + k4)                                                    */
void FN(orc_step)(const orc_grid* g, real* u, real* v, int64_t nsteps) {
  const size_t n = (size_t)g->ntot;
  real* buf = (real*)calloc(10 * n, sizeof(real));
  real *k1u = buf, *k1v = buf + n, *k2u = buf + 2 * n, *k2v = buf + 3 * n, *k3u = buf + 4 * n,
       *k3v = buf + 5 * n, *k4u = buf + 6 * n, *k4v = buf + 7 * n, *su = buf + 8 * n,
       *sv = buf + 9 * n;
  const real dt = (real)g->dt, half = (real)0.5, two = (real)2, six = (real)6;
  for (int64_t it = 0; it < nsteps; ++it) {
    FN(orc_rhs)(g, u, v, k1u, k1v);
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
      su[i] = u[i] + half * dt * k1u[i];
      sv[i] = v[i] + half * dt * k1v[i];
    }
    FN(orc_rhs)(g, su, sv, k2u, k2v);
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
      su[i] = u[i] + half * dt * k2u[i];
      sv[i] = v[i] + half * dt * k2v[i];
    }
    FN(orc_rhs)(g, su, sv, k3u, k3v);
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
      su[i] = u[i] + dt * k3u[i];
      sv[i] = v[i] + dt * k3v[i];
    }
    FN(orc_rhs)(g, su, sv, k4u, k4v);
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < n; ++i) {
      u[i] = u[i] + dt / six * (k1u[i] + two * k2u[i] + two * k3u[i] + k4u[i]);
      v[i] = v[i] + dt / six * (k1v[i] + two * k2v[i] + two * k3v[i] + k4v[i]);
    }
  }
  free(buf);
}

/* a5, C16: H = lap u + S (psi_BL + u)^-7 at interior points;
 *   mode 0: sqrt( sum w H^2 / sum w ), w = |h0 h1 h2| ;  mode 1: sqrt( sum H^2 / N_int ).
 * Sums in fp64, one partial per i2-plane added in ascending i2 (independent of threads).  */
void FN(orc_residual)(const orc_grid* g, const real* u, int32_t mode, double* out, real* H) {
  const int ng = g->ng;
  const int n2 = g->p.n[2];
  double* num = (double*)calloc((size_t)n2, sizeof(double));
  double* den = (double*)calloc((size_t)n2, sizeof(double));
  if (H) memset(H, 0, sizeof(real) * (size_t)g->ntot);
#pragma omp parallel for schedule(static)
  for (int i2 = ng; i2 < n2 + ng; ++i2) {
    double a = 0.0, b = 0.0;
    for (int i1 = ng; i1 < g->p.n[1] + ng; ++i1)
      for (int i0 = ng; i0 < g->p.n[0] + ng; ++i0) {
        const int64_t c = orc_idx(g, i0, i1, i2);
        const real lap = FN(orc_lap_point)(g, u, i0, i1, i2);
        const real h = lap + (real)g->S[c] * FN(orc_pow_m7)((real)g->psi[c] + u[c]);
        if (H) H[c] = h;
        /* C16 weight |h0 h1 h2| (C25: the plane holds |h0 h1|, zh the x2 factor; zh = 1 otherwise) */
        const double w = (mode == 0) ? g->w[(size_t)i0 + (size_t)g->T[0] * (size_t)i1] * g->zh[i2] : 1.0;
        a += w * (double)h * (double)h;
        b += w;
      }
    num[i2 - ng] = a;
    den[i2 - ng] = b;
  }
  double A = 0.0, B = 0.0;
  for (int j = 0; j < n2; ++j) {
    A += num[j];
    B += den[j];
  }
  out[0] = sqrt(A / B);
  out[1] = A;
  out[2] = B;
  free(num);
  free(den);
}
