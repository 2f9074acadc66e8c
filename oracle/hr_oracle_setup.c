/*
 * hr_oracle_setup.c -- fp64 set-up of the CPU ORACLE (test infrastructure; see hr_oracle.h).
 *
 * Follows PAPER.md:198-203 (Alg. 1 l.2-7): coordinate arrays, reference-metric
 * factors, boundary-condition containers, constant source terms; formulas are the
 * readings C1-C14 of SURVEY.md Sec. 8(c) (listed in DESIGN.md).  Plain loops, libm only.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "hr_oracle_internal.h"

#ifdef _OPENMP
#include <omp.h>
#endif

static const double ORC_PI = 3.14159265358979323846264338327950288;

int32_t orc_num_threads(void) {
#ifdef _OPENMP
  return (int32_t)omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * C11 ("finite-difference stencils", orders 2-12): centred weights on a
 * uniform grid with unit spacing, radius n = order/2:
 *   first derivative   c_k = (-1)^(k+1) (n!)^2 / ( k   (n-k)! (n+k)! ),  c_{-k} = -c_k, c_0 = 0
 *   second derivative  d_k = 2 (-1)^(k+1) (n!)^2 / ( k^2 (n-k)! (n+k)! ), d_{-k} = d_k,
 *                      d_0 = -2 sum_k d_k
 * ---------------------------------------------------------------------------------------- */
static double orc_factorial(int m) {
  double f = 1.0;
  for (int i = 2; i <= m; ++i) f *= (double)i;
  return f;
}

void orc_fd_weights(int32_t order, double* c1, double* d2) {
  const int n = order / 2;
  const double nf2 = orc_factorial(n) * orc_factorial(n);
  double sum = 0.0;
  c1[0] = 0.0;
  for (int k = 1; k <= n; ++k) {
    const double sign = (k % 2 == 1) ? 1.0 : -1.0;
    const double den = orc_factorial(n - k) * orc_factorial(n + k);
    c1[k] = sign * nf2 / ((double)k * den);
    d2[k] = 2.0 * sign * nf2 / ((double)k * (double)k * den);
    sum += d2[k];
  }
  d2[0] = -2.0 * sum;
}

/* ------------------------------------------------------------------------------------------
 * C4: radial map shared by both systems, rho(x0) = AMP sinh(x0/W) / sinh(1/W),
 *     rho' = AMP cosh(x0/W) / (W sinh(1/W)),  rho'' = rho / W^2.
 * ---------------------------------------------------------------------------------------- */
static void orc_rho(double amp, double W, double x0, double* r, double* rp, double* rpp) {
  const double s = sinh(1.0 / W);
  *r = amp * sinh(x0 / W) / s;
  *rp = amp * cosh(x0 / W) / (W * s);
  *rpp = *r / (W * W);
}

/* C4: (x0, x1 = theta, x2 = phi) -> Cartesian, grid-centred.
 *   SinhSpherical: (r sin th cos ph, r sin th sin ph, r cos th),            r = rho(x0)
 *   SinhSymTP:     (A sin th cos ph, A sin th sin ph, sqrt(A^2+b^2) cos th), A = rho(x0)
 * C24 ("cylindrical-like"): x0 in [0,1], x1 in [-1,1], x2 = phi in [-pi,pi);
 *   SinhCylindrical: (R cos ph, R sin ph, Z),  R = rho(x0), Z = rho(x1)  (the same sinh map, same
 *   amplitude and width, along the axis; the periodic coordinate is x2 as in the other systems)    */
void orc_map_to_cart(int32_t coord, double amp, double sinhw, double bscale, double x0,
                     double x1, double x2, double* xyz) {
  double r, rp, rpp;
  orc_rho(amp, sinhw, x0, &r, &rp, &rpp);
  if (coord == ORC_SINHCYLINDRICAL) {
    double z, zp, zpp;
    orc_rho(amp, sinhw, x1, &z, &zp, &zpp);
    xyz[0] = r * cos(x2);
    xyz[1] = r * sin(x2);
    xyz[2] = z;
    return;
  }
  if (coord == ORC_SINHCARTESIAN) { /* C25: x^a in [-1,1], X_a = rho(x^a), the same sinh map on every axis */
    double t, tp, tpp;
    xyz[0] = r;
    orc_rho(amp, sinhw, x1, &t, &tp, &tpp);
    xyz[1] = t;
    orc_rho(amp, sinhw, x2, &t, &tp, &tpp);
    xyz[2] = t;
    return;
  }
  const double st = sin(x1), ct = cos(x1), sp = sin(x2), cp = cos(x2);
  xyz[0] = r * st * cp;
  xyz[1] = r * st * sp;
  if (coord == ORC_SINHSPHERICAL)
    xyz[2] = r * ct;
  else
    xyz[2] = sqrt(r * r + bscale * bscale) * ct;
}

/* C14 (inverse map used to build the inner-boundary container):
 * Cartesian -> the representative with x0 >= 0, 0 <= theta <= pi, -pi <= phi < pi. */
void orc_map_from_cart(int32_t coord, double amp, double sinhw, double bscale,
                       const double* xyz, double* x012) {
  const double x = xyz[0], y = xyz[1], z = xyz[2];
  const double rc2 = x * x + y * y; /* cylindrical radius squared */
  const double rc = sqrt(rc2);
  double rad, th;
  if (coord == ORC_SINHCARTESIAN) { /* C25: axis by axis */
    for (int a = 0; a < 3; ++a) x012[a] = sinhw * asinh(xyz[a] * sinh(1.0 / sinhw) / amp);
    return;
  }
  if (coord == ORC_SINHCYLINDRICAL) { /* C24: x0 from the cylindrical radius, x1 from z, same sinh map */
    double ph = atan2(y, x);
    if (ph >= ORC_PI) ph -= 2.0 * ORC_PI;
    x012[0] = sinhw * asinh(rc * sinh(1.0 / sinhw) / amp);
    x012[1] = sinhw * asinh(z * sinh(1.0 / sinhw) / amp);
    x012[2] = ph;
    return;
  }
  if (coord == ORC_SINHSPHERICAL) {
    rad = sqrt(rc2 + z * z);
    th = atan2(rc, z);
  } else {
    /* A^2 is the non-negative root of  A^4 - (r^2 - b^2) A^2 - b^2 rc^2 = 0  */
    const double b2 = bscale * bscale;
    const double q = rc2 + z * z - b2;
    const double D = sqrt(q * q + 4.0 * b2 * rc2);
    const double A2 = (q >= 0.0) ? 0.5 * (q + D) : 2.0 * b2 * rc2 / (D - q);
    rad = sqrt(A2);
    th = atan2(rc / rad, z / sqrt(A2 + b2));
  }
  double ph = atan2(y, x);
  if (ph >= ORC_PI) ph -= 2.0 * ORC_PI;
  x012[0] = sinhw * asinh(rad * sinh(1.0 / sinhw) / amp);
  x012[1] = th;
  x012[2] = ph;
}

/* C4: scale factors h_a of the diagonal flat reference metric and the factors of the
 * expanded Laplacian
 *     lap u = g00 u_00 + g11 u_11 + g22 u_22 + g0 u_0 + g1 u_1      (no u_2, no mixed terms)
 * SinhSpherical: h = (r', r, r sin th);
 *     g00 = 1/r'^2, g11 = 1/r^2, g22 = 1/(r^2 sin^2 th),
 *     g0 = 2/(r r') - r''/r'^3, g1 = cos th / (r^2 sin th)
 * SinhSymTP: Sigma = A^2 + b^2 sin^2 th, AB = A^2 + b^2;
 *     h = (A' sqrt(Sigma/AB), sqrt(Sigma), A sin th);
 *     g00 = AB/(A'^2 Sigma), g0 = [(2A^2+b^2)/(A A') - AB A''/A'^3]/Sigma,
 *     g11 = 1/Sigma, g1 = cot th / Sigma, g22 = 1/(A^2 sin^2 th)                           */
void orc_metric_at(int32_t coord, double amp, double sinhw, double bscale, double x0, double x1,
                   double* h, double* gfac) {
  double r, rp, rpp;
  orc_rho(amp, sinhw, x0, &r, &rp, &rpp);
  if (coord == ORC_SINHCARTESIAN) {
    /* C25: h_a = X_a'(x^a);  lap u = sum_a [ u_aa / X_a'^2 - X_a''/X_a'^3 u_a ].  The x2 parts (h[2],
     * gfac[2] and the u_2 factor) are functions of x2 alone: orc_metric_axis2.                    */
    double t, tp, tpp;
    orc_rho(amp, sinhw, x1, &t, &tp, &tpp);
    h[0] = rp;
    h[1] = tp;
    h[2] = 1.0;
    gfac[0] = 1.0 / (rp * rp);
    gfac[1] = 1.0 / (tp * tp);
    gfac[2] = 1.0;
    gfac[3] = -rpp / (rp * rp * rp);
    gfac[4] = -tpp / (tp * tp * tp);
    return;
  }
  if (coord == ORC_SINHCYLINDRICAL) {
    /* C24: h = (R', Z', R);  lap u = u_00/R'^2 + u_11/Z'^2 + u_22/R^2
     *                                + [1/(R R') - R''/R'^3] u_0 - [Z''/Z'^3] u_1               */
    double z, zp, zpp;
    orc_rho(amp, sinhw, x1, &z, &zp, &zpp);
    h[0] = rp;
    h[1] = zp;
    h[2] = r;
    gfac[0] = 1.0 / (rp * rp);
    gfac[1] = 1.0 / (zp * zp);
    gfac[2] = 1.0 / (r * r);
    gfac[3] = 1.0 / (r * rp) - rpp / (rp * rp * rp);
    gfac[4] = -zpp / (zp * zp * zp);
    return;
  }
  const double st = sin(x1), ct = cos(x1);
  if (coord == ORC_SINHSPHERICAL) {
    h[0] = rp;
    h[1] = r;
    h[2] = r * st;
    gfac[0] = 1.0 / (rp * rp);
    gfac[1] = 1.0 / (r * r);
    gfac[2] = 1.0 / (r * r * st * st);
    gfac[3] = 2.0 / (r * rp) - rpp / (rp * rp * rp);
    gfac[4] = ct / (r * r * st);
  } else {
    const double b2 = bscale * bscale;
    const double AB = r * r + b2;
    const double Sg = r * r + b2 * st * st;
    h[0] = rp * sqrt(Sg / AB);
    h[1] = sqrt(Sg);
    h[2] = r * st;
    gfac[0] = AB / (rp * rp * Sg);
    gfac[1] = 1.0 / Sg;
    gfac[2] = 1.0 / (r * r * st * st);
    gfac[3] = ((2.0 * r * r + b2) / (r * rp) - AB * rpp / (rp * rp * rp)) / Sg;
    gfac[4] = (ct / st) / Sg;
  }
}

/* C25: the x2-dependent part of the SinhCartesian metric: h2 = X', u_22 factor 1/X'^2, u_2 factor -X''/X'^3. */
static void orc_metric_axis2(int32_t coord, double amp, double sinhw, double x2, double* h2, double* g22,
                             double* g2) {
  if (coord != ORC_SINHCARTESIAN) {
    *h2 = 1.0;
    *g22 = 1.0;
    *g2 = 0.0;
    return;
  }
  double t, tp, tpp;
  orc_rho(amp, sinhw, x2, &t, &tp, &tpp);
  *h2 = tp;
  *g22 = 1.0 / (tp * tp);
  *g2 = -tpp / (tp * tp * tp);
}

/* C13: radial derivative from coordinate derivatives, d_r f = rad0 d_0 f + rad1 d_1 f,
 * and 1/r with r = distance from the grid centre.
 *   SinhSpherical: rad0 = 1/r', rad1 = 0.
 *   SinhSymTP: r^2 = A^2 + b^2 cos^2 th;
 *       d_r f = [ A (A^2+b^2)/A' d_0 f - b^2 sin th cos th d_1 f ] / (r Sigma).             */
static void orc_radial_at(int32_t coord, double amp, double sinhw, double bscale, double x0,
                          double x1, double* rad0, double* rad1, double* invr) {
  double r, rp, rpp;
  orc_rho(amp, sinhw, x0, &r, &rp, &rpp);
  if (coord == ORC_SINHCYLINDRICAL) { /* C24: r^2 = R^2 + Z^2, d_r = (R/r) d_R + (Z/r) d_Z */
    double z, zp, zpp;
    orc_rho(amp, sinhw, x1, &z, &zp, &zpp);
    const double dist = sqrt(r * r + z * z);
    *rad0 = r / (dist * rp);
    *rad1 = z / (dist * zp);
    *invr = 1.0 / dist;
    return;
  }
  if (coord == ORC_SINHSPHERICAL) {
    *rad0 = 1.0 / rp;
    *rad1 = 0.0;
    *invr = 1.0 / r;
  } else {
    const double st = sin(x1), ct = cos(x1);
    const double b2 = bscale * bscale;
    const double AB = r * r + b2;
    const double Sg = r * r + b2 * st * st;
    const double dist = sqrt(r * r + b2 * ct * ct);
    *rad0 = r * AB / (rp * dist * Sg);
    *rad1 = -b2 * st * ct / (dist * Sg);
    *invr = 1.0 / dist;
  }
}

/* ------------------------------------------------------------------------------------------
 * C2 ("analytic solution to the momentum constraint"): Bowen-York extrinsic
 * curvature, summed over punctures BEFORE contraction.  With d = x - x_n, r = |d|, n = d/r:
 *   A^{ij} = 3/(2 r^2) [ P^i n^j + P^j n^i - (delta^{ij} - n^i n^j) (P.n) ]
 *          + 3/r^3     [ (S x n)^i n^j + (S x n)^j n^i ]
 * ---------------------------------------------------------------------------------------- */
void orc_bowen_york(int32_t n_punctures, const double* punctures, const double* xyz,
                    double* A) {
  for (int q = 0; q < 9; ++q) A[q] = 0.0;
  for (int p = 0; p < n_punctures; ++p) {
    const double* pp = punctures + 10 * p;
    const double* pos = pp + 1;
    const double* P = pp + 4;
    const double* S = pp + 7;
    double d[3], n[3], Sxn[3];
    for (int i = 0; i < 3; ++i) d[i] = xyz[i] - pos[i];
    const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    for (int i = 0; i < 3; ++i) n[i] = d[i] / r;
    const double Pn = P[0] * n[0] + P[1] * n[1] + P[2] * n[2];
    Sxn[0] = S[1] * n[2] - S[2] * n[1];
    Sxn[1] = S[2] * n[0] - S[0] * n[2];
    Sxn[2] = S[0] * n[1] - S[1] * n[0];
    const double fP = 3.0 / (2.0 * r * r);
    const double fS = 3.0 / (r * r * r);
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        const double delta = (i == j) ? 1.0 : 0.0;
        A[3 * i + j] += fP * (P[i] * n[j] + P[j] * n[i] - (delta - n[i] * n[j]) * Pn) +
                        fS * (Sxn[i] * n[j] + Sxn[j] * n[i]);
      }
  }
}

/* C1 (Eq. 3; Brandt-Bruegmann): psi_BL = 1 + sum_n m_n / (2 |x - x_n|). */
double orc_psi_bl(int32_t n_punctures, const double* punctures, const double* xyz) {
  double psi = 1.0;
  for (int p = 0; p < n_punctures; ++p) {
    const double* pp = punctures + 10 * p;
    const double dx = xyz[0] - pp[1], dy = xyz[1] - pp[2], dz = xyz[2] - pp[3];
    psi += pp[0] / (2.0 * sqrt(dx * dx + dy * dy + dz * dz));
  }
  return psi;
}

/* ------------------------------------------------------------------------------------------ */

static int orc_is_interior(const orc_grid* g, int a, int i) {
  return i >= g->ng && i < g->p.n[a] + g->ng;
}

/* C14: nearest grid index of coordinate x along axis a, and the fractional error. */
static int orc_nearest_index(const orc_grid* g, int a, double x, double* frac_err) {
  double xmin = (a == 2) ? -ORC_PI : ((a == 1 && g->p.coord == ORC_SINHCYLINDRICAL) ? -1.0 : 0.0);
  if (g->p.coord == ORC_SINHCARTESIAN) xmin = -1.0;
  const double j = (x - xmin) / g->dx[a] - 0.5 + (double)g->ng;
  const double jr = floor(j + 0.5);
  *frac_err = fabs(j - jr);
  return (int)jr;
}

/* C13: is the ghost point (i0,i1,i2) an OUTER point (radiation condition) rather than an inner one?
 *   SinhSpherical, SinhSymTP: i0 >= N0+NG with interior angles;
 *   SinhCylindrical (C24): beyond the outer cylinder or beyond either end face, i.e. x0 >= 0 and
 *   (i0 >= N0+NG or x1 outside [-1,1]), with interior phi.
 * These are exactly the ghost points whose Cartesian image maps back to themselves (a point
 * beyond the domain has no other representative); every other ghost point is an inner point. */
static int orc_is_outer(const orc_grid* g, int i0, int i1, int i2) {
  const int in1 = orc_is_interior(g, 1, i1), in2 = orc_is_interior(g, 2, i2);
  if (g->p.coord == ORC_SINHCARTESIAN) return 1; /* C25: no point has a second representative */
  if (!in2 || i0 < g->ng) return 0;
  if (g->p.coord == ORC_SINHCYLINDRICAL) return (i0 >= g->p.n[0] + g->ng) || !in1;
  return (i0 >= g->p.n[0] + g->ng) && in1;
}

/* PAPER.md:200 (Alg. 1 l.4), C13 + C14: classify every ghost point.
 *   outer : see orc_is_outer (the radiation condition is applied there);
 *   inner : every other ghost point; its Cartesian image mapped back into the fundamental
 *           domain lands on another grid point src, and value[dst] = +1 * value[src].      */
static int orc_build_bc(orc_grid* g) {
  const int T0 = g->T[0], T1 = g->T[1], T2 = g->T[2];
  int64_t n_inner = 0, n_outer = 0;
  for (int i2 = 0; i2 < T2; ++i2)
    for (int i1 = 0; i1 < T1; ++i1)
      for (int i0 = 0; i0 < T0; ++i0) {
        const int in0 = orc_is_interior(g, 0, i0), in1 = orc_is_interior(g, 1, i1),
                  in2 = orc_is_interior(g, 2, i2);
        if (in0 && in1 && in2) continue;
        if (orc_is_outer(g, i0, i1, i2))
          ++n_outer;
        else
          ++n_inner;
      }
  g->n_inner = n_inner;
  g->n_outer = n_outer;
  g->inner_dst = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_inner > 0 ? n_inner : 1));
  g->inner_src = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_inner > 0 ? n_inner : 1));
  g->outer_idx = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_outer > 0 ? n_outer : 1));
  int64_t ki = 0, ko = 0;
  double worst = 0.0;
  for (int i2 = 0; i2 < T2; ++i2)
    for (int i1 = 0; i1 < T1; ++i1)
      for (int i0 = 0; i0 < T0; ++i0) {
        const int in0 = orc_is_interior(g, 0, i0), in1 = orc_is_interior(g, 1, i1),
                  in2 = orc_is_interior(g, 2, i2);
        if (in0 && in1 && in2) continue;
        const int64_t idx = orc_idx(g, i0, i1, i2);
        if (orc_is_outer(g, i0, i1, i2)) {
          g->outer_idx[ko++] = (int32_t)idx;
          continue;
        }
        double xyz[3], x012[3], fe;
        orc_map_to_cart(g->p.coord, g->p.amp, g->p.sinhw, g->p.bscale, g->x0[i0], g->x1[i1],
                        g->x2[i2], xyz);
        orc_map_from_cart(g->p.coord, g->p.amp, g->p.sinhw, g->p.bscale, xyz, x012);
        int s[3];
        for (int a = 0; a < 3; ++a) {
          s[a] = orc_nearest_index(g, a, x012[a], &fe);
          if (fe > worst) worst = fe;
        }
        if (s[0] < 0 || s[0] >= T0 || s[1] < 0 || s[1] >= T1 || s[2] < 0 || s[2] >= T2)
          return -1;
        if (s[0] == i0 && s[1] == i1 && s[2] == i2) return -1; /* an inner point has another representative */
        g->inner_dst[ki] = (int32_t)idx;
        g->inner_src[ki] = (int32_t)orc_idx(g, s[0], s[1], s[2]);
        ++ki;
      }
  g->bc_max_frac_err = worst;
  return 0;
}

orc_grid* orc_create(const orc_params* p) {
  if (!p) return NULL;
  if (p->fd_order < 2 || p->fd_order > 2 * ORC_MAX_NG || (p->fd_order % 2)) return NULL;
  if (p->coord < ORC_SINHSPHERICAL || p->coord > ORC_SINHCARTESIAN) return NULL;
  const int ng = p->fd_order / 2;
  for (int a = 0; a < 3; ++a)
    if (p->n[a] < ng) return NULL;
  if (p->n[2] % 2) return NULL;
  if (!(p->amp > 0.0) || !(p->sinhw > 0.0) || !(p->cfl > 0.0) || !(p->c_min > 0.0) ||
      p->eta < 0.0 || p->n_punctures < 0)
    return NULL;
  if (p->coord == ORC_SINHSYMTP && !(p->bscale > 0.0)) return NULL;
  for (int q = 0; q < p->n_punctures; ++q)
    if (!(p->punctures[10 * q] > 0.0)) return NULL;

  orc_grid* g = (orc_grid*)calloc(1, sizeof(orc_grid));
  g->p = *p;
  g->punctures = (double*)malloc(sizeof(double) * 10 * (size_t)(p->n_punctures + 1));
  memcpy(g->punctures, p->punctures, sizeof(double) * 10 * (size_t)p->n_punctures);
  g->p.punctures = g->punctures;
  g->ng = ng;
  for (int a = 0; a < 3; ++a) g->T[a] = p->n[a] + 2 * ng;
  g->ntot = (int64_t)g->T[0] * g->T[1] * g->T[2];
  if (g->ntot >= (int64_t)2147483647) { /* int32 index lists */
    orc_destroy(g);
    return NULL;
  }

  /* C8: cell-centred uniform coordinates, x0 in [0,1], x1 in [0,pi] (C24: [-1,1]), x2 in [-pi,pi]. */
  const int cart = p->coord == ORC_SINHCARTESIAN;
  const double x1min = (p->coord == ORC_SINHCYLINDRICAL || cart) ? -1.0 : 0.0;
  const double x0min = cart ? -1.0 : 0.0, x2min = cart ? -1.0 : -ORC_PI;
  g->dx[0] = (cart ? 2.0 : 1.0) / (double)p->n[0];
  g->dx[1] = ((p->coord == ORC_SINHCYLINDRICAL || cart) ? 2.0 : ORC_PI) / (double)p->n[1];
  g->dx[2] = (cart ? 2.0 : 2.0 * ORC_PI) / (double)p->n[2];
  g->x0 = (double*)malloc(sizeof(double) * (size_t)g->T[0]);
  g->x1 = (double*)malloc(sizeof(double) * (size_t)g->T[1]);
  g->x2 = (double*)malloc(sizeof(double) * (size_t)g->T[2]);
  for (int i = 0; i < g->T[0]; ++i) g->x0[i] = x0min + ((double)(i - ng) + 0.5) * g->dx[0];
  for (int i = 0; i < g->T[1]; ++i) g->x1[i] = x1min + ((double)(i - ng) + 0.5) * g->dx[1];
  for (int i = 0; i < g->T[2]; ++i) g->x2[i] = x2min + ((double)(i - ng) + 0.5) * g->dx[2];
  /* C25: x2-dependent factors and, per axis, X_a and 1/h_a (1, 0, +inf, 1 and unused otherwise) */
  g->z22 = (double*)malloc(sizeof(double) * (size_t)g->T[2]);
  g->z2 = (double*)malloc(sizeof(double) * (size_t)g->T[2]);
  g->zds = (double*)malloc(sizeof(double) * (size_t)g->T[2]);
  g->zh = (double*)malloc(sizeof(double) * (size_t)g->T[2]);
  for (int i = 0; i < g->T[2]; ++i) {
    double h2, g22, g2;
    orc_metric_axis2(p->coord, p->amp, p->sinhw, g->x2[i], &h2, &g22, &g2);
    g->z22[i] = g22;
    g->z2[i] = g2;
    g->zh[i] = h2;
    g->zds[i] = cart ? fabs(h2) * g->dx[2] : INFINITY;
  }
  for (int a = 0; a < 3; ++a) {
    const double* xa = (a == 0) ? g->x0 : ((a == 1) ? g->x1 : g->x2);
    g->X[a] = (double*)malloc(sizeof(double) * (size_t)g->T[a]);
    g->ih[a] = (double*)malloc(sizeof(double) * (size_t)g->T[a]);
    for (int i = 0; i < g->T[a]; ++i) {
      double t, tp, tpp;
      orc_rho(p->amp, p->sinhw, xa[i], &t, &tp, &tpp);
      g->X[a][i] = t;
      g->ih[a][i] = 1.0 / tp;
    }
  }

  orc_fd_weights(p->fd_order, g->c1, g->d2);

  /* Alg. 1 l.3: reference-metric factors on the (i0,i1) plane (nothing depends on x2). */
  const size_t np = (size_t)g->T[0] * (size_t)g->T[1];
  double** planes[] = {&g->g00, &g->g11, &g->g22, &g->g0, &g->g1, &g->c,
                       &g->w,   &g->ds,  &g->rad0, &g->rad1, &g->invr};
  for (size_t q = 0; q < sizeof(planes) / sizeof(planes[0]); ++q)
    *planes[q] = (double*)malloc(sizeof(double) * np);
  for (int i1 = 0; i1 < g->T[1]; ++i1)
    for (int i0 = 0; i0 < g->T[0]; ++i0) {
      const size_t q = (size_t)i0 + (size_t)g->T[0] * (size_t)i1;
      double h[3], gf[5];
      orc_metric_at(p->coord, p->amp, p->sinhw, p->bscale, g->x0[i0], g->x1[i1], h, gf);
      g->g00[q] = gf[0];
      g->g11[q] = gf[1];
      g->g22[q] = gf[2];
      g->g0[q] = gf[3];
      g->g1[q] = gf[4];
      g->w[q] = fabs(h[0] * h[1] * h[2]);
      /* C9: local proper grid spacing ds = min_a |h_a| dx^a */
      double ds = fabs(h[0]) * g->dx[0];
      if (fabs(h[1]) * g->dx[1] < ds) ds = fabs(h[1]) * g->dx[1];
      if (!cart && fabs(h[2]) * g->dx[2] < ds) ds = fabs(h[2]) * g->dx[2]; /* C25: x2 part in zds */
      g->ds[q] = ds;
      orc_radial_at(p->coord, p->amp, p->sinhw, p->bscale, g->x0[i0], g->x1[i1], &g->rad0[q],
                    &g->rad1[q], &g->invr[q]);
    }
  /* C9 / PAPER.md:74, 213: ds_min over INTERIOR points, dt = CFL ds_min,
   * c(x) = c_min ds(x)/ds_min, so that c dt / ds = CFL c_min everywhere. */
  double dsmin = INFINITY;
  for (int i1 = ng; i1 < p->n[1] + ng; ++i1)
    for (int i0 = ng; i0 < p->n[0] + ng; ++i0) {
      const double ds = g->ds[(size_t)i0 + (size_t)g->T[0] * (size_t)i1];
      if (ds < dsmin) dsmin = ds;
    }
  for (int i2 = ng; i2 < p->n[2] + ng; ++i2) /* C25: the x2 spacing takes part in the minimum */
    if (g->zds[i2] < dsmin) dsmin = g->zds[i2];
  g->dsmin = dsmin;
  g->dt = p->cfl * dsmin;
  for (size_t q = 0; q < np; ++q) g->c[q] = p->c_min * g->ds[q] / dsmin;

  if (orc_build_bc(g) != 0) {
    orc_destroy(g);
    return NULL;
  }

  /* Alg. 1 l.7: constant source terms at every grid point (C1, C2); S = (1/8) A_ij A^ij with
   * Cartesian components and the flat metric. */
  g->psi = (double*)malloc(sizeof(double) * (size_t)g->ntot);
  g->S = (double*)malloc(sizeof(double) * (size_t)g->ntot);
  int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
  for (int i2 = 0; i2 < g->T[2]; ++i2)
    for (int i1 = 0; i1 < g->T[1]; ++i1)
      for (int i0 = 0; i0 < g->T[0]; ++i0) {
        double xyz[3], A[9];
        orc_map_to_cart(p->coord, p->amp, p->sinhw, p->bscale, g->x0[i0], g->x1[i1], g->x2[i2],
                        xyz);
        for (int a = 0; a < 3; ++a) xyz[a] += p->origin[a];
        const int64_t idx = orc_idx(g, i0, i1, i2);
        g->psi[idx] = orc_psi_bl(p->n_punctures, g->punctures, xyz);
        orc_bowen_york(p->n_punctures, g->punctures, xyz, A);
        double AA = 0.0;
        for (int q = 0; q < 9; ++q) AA += A[q] * A[q];
        g->S[idx] = 0.125 * AA;
        if (!isfinite(g->psi[idx]) || !isfinite(g->S[idx])) bad |= 1;
      }
  if (bad) { /* a puncture sits on a grid point */
    orc_destroy(g);
    return NULL;
  }
  return g;
}

void orc_destroy(orc_grid* g) {
  if (!g) return;
  free(g->punctures);
  free(g->x0);
  free(g->x1);
  free(g->x2);
  free(g->g00);
  free(g->g11);
  free(g->g22);
  free(g->g0);
  free(g->g1);
  free(g->c);
  free(g->w);
  free(g->ds);
  free(g->rad0);
  free(g->rad1);
  free(g->invr);
  free(g->z22);
  free(g->z2);
  free(g->zds);
  free(g->zh);
  for (int a = 0; a < 3; ++a) {
    free(g->X[a]);
    free(g->ih[a]);
  }
  free(g->inner_dst);
  free(g->inner_src);
  free(g->outer_idx);
  free(g->psi);
  free(g->S);
  free(g);
}

void orc_info(const orc_grid* g, double* dt, double* dsmin, int32_t* ng, int32_t* T,
              int64_t* ntot, int64_t* n_inner, int64_t* n_outer) {
  if (dt) *dt = g->dt;
  if (dsmin) *dsmin = g->dsmin;
  if (ng) *ng = g->ng;
  if (T)
    for (int a = 0; a < 3; ++a) T[a] = g->T[a];
  if (ntot) *ntot = g->ntot;
  if (n_inner) *n_inner = g->n_inner;
  if (n_outer) *n_outer = g->n_outer;
}

void orc_get_coords(const orc_grid* g, double* x0, double* x1, double* x2) {
  memcpy(x0, g->x0, sizeof(double) * (size_t)g->T[0]);
  memcpy(x1, g->x1, sizeof(double) * (size_t)g->T[1]);
  memcpy(x2, g->x2, sizeof(double) * (size_t)g->T[2]);
}

void orc_get_bc_lists(const orc_grid* g, int32_t* inner_dst, int32_t* inner_src,
                      int32_t* outer_idx) {
  if (inner_dst) memcpy(inner_dst, g->inner_dst, sizeof(int32_t) * (size_t)g->n_inner);
  if (inner_src) memcpy(inner_src, g->inner_src, sizeof(int32_t) * (size_t)g->n_inner);
  if (outer_idx) memcpy(outer_idx, g->outer_idx, sizeof(int32_t) * (size_t)g->n_outer);
}

double orc_bc_max_frac_err(const orc_grid* g) { return g->bc_max_frac_err; }

void orc_get_axis2(const orc_grid* g, double* z22, double* z2, double* zds, double* zh) {
  const size_t nb = sizeof(double) * (size_t)g->T[2];
  if (z22) memcpy(z22, g->z22, nb);
  if (z2) memcpy(z2, g->z2, nb);
  if (zds) memcpy(zds, g->zds, nb);
  if (zh) memcpy(zh, g->zh, nb);
}

void orc_get_source(const orc_grid* g, double* psi, double* S) {
  if (psi) memcpy(psi, g->psi, sizeof(double) * (size_t)g->ntot);
  if (S) memcpy(S, g->S, sizeof(double) * (size_t)g->ntot);
}

void orc_get_planes(const orc_grid* g, double* g00, double* g11, double* g22, double* g0,
                    double* g1, double* c, double* w, double* ds) {
  const size_t nb = sizeof(double) * (size_t)g->T[0] * (size_t)g->T[1];
  if (g00) memcpy(g00, g->g00, nb);
  if (g11) memcpy(g11, g->g11, nb);
  if (g22) memcpy(g22, g->g22, nb);
  if (g0) memcpy(g0, g->g0, nb);
  if (g1) memcpy(g1, g->g1, nb);
  if (c) memcpy(c, g->c, nb);
  if (w) memcpy(w, g->w, nb);
  if (ds) memcpy(ds, g->ds, nb);
}
