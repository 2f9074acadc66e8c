/*
 * hr_oracle.h -- CPU ORACLE for the hyperbolic-relaxation hot path of arxiv 2501.14030.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path
 * (paper_2501_14030_b200/csrc/) and neither includes the other.
 *
 * It is a plain, slow, literal restatement of
 *   PAPER.md:61-68   (Sec. 2, Eq. 4-5: the (u, v) relaxation system),
 *   PAPER.md:203-213 (Alg. 1 l.7, 9, 11-17: source terms, H, L2 norm, RHS -> BC -> RK),
 * with every formula the paper defers to its refs [9, 32, 33, 37] taken from the
 * readings C1-C21 of SURVEY.md Sec. 8(c), which DESIGN.md lists.  Each function
 * below names the passage or reading it follows.
 *
 * Parity status: every function is pinned by tests/test_oracle_*.py against
 * closed forms / invariants / brute force (pins P1-P12), EXCEPT the absolute
 * values of u and ||H|| after N steps, which the paper never prints:
 * "parity unpinned" for those two outputs (fixed only by oracle == GPU and by
 * the P11 invariants).
 *
 * Floating point: set-up (coordinates, reference-metric factors, wave speed,
 * dt, source terms, boundary maps) is always fp64 (reading C19).  The
 * evolution functions exist twice, suffix _f64 and _f32, compiled from the same
 * C file with ORC_REAL = double / float; they keep state, k, psi_BL, S and the
 * coefficient planes in ORC_REAL and accumulate the residual norm in fp64.
 */
#ifndef HR_ORACLE_H
#define HR_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* "Cartesian-like, spherical-like, cylindrical-like, and bispherical-like" reference metrics.
 * 0, 1: readings C4; 2: reading C24; 3: reading C25. */
enum { ORC_SINHSPHERICAL = 0, ORC_SINHSYMTP = 1, ORC_SINHCYLINDRICAL = 2, ORC_SINHCARTESIAN = 3 };

/* One puncture = 10 doubles: m, pos[3], P[3], S[3] (Cartesian). */
typedef struct {
  int32_t n[3];        /* interior points N0 N1 N2 (N2 even)                         */
  int32_t coord;       /* ORC_SINHSPHERICAL | ORC_SINHSYMTP (C4) | ORC_SINHCYLINDRICAL (C24) */
  int32_t fd_order;    /* 2,4,...,12; NG = fd_order/2 (C7)             */
  int32_t n_punctures;
  double amp, sinhw;   /* AMPL/SINHW or AMAX/SINHWAA (C4, C5)                        */
  double bscale;       /* SinhSymTP focal half-distance b (C4)                       */
  double origin[3];    /* Cartesian position of the grid centre (C6)                 */
  const double* punctures; /* n_punctures x 10 doubles                               */
  double eta;          /* damping factor of Eq. 5 (C10)                 */
  double cfl;          /* dt = cfl * ds_min (C9)                                     */
  double c_min;        /* wave-speed normalisation, c = c_min ds/ds_min (C9)         */
} orc_params;

typedef struct orc_grid orc_grid;

/* ---- set-up, fp64 (hr_oracle_setup.c) ---- */
orc_grid* orc_create(const orc_params* p);            /* NULL on invalid parameters */
void orc_destroy(orc_grid* g);
void orc_info(const orc_grid* g, double* dt, double* dsmin, int32_t* ng, int32_t* T,
              int64_t* ntot, int64_t* n_inner, int64_t* n_outer);
void orc_get_coords(const orc_grid* g, double* x0, double* x1, double* x2);
void orc_get_bc_lists(const orc_grid* g, int32_t* inner_dst, int32_t* inner_src,
                      int32_t* outer_idx);
double orc_bc_max_frac_err(const orc_grid* g);        /* worst |fractional index error| */
void orc_get_source(const orc_grid* g, double* psi, double* S);   /* ntot each, fp64 */
/* (i0,i1) planes, T0*T1 doubles each: Laplacian factors g00 g11 g22 g0 g1 (C4),
 * wave speed c (C9), volume weight |h0 h1 h2| (C16), local spacing ds (C9). */
void orc_get_planes(const orc_grid* g, double* g00, double* g11, double* g22, double* g0,
                    double* g1, double* c, double* w, double* ds);
/* C25 only (SinhCartesian): what depends on x2, T2 doubles each: the u_22 and u_2 factors 1/h2^2 and
 * -X2''/X2'^3, the spacing h2 dx2 and h2.  There lap u = g00 u_00 + g11 u_11 + z22 u_22 + g0 u_0 + g1 u_1
 * + z2 u_2, ds = min(ds plane, zds), |h0 h1 h2| = w plane * zh, and the c plane holds c_min ds_plane/ds_min.
 * For the other systems: 1, 0, +inf, 1. */
void orc_get_axis2(const orc_grid* g, double* z22, double* z2, double* zds, double* zh);

/* ---- stand-alone pieces exposed for the pins ---- */
/* C11: centred weights; c1[0..n] (c1[0]=0), d2[0..n], n = order/2, unit spacing. */
void orc_fd_weights(int32_t order, double* c1, double* d2);
/* C4: grid coordinates -> Cartesian (without origin shift). */
void orc_map_to_cart(int32_t coord, double amp, double sinhw, double bscale,
                     double x0, double x1, double x2, double* xyz);
/* C14: Cartesian -> (x0 >= 0, 0 <= th <= pi, -pi <= ph < pi). */
void orc_map_from_cart(int32_t coord, double amp, double sinhw, double bscale,
                       const double* xyz, double* x012);
/* C4: scale factors h0 h1 h2 and Laplacian factors at one coordinate. */
void orc_metric_at(int32_t coord, double amp, double sinhw, double bscale,
                   double x0, double x1, double* h, double* gfac);
/* C2: Bowen-York A~^{ij} (3x3 row-major, summed over punctures) at Cartesian x. */
void orc_bowen_york(int32_t n_punctures, const double* punctures, const double* xyz,
                    double* A);
/* C1: psi_BL at Cartesian x. */
double orc_psi_bl(int32_t n_punctures, const double* punctures, const double* xyz);

/* ---- evolution, typed (hr_oracle_step.c compiled twice) ---- */
#define ORC_DECL_TYPED(SUF, REAL)                                                          \
  /* a1: curvilinear FD Laplacian of u at interior points, 0 elsewhere (C4, C11, C12) */   \
  void orc_laplacian_##SUF(const orc_grid* g, const REAL* u, REAL* lap);                   \
  /* a1 only: k at interior points, ghosts left 0 (Eq. 5) */                               \
  void orc_rhs_interior_##SUF(const orc_grid* g, const REAL* u, const REAL* v, REAL* ku,   \
                              REAL* kv);                                                   \
  /* a2 only: radiation k at the outer points (C13); other entries untouched */            \
  void orc_bc_outer_##SUF(const orc_grid* g, const REAL* u, const REAL* v, REAL* ku,       \
                          REAL* kv);                                                       \
  /* a3 only: k[dst] = k[src] over the inner list (C14) */                                 \
  void orc_bc_inner_##SUF(const orc_grid* g, REAL* f);                                     \
  /* Alg. 1 l.13-14: a1 then a2 then a3; every one of the ntot entries is written */       \
  void orc_rhs_##SUF(const orc_grid* g, const REAL* u, const REAL* v, REAL* ku, REAL* kv); \
  /* Alg. 1 l.12-16 x nsteps: classic RK4 (C15), in place */                               \
  void orc_step_##SUF(const orc_grid* g, REAL* u, REAL* v, int64_t nsteps);                \
  /* a5: H at interior points (optional out, may be NULL) and its norm (C16).              \
   * out[0] = norm; out[1] = numerator sum; out[2] = denominator sum. */                   \
  void orc_residual_##SUF(const orc_grid* g, const REAL* u, int32_t mode, double* out,     \
                          REAL* H);

ORC_DECL_TYPED(f64, double)
ORC_DECL_TYPED(f32, float)

int32_t orc_num_threads(void); /* OpenMP threads the loops will use (1 if built without) */

#ifdef __cplusplus
}
#endif
#endif
