// hr_api.cu -- the extern "C" boundary of include/hr.h and the host-side set-up
// (Alg. 1 l.2-7).  Host logic only: coordinate tables, reference-metric
// factor planes, wave speed / dt, the closed-form integer boundary maps, workspace carving,
// CUDA-graph capture of one RK4 step.  Every per-point operation of the hot path runs in
// hr_kernels.cu; there is no CPU fallback.  Product code: nothing here touches oracle/.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>

#include "hr_internal.h"

namespace {

thread_local char g_err[512] = "";

hr_status fail(hr_status st, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return st;
}

#define HR_CUDA(call)                                                                       \
  do {                                                                                      \
    cudaError_t e__ = (call);                                                               \
    if (e__ != cudaSuccess)                                                                 \
      return fail(HR_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__),     \
                  __FILE__, __LINE__);                                                      \
  } while (0)

#define HR_TRY(expr)                \
  do {                              \
    hr_status st__ = (expr);        \
    if (st__ != HR_OK) return st__; \
  } while (0)

constexpr double kPi = 3.141592653589793238462643383279502884;

size_t align_up(size_t x, size_t a = 1024) { return (x + a - 1) / a * a; }

hr_status validate(const hr_params* p) {
  if (!p) return fail(HR_ERR_INVALID_ARG, "params is NULL");
  if (p->fd_order % 2 != 0 || p->fd_order < 2 || p->fd_order > 2 * HR_MAX_NG)
    return fail(HR_ERR_UNSUPPORTED, "fd_order %d not in {2,4,...,%d}", p->fd_order, 2 * HR_MAX_NG);
  if (p->coord < HR_SINHSPHERICAL || p->coord > HR_SINHCARTESIAN)
    return fail(HR_ERR_UNSUPPORTED, "coord %d unknown", p->coord);
  if (p->dtype != HR_F64 && p->dtype != HR_F32)
    return fail(HR_ERR_UNSUPPORTED, "dtype %d unknown", p->dtype);
  if (p->variant < 0 || p->variant > 3)
    return fail(HR_ERR_UNSUPPORTED, "variant %d unknown", p->variant);
  if ((p->coord == HR_SINHCYLINDRICAL || p->coord == HR_SINHCARTESIAN) && (p->variant == 1 || p->variant == 2))
    return fail(HR_ERR_UNSUPPORTED,
                "SinhCylindrical / SinhCartesian run in the marching arrangements (variant 0 or 3) only");
  const int ng = p->fd_order / 2;
  for (int a = 0; a < 3; ++a)
    if (p->n[a] < ng)
      return fail(HR_ERR_INVALID_ARG, "n[%d] = %d is smaller than NG = %d", a, p->n[a], ng);
  if (p->n[2] % 2) return fail(HR_ERR_INVALID_ARG, "n[2] = %d must be even (C14)", p->n[2]);
  {  // the kernels index the PADDED layout (row pitch P0) with int32: bound that, not N_tot
    int P0 = 0, off0 = 0;
    hrk_row_geometry(p->n[0] + 2 * ng, ng, p->dtype == HR_F64 ? 8 : 4, &P0, &off0);
    const double npad = double(P0) * double(p->n[1] + 2 * ng) * double(p->n[2] + 2 * ng + 1);
    if (npad + 1e6 >= 2147483647.0)
      return fail(HR_ERR_INVALID_ARG, "grid exceeds the int32 index range of the stored layout");
  }
  if (!(p->amp > 0) || !(p->sinhw > 0)) return fail(HR_ERR_INVALID_ARG, "amp, sinhw must be > 0");
  if (p->coord == HR_SINHSYMTP && !(p->bscale > 0))
    return fail(HR_ERR_INVALID_ARG, "bscale must be > 0 for SinhSymTP");
  if (!(p->cfl > 0) || !(p->c_min > 0) || !(p->eta >= 0))
    return fail(HR_ERR_INVALID_ARG, "need cfl > 0, c_min > 0, eta >= 0");
  if (p->residual_mode != 0 && p->residual_mode != 1)
    return fail(HR_ERR_INVALID_ARG, "residual_mode must be 0 or 1");
  if (p->n_punctures < 0 || (p->n_punctures > 0 && !p->punctures))
    return fail(HR_ERR_INVALID_ARG, "bad puncture list");
  for (int q = 0; q < p->n_punctures; ++q)
    if (!(p->punctures[q].m > 0)) return fail(HR_ERR_INVALID_ARG, "puncture %d: m must be > 0", q);
  return HR_OK;
}

// Workspace carving shared by hr_workspace_bytes and hr_create.
struct Layout {
  size_t off_field[10];
  size_t off_plane[6];
  size_t off_rad[3];
  size_t off_opos, off_zax[3], off_zh, off_ax;
  int axs;
  size_t off_wvol, off_inner_dst, off_inner_src, off_partials, off_result, off_counters;
  size_t off_rho, off_rhoz, off_sinth, off_costh, off_sinph, off_cosph, off_punct;
  size_t total;
  int64_t ntot, n_inner, npad;
  int T[3], ng, P0, off0;
  int nblocks;
};

Layout make_layout(const hr_params* p) {
  Layout L{};
  L.ng = p->fd_order / 2;
  for (int a = 0; a < 3; ++a) L.T[a] = p->n[a] + 2 * L.ng;
  L.ntot = (int64_t)L.T[0] * L.T[1] * L.T[2];
  // outer points (C13): NG layers beyond x0 at interior angles; C24: beyond the cylinder (all x1) and both ends
  int64_t n_outer = p->coord == HR_SINHCYLINDRICAL
                        ? ((int64_t)L.ng * L.T[1] + 2 * (int64_t)L.ng * p->n[0]) * p->n[2]
                        : (int64_t)L.ng * p->n[1] * p->n[2];
  if (p->coord == HR_SINHCARTESIAN) n_outer = L.ntot - (int64_t)p->n[0] * p->n[1] * p->n[2];  // C25: all ghosts
  L.n_inner = L.ntot - (int64_t)p->n[0] * p->n[1] * p->n[2] - n_outer;
  const size_t w = p->dtype == HR_F64 ? 8 : 4;
  hrk_row_geometry(L.T[0], L.ng, w, &L.P0, &L.off0);
  L.npad = (int64_t)L.P0 * L.T[1] * L.T[2];
  size_t off = 0;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off = align_up(off + bytes);
    return o;
  };
  for (int f = 0; f < 10; ++f) L.off_field[f] = take((size_t)L.npad * w);
  const size_t np = (size_t)L.T[0] * L.T[1];
  for (int f = 0; f < 6; ++f) L.off_plane[f] = take(np * w);
  // outer positions in the (i0,i1) plane: NG columns beyond x0 (all rows) + 2 NG rows beyond x1 (C24)
  const size_t n_o2_max = (size_t)L.ng * L.T[1] + 2 * (size_t)L.ng * L.T[0];
  for (int f = 0; f < 3; ++f) L.off_rad[f] = take(n_o2_max * w);
  L.off_opos = take(n_o2_max * 4);
  L.axs = std::max(L.T[0], std::max(L.T[1], L.T[2]));
  for (int f = 0; f < 3; ++f) L.off_zax[f] = take((size_t)L.T[2] * w);
  L.off_zh = take((size_t)L.T[2] * 8);
  L.off_ax = take((size_t)9 * L.axs * w);
  L.off_wvol = take(np * 8);
  L.off_inner_dst = take((size_t)L.n_inner * 4 + 4);
  L.off_inner_src = take((size_t)L.n_inner * 4 + 4);
  L.nblocks = hrk_max_partials(p->n, L.ng, p->dtype);
  L.off_partials = take((size_t)L.nblocks * 16);
  L.off_result = take(64);
  L.off_counters = take(256);
  L.off_rho = take((size_t)L.T[0] * 8);
  L.off_rhoz = take((size_t)L.T[0] * 8);
  L.off_sinth = take((size_t)L.T[1] * 8);
  L.off_costh = take((size_t)L.T[1] * 8);
  L.off_sinph = take((size_t)L.T[2] * 8);
  L.off_cosph = take((size_t)L.T[2] * 8);
  L.off_punct = take((size_t)(p->n_punctures + 1) * 80);
  L.total = off;
  return L;
}

// Reference-metric quantities at one (x0, theta) (reading C4 for the factors of
//   lap u = g00 u_00 + g11 u_11 + g22 u_22 + g0 u_0 + g1 u_1,
// C9 for the proper spacings, C13 for the radial-derivative factors).
struct MetricPoint {
  double g00, g11, g22, g0, g1;
  double h0, h1, h2;
  double rad0, rad1, invr;
};

struct Radial {  // rho(x0) = AMP sinh(x0/W)/sinh(1/W) and derivatives
  double f, d1, d2;
};

Radial radial_map(const hr_params& p, double x0) {
  const double inv = 1.0 / std::sinh(1.0 / p.sinhw);
  Radial r;
  r.f = p.amp * std::sinh(x0 / p.sinhw) * inv;
  r.d1 = p.amp * std::cosh(x0 / p.sinhw) * inv / p.sinhw;
  r.d2 = r.f / (p.sinhw * p.sinhw);
  return r;
}

// (SinhCylindrical, reading C24: Z = the same sinh map evaluated at x1.)
MetricPoint metric_point(const hr_params& p, const Radial& R, double sth, double cth, const Radial& Z) {
  MetricPoint m;
  const double A = R.f, A1 = R.d1, A2 = R.d2;
  if (p.coord == HR_SINHCARTESIAN) {
    // C25: h_a = X_a'; the x2 parts (h2, the u_22 and u_2 factors) are per-plane tables, not plane entries
    m.h0 = A1;
    m.h1 = Z.d1;
    m.h2 = std::numeric_limits<double>::infinity();  // takes no part in the plane's spacing minimum
    m.g00 = 1.0 / (A1 * A1);
    m.g11 = 1.0 / (Z.d1 * Z.d1);
    m.g22 = 1.0;
    m.g0 = -A2 / (A1 * A1 * A1);
    m.g1 = -Z.d2 / (Z.d1 * Z.d1 * Z.d1);
    m.rad0 = m.rad1 = m.invr = 0.0;  // the radiation factors depend on all three coordinates: in-kernel
  } else if (p.coord == HR_SINHCYLINDRICAL) {
    // flat metric in cylindrical coordinates (R(x0), Z(x1), phi): h = (R', Z', R)
    m.h0 = A1;
    m.h1 = Z.d1;
    m.h2 = A;
    m.g00 = 1.0 / (A1 * A1);
    m.g11 = 1.0 / (Z.d1 * Z.d1);
    m.g22 = 1.0 / (A * A);
    m.g0 = (1.0 / A - A2 / (A1 * A1)) / A1;
    m.g1 = -Z.d2 / (Z.d1 * Z.d1 * Z.d1);
    const double r = std::sqrt(A * A + Z.f * Z.f);  // distance from the grid centre
    m.rad0 = A / (r * A1);
    m.rad1 = Z.f / (r * Z.d1);
    m.invr = 1.0 / r;
  } else if (p.coord == HR_SINHSPHERICAL) {
    // flat metric in spherical coordinates with r = rho(x0)
    m.h0 = A1;
    m.h1 = A;
    m.h2 = A * sth;
    m.g00 = 1.0 / (A1 * A1);
    m.g11 = 1.0 / (A * A);
    m.g22 = m.g11 / (sth * sth);
    m.g0 = (2.0 / A - A2 / (A1 * A1)) / A1;
    m.g1 = m.g11 * cth / sth;
    m.rad0 = 1.0 / A1;
    m.rad1 = 0.0;
    m.invr = 1.0 / A;
  } else {
    // prolate-spheroidal-like (foci at z = +-b): Sigma = A^2 + b^2 sin^2, AB = A^2 + b^2
    const double b2 = p.bscale * p.bscale;
    const double AB = A * A + b2;
    const double Sig = A * A + b2 * sth * sth;
    const double iSig = 1.0 / Sig;
    m.h0 = A1 * std::sqrt(Sig / AB);
    m.h1 = std::sqrt(Sig);
    m.h2 = A * sth;
    m.g00 = AB * iSig / (A1 * A1);
    m.g11 = iSig;
    m.g22 = 1.0 / (A * A * sth * sth);
    m.g0 = iSig * ((2.0 * A * A + b2) / (A * A1) - AB * A2 / (A1 * A1 * A1));
    m.g1 = iSig * cth / sth;
    const double r = std::sqrt(A * A + b2 * cth * cth);  // distance from the grid centre
    m.rad0 = A * AB / (A1 * r * Sig);
    m.rad1 = -b2 * sth * cth / (r * Sig);
    m.invr = 1.0 / r;
  }
  return m;
}

// Closed-form integer inner map (reading C14).  Returns the source index triple of ghost point
// (i0,i1,i2); the caller has already excluded interior and outer points.
inline void inner_source(const hr_params& p, int ng, const int T[3], int i0, int i1, int i2,
                         int& j0, int& j1, int& j2) {
  const int N1 = p.n[1], N2 = p.n[2];
  int flips = 0;
  j0 = i0;
  j1 = i1;
  if (i0 < ng) {  // x0 -> -x0 : rho -> -rho
    j0 = 2 * ng - 1 - i0;
    ++flips;
    if (p.coord == HR_SINHSPHERICAL) j1 = T[1] - 1 - j1;  // r -> -r also sends theta -> pi - theta
  }
  if (p.coord == HR_SINHCYLINDRICAL) {
    // C24: x1 is the axial coordinate, points beyond its ends are outer points, nothing reflects
  } else if (j1 < ng) {  // theta -> -theta
    j1 = 2 * ng - 1 - j1;
    ++flips;
  } else if (j1 >= N1 + ng) {  // theta -> 2 pi - theta
    j1 = 2 * (N1 + ng) - 1 - j1;
    ++flips;
  }
  int k = i2 - ng + (flips & 1) * (N2 / 2);  // each flip shifts phi by pi
  k %= N2;
  if (k < 0) k += N2;
  j2 = k + ng;
}

template <typename T>
void to_working(const std::vector<double>& src, std::vector<char>& dst) {
  dst.resize(src.size() * sizeof(T));
  T* d = reinterpret_cast<T*>(dst.data());
  for (size_t i = 0; i < src.size(); ++i) d[i] = (T)src[i];  // setup in fp64, rounded once (C19)
}

hr_status upload(void* dst, const void* src, size_t bytes, cudaStream_t st) {
  if (bytes == 0) return HR_OK;
  HR_CUDA(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st));
  HR_CUDA(cudaStreamSynchronize(st));  // src is pageable and about to be freed
  return HR_OK;
}

hr_status upload_plane(const hr_solver* s, void* dst, const std::vector<double>& v) {
  std::vector<char> tmp;
  if (s->p.dtype == HR_F64)
    to_working<double>(v, tmp);
  else
    to_working<float>(v, tmp);
  return upload(dst, tmp.data(), tmp.size(), s->stream);
}

// Everything hr_create computes on the host (Alg. 1 l.2-4) before touching the device.
struct HostSetup {
  int ng, T[3];
  double dx[3], dsmin, dt;
  std::vector<double> rho, rhoz, sth, cth, sph, cph;           // 1-D coordinate tables
  std::vector<double> l00, l11, l22, l0, l1, c2, wv;           // (i0,i1) planes
  std::vector<double> r0, r1, ri;                              // compact outer planes (ng x T1)
  // the outer positions of the (i0,i1) plane in ascending order, what the kernels walk (C13): position
  // i0 + T0 i1 in the low 28 bits, stencil bits above (1: beyond x0, backward d_0; 2: beyond the high end
  // of x1, backward d_1; 4: beyond the low end of x1, forward d_1; centred otherwise) and their factors
  std::vector<int32_t> opos;
  std::vector<double> o_r0, o_r1, o_ri;
  // C25: per-plane tables (T2 each) and the nine per-axis tables of the six-face radiation condition
  std::vector<double> z22, z2, zc2, zh, ax;
  int axs = 0;
  std::vector<int32_t> inner_dst, inner_src, outer_idx;
};

hr_status host_setup(const hr_params* p, HostSetup& H) {
  const int ng = H.ng = p->fd_order / 2;
  for (int a = 0; a < 3; ++a) H.T[a] = p->n[a] + 2 * ng;
  const int T0 = H.T[0], T1 = H.T[1], T2 = H.T[2];
  const int n0 = p->n[0], n1 = p->n[1], n2 = p->n[2];
  // ---- Alg. 1 l.2: cell-centred coordinate tables (C8) ----
  const bool cart = p->coord == HR_SINHCARTESIAN;
  const bool cyl = p->coord == HR_SINHCYLINDRICAL;
  H.dx[0] = (cart ? 2.0 : 1.0) / n0;
  H.dx[1] = ((cyl || cart) ? 2.0 : kPi) / n1;
  H.dx[2] = (cart ? 2.0 : 2.0 * kPi) / n2;
  if ((int64_t)T0 * T1 >= (1 << 28)) return fail(HR_ERR_INVALID_ARG, "T0 * T1 exceeds 2^28");
  std::vector<Radial> R(T0), Zt(T1);
  H.rho.resize(T0); H.rhoz.resize(T0); H.sth.resize(T1); H.cth.resize(T1); H.sph.resize(T2);
  H.cph.resize(T2);
  for (int i = 0; i < T0; ++i) {
    R[i] = radial_map(*p, (cart ? -1.0 : 0.0) + (i - ng + 0.5) * H.dx[0]);
    H.rho[i] = R[i].f;
    H.rhoz[i] =
        p->coord == HR_SINHSYMTP ? std::sqrt(R[i].f * R[i].f + p->bscale * p->bscale) : R[i].f;
    if (cyl) H.rhoz[i] = 1.0;  // the source kernel forms z = rhoz[i0] * costh[i1]: here z = Z(x1)
    // (C25: the source kernel takes (x, y, z) = (rho[i0], costh[i1], cosph[i2]))
  }
  for (int i = 0; i < T1; ++i) {
    const double th = (i - ng + 0.5) * H.dx[1];
    H.sth[i] = std::sin(th);
    H.cth[i] = std::cos(th);
    Zt[i] = Radial{0.0, 0.0, 0.0};
    if (cyl || cart) {  // x1 in [-1,1]; (x, y, z) = (R cos phi, R sin phi, Z) or (X0, X1, X2)
      Zt[i] = radial_map(*p, -1.0 + (i - ng + 0.5) * H.dx[1]);
      H.sth[i] = 1.0;
      H.cth[i] = Zt[i].f;
    }
  }
  for (int i = 0; i < T2; ++i) {
    const double ph = -kPi + (i - ng + 0.5) * H.dx[2];
    H.sph[i] = std::sin(ph);
    H.cph[i] = std::cos(ph);
  }
  std::vector<Radial> X2t(T2);
  if (cart)
    for (int i = 0; i < T2; ++i) {
      X2t[i] = radial_map(*p, -1.0 + (i - ng + 0.5) * H.dx[2]);
      H.sph[i] = 0.0;
      H.cph[i] = X2t[i].f;
    }

  // ---- Alg. 1 l.3: reference-metric factor planes, wave speed, dt (C4, C9, C13, C16) ----
  const size_t np = (size_t)T0 * T1;
  for (auto* v : {&H.l00, &H.l11, &H.l22, &H.l0, &H.l1, &H.c2, &H.wv}) v->resize(np);
  std::vector<double> ds(np);
  std::vector<MetricPoint> mp(np);
  double dsmin = std::numeric_limits<double>::infinity();
  for (int i1 = 0; i1 < T1; ++i1)
    for (int i0 = 0; i0 < T0; ++i0) {
      const size_t q = (size_t)i0 + (size_t)T0 * i1;
      const MetricPoint m = metric_point(*p, R[i0], H.sth[i1], H.cth[i1], Zt[i1]);
      mp[q] = m;
      const double d = std::fmin(std::fabs(m.h0) * H.dx[0],
                                 std::fmin(std::fabs(m.h1) * H.dx[1], std::fabs(m.h2) * H.dx[2]));
      ds[q] = d;
      H.wv[q] = std::fabs(m.h0 * m.h1 * (cart ? 1.0 : m.h2));  // C25: the x2 factor is the ZH table
      const bool interior = i0 >= ng && i0 < n0 + ng && i1 >= ng && i1 < n1 + ng;
      if (interior && d < dsmin) dsmin = d;
    }
  if (cart)  // C25: the x2 spacing h2 dx2 takes part in the minimum
    for (int i2 = ng; i2 < n2 + ng; ++i2) dsmin = std::fmin(dsmin, std::fabs(X2t[i2].d1) * H.dx[2]);
  H.dsmin = dsmin;
  H.dt = p->cfl * dsmin;
  H.r0.assign((size_t)ng * T1, 0.0);
  H.r1.assign((size_t)ng * T1, 0.0);
  H.ri.assign((size_t)ng * T1, 0.0);
  for (int i1 = 0; i1 < T1; ++i1)
    for (int i0 = 0; i0 < T0; ++i0) {
      const size_t q = (size_t)i0 + (size_t)T0 * i1;
      const MetricPoint& m = mp[q];
      const double c = p->c_min * ds[q] / dsmin;
      H.l00[q] = m.g00 / (H.dx[0] * H.dx[0]);
      H.l11[q] = m.g11 / (H.dx[1] * H.dx[1]);
      H.l22[q] = m.g22 / (H.dx[2] * H.dx[2]);
      H.l0[q] = m.g0 / H.dx[0];
      H.l1[q] = m.g1 / H.dx[1];
      H.c2[q] = c * c;
      if (i0 >= n0 + ng) {
        const size_t qo = (size_t)(i0 - (n0 + ng)) + (size_t)ng * i1;
        H.r0[qo] = c * m.rad0 / (2.0 * H.dx[0]);
        H.r1[qo] = c * m.rad1 / (2.0 * H.dx[1]);
        H.ri[qo] = c * m.invr;
      }
      const bool in1 = i1 >= ng && i1 < n1 + ng;
      const bool outer = !cart && i0 >= ng && (cyl ? (i0 >= n0 + ng || !in1) : (i0 >= n0 + ng && in1));
      if (outer) {
        const int bits = (i0 >= n0 + ng ? 1 : 0) | (i1 >= n1 + ng ? 2 : 0) | (i1 < ng ? 4 : 0);
        H.opos.push_back((int32_t)q | (bits << 28));
        H.o_r0.push_back(c * m.rad0 / (2.0 * H.dx[0]));
        H.o_r1.push_back(c * m.rad1 / (2.0 * H.dx[1]));
        H.o_ri.push_back(c * m.invr);
      }
    }

  if (cart) {
    // per-plane tables and the per-axis tables of the radiation condition on the six faces
    for (auto* v : {&H.z22, &H.z2, &H.zc2, &H.zh}) v->resize((size_t)T2);
    for (int i = 0; i < T2; ++i) {
      const double h2 = X2t[i].d1;
      H.z22[i] = 1.0 / (h2 * h2 * H.dx[2] * H.dx[2]);
      H.z2[i] = -X2t[i].d2 / (h2 * h2 * h2) / H.dx[2];
      const double c = p->c_min * std::fabs(h2) * H.dx[2] / dsmin;
      H.zc2[i] = c * c;
      H.zh[i] = h2;
    }
    H.axs = std::max(T0, std::max(T1, T2));
    H.ax.assign((size_t)9 * H.axs, 0.0);
    const std::vector<Radial>* tabs[3] = {&R, &Zt, &X2t};
    const int Ta[3] = {T0, T1, T2};
    for (int a = 0; a < 3; ++a)
      for (int i = 0; i < Ta[a]; ++i) {
        const Radial& r = (*tabs[a])[i];
        H.ax[(size_t)(3 * a + 0) * H.axs + i] = r.f;
        H.ax[(size_t)(3 * a + 1) * H.axs + i] = 1.0 / (2.0 * H.dx[a] * r.d1);
        H.ax[(size_t)(3 * a + 2) * H.axs + i] = p->c_min * std::fabs(r.d1) * H.dx[a] / dsmin;
      }
  }

  // ---- Alg. 1 l.4: boundary containers (C13, C14), ascending destination index ----
  const int64_t ntot = (int64_t)T0 * T1 * T2;
  const int64_t n_outer = cart ? ntot - (int64_t)n0 * n1 * n2 : (int64_t)H.opos.size() * n2;
  const int64_t n_inner = ntot - (int64_t)n0 * n1 * n2 - n_outer;
  H.inner_dst.reserve((size_t)n_inner);
  H.inner_src.reserve((size_t)n_inner);
  H.outer_idx.reserve((size_t)n_outer);
  for (int i2 = 0; i2 < T2; ++i2)
    for (int i1 = 0; i1 < T1; ++i1) {
      const bool in1 = i1 >= ng && i1 < n1 + ng, in2 = i2 >= ng && i2 < n2 + ng;
      for (int i0 = 0; i0 < T0; ++i0) {
        const bool in0 = i0 >= ng && i0 < n0 + ng;
        if (in0 && in1 && in2) continue;  // interior
        if (cart || (in2 && i0 >= ng && (cyl ? (i0 >= n0 + ng || !in1) : (i0 >= n0 + ng && in1)))) {
          H.outer_idx.push_back(i0 + T0 * (i1 + T1 * i2));
          continue;  // outer
        }
        int j0, j1, j2;
        inner_source(*p, ng, H.T, i0, i1, i2, j0, j1, j2);
        H.inner_dst.push_back(i0 + T0 * (i1 + T1 * i2));
        H.inner_src.push_back(j0 + T0 * (j1 + T1 * j2));
      }
    }
  if ((int64_t)H.inner_dst.size() != n_inner || (int64_t)H.outer_idx.size() != n_outer)
    return fail(HR_ERR_INVALID_ARG, "internal: boundary list sizes inconsistent");
  return HR_OK;
}

hr_status enqueue_rk4_step(const hr_solver* s) {
  for (int stage = 1; stage <= 4; ++stage) HR_CUDA(hrk_substep(s, stage));
  return HR_OK;
}

void forget_many_graphs(const hr_solver* s);  // hr_step_many's cached graphs, below

}  // namespace

extern "C" {

const char* hr_last_error(void) { return g_err; }

const char* hr_version(void) { return "hr-b200 0.1 (sm_100a)"; }

hr_status hr_workspace_bytes(const hr_params* p, size_t* bytes) {
  hr_status st = validate(p);
  if (st != HR_OK) return st;
  if (!bytes) return fail(HR_ERR_INVALID_ARG, "bytes is NULL");
  *bytes = make_layout(p).total;
  return HR_OK;
}

hr_status hr_create(const hr_params* p, void* workspace_dev, size_t workspace_bytes,
                    hr_solver** out) {
  hr_status st = validate(p);
  if (st != HR_OK) return st;
  if (!out) return fail(HR_ERR_INVALID_ARG, "out is NULL");
  const Layout L = make_layout(p);
  if (!workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) & 255u))
    return fail(HR_ERR_WORKSPACE, "workspace must be a 256-byte aligned device pointer");
  if (workspace_bytes < L.total)
    return fail(HR_ERR_WORKSPACE, "workspace has %zu bytes, %zu needed", workspace_bytes, L.total);
  HR_CUDA(cudaSetDevice(p->device));

  hr_solver* s = new (std::nothrow) hr_solver();
  if (!s) return fail(HR_ERR_INVALID_ARG, "out of host memory");
  struct Guard {
    hr_solver* s;
    ~Guard() { if (s) hr_destroy(s); }
  } guard{s};

  s->p = *p;
  s->punctures.assign(p->punctures, p->punctures + p->n_punctures);
  s->p.punctures = s->punctures.data();
  s->stream = static_cast<cudaStream_t>(p->stream);
  s->step_graph = nullptr;
  s->step_resid_graph[0] = s->step_resid_graph[1] = nullptr;
  s->workspace = workspace_dev;
  s->workspace_bytes = workspace_bytes;
  s->scalar_bytes = p->dtype == HR_F64 ? 8 : 4;
  const int ng = L.ng;
  HrGrid& g = s->g;
  g.n0 = p->n[0]; g.n1 = p->n[1]; g.n2 = p->n[2];
  g.ng = ng;
  g.T0 = L.T[0]; g.T1 = L.T[1]; g.T2 = L.T[2];
  g.P0 = L.P0;
  g.off0 = L.off0;
  g.s1 = g.P0;
  g.s2 = (int64_t)g.P0 * g.T1;
  g.npad = L.npad;
  g.ntot = L.ntot;
  g.n_inner = L.n_inner;
  g.n_outer_cols = ng;
  s->n_outer = 0;  // set from the host tables below
  s->max_partials = L.nblocks;
  s->plan = hrk_make_plan(p->n, ng, p->coord, p->dtype);
  HR_CUDA(cudaDeviceGetAttribute(&s->num_sms, cudaDevAttrMultiProcessorCount, p->device));

  char* base = static_cast<char*>(workspace_dev);
  HrArrays& a = s->a;
  a.Y[0] = base + L.off_field[0];   a.Y[1] = base + L.off_field[1];
  a.A[0] = base + L.off_field[2];   a.A[1] = base + L.off_field[3];
  a.B[0] = base + L.off_field[4];   a.B[1] = base + L.off_field[5];
  a.ACC[0] = base + L.off_field[6]; a.ACC[1] = base + L.off_field[7];
  a.psi = base + L.off_field[8];    a.S = base + L.off_field[9];
  a.L00 = base + L.off_plane[0]; a.L11 = base + L.off_plane[1]; a.L22 = base + L.off_plane[2];
  a.L0 = base + L.off_plane[3];  a.L1 = base + L.off_plane[4];  a.C2 = base + L.off_plane[5];
  a.RAD0 = base + L.off_rad[0]; a.RAD1 = base + L.off_rad[1]; a.RADI = base + L.off_rad[2];
  a.OPOS = reinterpret_cast<int32_t*>(base + L.off_opos);
  a.Z22 = base + L.off_zax[0]; a.Z2 = base + L.off_zax[1]; a.ZC2 = base + L.off_zax[2];
  a.ZH = reinterpret_cast<double*>(base + L.off_zh);
  a.AX = base + L.off_ax;
  a.AXS = L.axs;
  a.Wvol = reinterpret_cast<double*>(base + L.off_wvol);
  a.inner_dst = reinterpret_cast<int32_t*>(base + L.off_inner_dst);
  a.inner_src = reinterpret_cast<int32_t*>(base + L.off_inner_src);
  a.partials = reinterpret_cast<double*>(base + L.off_partials);
  a.result2 = reinterpret_cast<double*>(base + L.off_result);
  s->plan.counters = reinterpret_cast<int*>(base + L.off_counters);
  s->plan.flag = s->plan.counters + 62;
  HR_CUDA(cudaMemsetAsync(s->plan.counters, 0, 256, s->stream));
  HR_CUDA(cudaHostAlloc(reinterpret_cast<void**>(&s->pinned), 8 * sizeof(double), cudaHostAllocDefault));
  for (auto& e : s->relax_ev) HR_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  a.rho = reinterpret_cast<double*>(base + L.off_rho);
  a.rhoz = reinterpret_cast<double*>(base + L.off_rhoz);
  a.sinth = reinterpret_cast<double*>(base + L.off_sinth);
  a.costh = reinterpret_cast<double*>(base + L.off_costh);
  a.sinph = reinterpret_cast<double*>(base + L.off_sinph);
  a.cosph = reinterpret_cast<double*>(base + L.off_cosph);
  a.punct = reinterpret_cast<double*>(base + L.off_punct);

  HR_CUDA(hrk_prepare(s));  // tensor maps, shared-memory opt-in, persistent grid sizes
  if ((int64_t)s->plan.ntx * s->plan.nty * s->plan.nzc > s->max_partials)
    return fail(HR_ERR_WORKSPACE, "internal: %lld work items but room for %d residual partials",
                (long long)s->plan.ntx * s->plan.nty * s->plan.nzc, s->max_partials);

  // ---- Alg. 1 l.2-4 on the host ----
  HostSetup H;
  HR_TRY(host_setup(p, H));
  for (int a = 0; a < 3; ++a) s->dx[a] = H.dx[a];
  s->dsmin = H.dsmin;
  s->dt = H.dt;
  s->inner_dst = std::move(H.inner_dst);
  s->inner_src = std::move(H.inner_src);
  s->outer_idx = std::move(H.outer_idx);
  const size_t np = (size_t)g.T0 * g.T1;

  // ---- upload tables ----
  HR_TRY(upload_plane(s, a.L00, H.l00));
  HR_TRY(upload_plane(s, a.L11, H.l11));
  HR_TRY(upload_plane(s, a.L22, H.l22));
  HR_TRY(upload_plane(s, a.L0, H.l0));
  HR_TRY(upload_plane(s, a.L1, H.l1));
  HR_TRY(upload_plane(s, a.C2, H.c2));
  HR_TRY(upload_plane(s, a.RAD0, H.o_r0));
  HR_TRY(upload_plane(s, a.RAD1, H.o_r1));
  HR_TRY(upload_plane(s, a.RADI, H.o_ri));
  HR_TRY(upload(a.OPOS, H.opos.data(), H.opos.size() * 4, s->stream));
  if (p->coord == HR_SINHCARTESIAN) {
    HR_TRY(upload_plane(s, a.Z22, H.z22));
    HR_TRY(upload_plane(s, a.Z2, H.z2));
    HR_TRY(upload_plane(s, a.ZC2, H.zc2));
    HR_TRY(upload(a.ZH, H.zh.data(), H.zh.size() * 8, s->stream));
    HR_TRY(upload_plane(s, a.AX, H.ax));
  }
  s->n_outer = (int64_t)s->outer_idx.size();
  s->g.n_o2 = (int32_t)H.opos.size();
  hrk_replan(s, 1);  // the plan carries the multiply-shift constants of g.n_o2 (outer-point loop)
  HR_TRY(upload(a.Wvol, H.wv.data(), np * 8, s->stream));
  {
    // device copies of the inner lists in stored (padded) indices; the host copies stay public
    auto stored = [&](const std::vector<int32_t>& v) {
      std::vector<int32_t> r(v.size());
      for (size_t i = 0; i < v.size(); ++i) {
        const int32_t row = v[i] / g.T0;
        r[i] = g.off0 + (v[i] - row * g.T0) + g.P0 * row;
      }
      return r;
    };
    const std::vector<int32_t> d = stored(s->inner_dst), sr = stored(s->inner_src);
    HR_TRY(upload(a.inner_dst, d.data(), d.size() * 4, s->stream));
    HR_TRY(upload(a.inner_src, sr.data(), sr.size() * 4, s->stream));
  }
  HR_TRY(upload(a.rho, H.rho.data(), H.rho.size() * 8, s->stream));
  HR_TRY(upload(a.rhoz, H.rhoz.data(), H.rhoz.size() * 8, s->stream));
  HR_TRY(upload(a.sinth, H.sth.data(), H.sth.size() * 8, s->stream));
  HR_TRY(upload(a.costh, H.cth.data(), H.cth.size() * 8, s->stream));
  HR_TRY(upload(a.sinph, H.sph.data(), H.sph.size() * 8, s->stream));
  HR_TRY(upload(a.cosph, H.cph.data(), H.cph.size() * 8, s->stream));
  static_assert(sizeof(hr_puncture) == 80, "hr_puncture is 10 packed doubles");
  HR_TRY(upload(a.punct, s->punctures.data(), s->punctures.size() * sizeof(hr_puncture), s->stream));

  // ---- Alg. 1 l.5, 7: zero state (C17) and constant source terms on the device ----
  const size_t fb = (size_t)g.npad * s->scalar_bytes;
  for (void* f : {a.Y[0], a.Y[1], a.A[0], a.A[1], a.B[0], a.B[1], a.ACC[0], a.ACC[1], a.psi, a.S})
    HR_CUDA(cudaMemsetAsync(f, 0, fb, s->stream));
  HR_CUDA(hrk_source(s));
  int bad = 0;
  HR_CUDA(cudaMemcpyAsync(&bad, a.result2, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  HR_CUDA(cudaStreamSynchronize(s->stream));
  if (bad) return fail(HR_ERR_NUMERIC, "a puncture coincides with a grid point");

  // ---- one RK4 step as a CUDA graph (launch-bound on small grids) ----
  s->launches_per_step = 4 * hrk_launches_per_substep(s);
  if (s->stream != nullptr) {
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      hr_status cst = enqueue_rk4_step(s);
      cudaError_t ce = cudaStreamEndCapture(s->stream, &graph);
      if (cst == HR_OK && ce == cudaSuccess && graph) {
        if (cudaGraphInstantiate(&s->step_graph, graph, 0) != cudaSuccess) s->step_graph = nullptr;
      }
      if (graph) cudaGraphDestroy(graph);
    }
    cudaGetLastError();  // a failed capture falls back to direct launches of the same kernels
  }

  guard.s = nullptr;
  *out = s;
  return HR_OK;
}

hr_status hr_host_setup(const hr_params* p, double* dt, double* dsmin, int64_t* n_inner,
                        int64_t* n_outer, int32_t* inner_dst, int32_t* inner_src,
                        int32_t* outer_idx, double* planes7, double* outer3) {
  hr_status st = validate(p);
  if (st != HR_OK) return st;
  HostSetup H;
  HR_TRY(host_setup(p, H));
  if (dt) *dt = H.dt;
  if (dsmin) *dsmin = H.dsmin;
  if (n_inner) *n_inner = (int64_t)H.inner_dst.size();
  if (n_outer) *n_outer = (int64_t)H.outer_idx.size();
  if (inner_dst) memcpy(inner_dst, H.inner_dst.data(), H.inner_dst.size() * 4);
  if (inner_src) memcpy(inner_src, H.inner_src.data(), H.inner_src.size() * 4);
  if (outer_idx) memcpy(outer_idx, H.outer_idx.data(), H.outer_idx.size() * 4);
  if (planes7) {
    const size_t np = H.l00.size();
    const std::vector<double>* v[7] = {&H.l00, &H.l11, &H.l22, &H.l0, &H.l1, &H.c2, &H.wv};
    for (int f = 0; f < 7; ++f) memcpy(planes7 + f * np, v[f]->data(), np * 8);
  }
  if (outer3) {
    const size_t no = H.r0.size();
    memcpy(outer3, H.r0.data(), no * 8);
    memcpy(outer3 + no, H.r1.data(), no * 8);
    memcpy(outer3 + 2 * no, H.ri.data(), no * 8);
  }
  return HR_OK;
}

hr_status hr_destroy(hr_solver* s) {
  if (!s) return HR_OK;
  forget_many_graphs(s);
  if (s->step_graph) cudaGraphExecDestroy(s->step_graph);
  for (cudaGraphExec_t g : s->step_resid_graph)
    if (g) cudaGraphExecDestroy(g);
  if (s->pinned) cudaFreeHost(s->pinned);
  for (cudaEvent_t e : s->relax_ev)
    if (e) cudaEventDestroy(e);
  delete s;
  return HR_OK;
}

hr_status hr_step(hr_solver* s, int64_t n_steps) {
  if (!s) return fail(HR_ERR_INVALID_ARG, "solver is NULL");
  if (n_steps < 0) return fail(HR_ERR_INVALID_ARG, "n_steps < 0");
  for (int64_t i = 0; i < n_steps; ++i) {
    if (s->step_graph) {
      HR_CUDA(cudaGraphLaunch(s->step_graph, s->stream));
    } else {
      hr_status st = enqueue_rk4_step(s);
      if (st != HR_OK) return st;
    }
  }
  return HR_OK;
}

hr_status hr_step_residual_async(hr_solver* s, int32_t mode, double* out2_dev) {
  if (!s || !out2_dev) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  if (mode != 0 && mode != 1) return fail(HR_ERR_INVALID_ARG, "mode must be 0 or 1");
  double* slot = s->a.result2 + 6;  // the graph's fixed output; copied on to the caller's pointer
  if (s->stream != nullptr && !s->step_resid_graph[mode] && !s->step_resid_tried[mode]) {
    // captured on first use, one graph per residual mode (launch-bound on small grids)
    s->step_resid_tried[mode] = true;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      const cudaError_t le = hrk_step_with_residual(s, mode, slot);
      const cudaError_t ce = cudaStreamEndCapture(s->stream, &graph);
      if (le == cudaSuccess && ce == cudaSuccess && graph &&
          cudaGraphInstantiate(&s->step_resid_graph[mode], graph, 0) != cudaSuccess)
        s->step_resid_graph[mode] = nullptr;
      if (graph) cudaGraphDestroy(graph);
    }
    cudaGetLastError();  // a failed capture falls back to direct launches of the same kernels
  }
  if (s->step_resid_graph[mode]) {
    HR_CUDA(cudaGraphLaunch(s->step_resid_graph[mode], s->stream));
    HR_CUDA(cudaMemcpyAsync(out2_dev, slot, 2 * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
  } else {
    HR_CUDA(hrk_step_with_residual(s, mode, out2_dev));
  }
  return HR_OK;
}

// hr_step_many: the N solvers' steps as ONE CUDA graph with N parallel branches of k RK4 steps each (captured
// once per solver set and k, cached).  On small grids a step is four ~6 us kernels that fill a fraction of the
// SMs: replaying per-solver graphs from the host is bound by the host's launch rate (profiles/r1c.md: 1.5-1.7x
// at N = 7), while one graph lets the device overlap the branches and costs one launch per k steps of all N.
}  // extern "C"

namespace {

struct ManyGraph {
  std::vector<hr_solver*> key;
  int k;
  cudaGraphExec_t exec;
};
std::mutex g_many_mu;
std::vector<ManyGraph> g_many;
constexpr int kManyStepsPerGraph = 8;

cudaGraphExec_t many_graph(hr_solver* const* solvers, int32_t n, int k) {
  std::lock_guard<std::mutex> lock(g_many_mu);
  for (const ManyGraph& m : g_many)
    if (m.k == k && (int32_t)m.key.size() == n && std::equal(m.key.begin(), m.key.end(), solvers)) return m.exec;
  cudaStream_t s0 = solvers[0]->stream;
  std::vector<cudaEvent_t> ev((size_t)n, nullptr);
  bool ok = true;
  for (auto& e : ev) ok = ok && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  if (ok && cudaStreamBeginCapture(s0, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
    ok = cudaEventRecord(ev[0], s0) == cudaSuccess;  // fork
    for (int32_t i = 1; i < n && ok; ++i)
      if (solvers[i]->stream != s0) ok = cudaStreamWaitEvent(solvers[i]->stream, ev[0], 0) == cudaSuccess;
    // the branches run side by side: each solver chunks its grid as if 1/n of the CTA slots were its own
    // (longer chunks, fewer window primings; bit-identical results, the plan only orders the work)
    for (int32_t i = 0; i < n; ++i) hrk_replan(solvers[i], n);
    for (int32_t i = 0; i < n && ok; ++i)
      for (int it = 0; it < k && ok; ++it) ok = enqueue_rk4_step(solvers[i]) == HR_OK;
    for (int32_t i = 0; i < n; ++i) hrk_replan(solvers[i], 1);
    for (int32_t i = 1; i < n && ok; ++i) {  // join
      if (solvers[i]->stream == s0) continue;
      ok = cudaEventRecord(ev[i], solvers[i]->stream) == cudaSuccess &&
           cudaStreamWaitEvent(s0, ev[i], 0) == cudaSuccess;
    }
    const cudaError_t ce = cudaStreamEndCapture(s0, &graph);
    if (!ok || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) exec = nullptr;
    if (graph) cudaGraphDestroy(graph);
  }
  cudaGetLastError();
  for (cudaEvent_t e : ev)
    if (e) cudaEventDestroy(e);
  if (exec) g_many.push_back(ManyGraph{std::vector<hr_solver*>(solvers, solvers + n), k, exec});
  return exec;
}

void forget_many_graphs(const hr_solver* s) {  // hr_destroy: graphs that replay this solver's kernels
  std::lock_guard<std::mutex> lock(g_many_mu);
  for (size_t i = 0; i < g_many.size();) {
    if (std::find(g_many[i].key.begin(), g_many[i].key.end(), s) != g_many[i].key.end()) {
      cudaGraphExecDestroy(g_many[i].exec);
      g_many.erase(g_many.begin() + (long)i);
    } else {
      ++i;
    }
  }
}

}  // namespace

extern "C" {

hr_status hr_step_many(hr_solver* const* solvers, int32_t n, int64_t n_steps) {
  if (n < 0 || n_steps < 0 || (n > 0 && !solvers)) return fail(HR_ERR_INVALID_ARG, "bad arguments");
  for (int32_t i = 0; i < n; ++i)
    if (!solvers[i]) return fail(HR_ERR_INVALID_ARG, "solver %d is NULL", i);
  bool graphable = n >= 2;
  for (int32_t i = 0; i < n && graphable; ++i) {
    graphable = solvers[i]->stream != nullptr && solvers[i]->p.device == solvers[0]->p.device;
    for (int32_t j = 0; j < i && graphable; ++j) graphable = solvers[j] != solvers[i];
  }
  int64_t left = n_steps;
  if (graphable && left > 0) {
    cudaStream_t s0 = solvers[0]->stream;
    // the graph runs in solver 0's stream: it starts after the work already queued in the other streams ...
    for (int32_t i = 1; i < n; ++i) {
      if (solvers[i]->stream == s0) continue;
      HR_CUDA(cudaEventRecord(solvers[i]->relax_ev[0], solvers[i]->stream));
      HR_CUDA(cudaStreamWaitEvent(s0, solvers[i]->relax_ev[0], 0));
    }
    while (left > 0) {
      const int k = left >= kManyStepsPerGraph ? kManyStepsPerGraph : (int)left;
      cudaGraphExec_t exec = many_graph(solvers, n, k);
      if (!exec) break;  // capture failed: plain round robin below
      HR_CUDA(cudaGraphLaunch(exec, s0));
      left -= k;
    }
    // ... and whatever is queued in them next waits for it
    HR_CUDA(cudaEventRecord(solvers[0]->relax_ev[1], s0));
    for (int32_t i = 1; i < n; ++i)
      if (solvers[i]->stream != s0) HR_CUDA(cudaStreamWaitEvent(solvers[i]->stream, solvers[0]->relax_ev[1], 0));
  }
  for (int64_t it = 0; it < left; ++it)
    for (int32_t i = 0; i < n; ++i) HR_TRY(hr_step(solvers[i], 1));
  return HR_OK;
}

hr_status hr_residual_async(hr_solver* s, int32_t mode, double* out2_dev) {
  if (!s || !out2_dev) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  if (mode != 0 && mode != 1) return fail(HR_ERR_INVALID_ARG, "mode must be 0 or 1");
  HR_CUDA(hrk_residual(s, mode, out2_dev));
  return HR_OK;
}

hr_status hr_residual_static(hr_solver* s, int32_t mode, double* out2_dev) {
  if (!s || !out2_dev) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  if (mode != 0 && mode != 1) return fail(HR_ERR_INVALID_ARG, "mode must be 0 or 1");
  if (s->p.variant == 1 || s->p.variant == 2)
    return fail(HR_ERR_INVALID_ARG, "hr_residual_static serves the marching arrangements (variant 0 or 3), not variant %d",
                (int)s->p.variant);
  const int64_t items = (int64_t)s->plan.ntx * s->plan.nty * s->plan.nzc;
  if (items > HR_STATIC_MAX_PARTIALS)
    return fail(HR_ERR_WORKSPACE,
                "hr_residual_static: %lld (tile, chunk) partials, the static scratch holds %d; use hr_residual_async",
                (long long)items, HR_STATIC_MAX_PARTIALS);
  HR_CUDA(hrk_residual_static(s, mode, out2_dev));
  return HR_OK;
}

hr_status hr_residual_ex(hr_solver* s, int32_t mode, double* out3) {
  if (!s || !out3) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  hr_status st = hr_residual_async(s, mode, s->a.result2);
  if (st != HR_OK) return st;
  double* h = s->pinned + 4;  // pinned: {num, den}, then the numeric flag
  int* flag = reinterpret_cast<int*>(s->pinned + 6);
  HR_CUDA(cudaMemcpyAsync(h, s->a.result2, 2 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
  HR_CUDA(cudaMemcpyAsync(flag, s->plan.flag, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  HR_CUDA(cudaStreamSynchronize(s->stream));
  if (*flag) return fail(HR_ERR_NUMERIC, "psi_BL + u <= 0 or a non-finite value at an interior point");
  out3[0] = std::sqrt(h[0] / h[1]);
  out3[1] = h[0];
  out3[2] = h[1];
  return HR_OK;
}

hr_status hr_relax(hr_solver* s, int64_t max_steps, int64_t check_every, double tol, int32_t mode,
                   int64_t* steps_done, double* final_residual, double* history,
                   int64_t history_cap, int64_t* n_history) {
  if (!s) return fail(HR_ERR_INVALID_ARG, "solver is NULL");
  if (max_steps < 0 || check_every < 1 || !(tol >= 0) || (mode != 0 && mode != 1))
    return fail(HR_ERR_INVALID_ARG, "need max_steps >= 0, check_every >= 1, tol >= 0, mode 0 or 1");
  if (history && history_cap < 0) return fail(HR_ERR_INVALID_ARG, "history_cap < 0");
  // two pinned slots and two events (owned by the solver): the host tests block k-1 while block k runs
  struct {
    double* h;
    cudaEvent_t* ev;
  } pin{s->pinned, s->relax_ev};
  double* dev = s->a.result2 + 2;  // device slots {num, den} x 2 behind hr_residual's own pair
  int64_t done = 0, nh = 0, k = 0;
  double last_r = 0.0;
  bool met = false;
  auto test_block = [&](int64_t kk) -> hr_status {
    HR_CUDA(cudaEventSynchronize(pin.ev[kk & 1]));
    const double r = std::sqrt(pin.h[2 * (kk & 1)] / pin.h[2 * (kk & 1) + 1]);
    last_r = r;
    if (history && nh < history_cap) history[nh] = r;
    ++nh;
    if (tol > 0 && r <= tol) met = true;
    return HR_OK;
  };
  while (true) {
    // residual k belongs to the state after k blocks.  It is reduced by the first substep of the
    // block that follows (hr_step_residual_async: no pass of its own) -- unless no block follows.
    if (k > 0) HR_TRY(test_block(k - 1));  // long complete: the device is busy with block k-1
    const int64_t n = max_steps - done < check_every ? max_steps - done : check_every;
    const bool last = met || n <= 0;
    if (last) {
      HR_CUDA(hrk_residual(s, mode, dev + 2 * (k & 1)));
    } else {
      HR_TRY(hr_step_residual_async(s, mode, dev + 2 * (k & 1)));
    }
    HR_CUDA(cudaMemcpyAsync(pin.h + 2 * (k & 1), dev + 2 * (k & 1), 2 * sizeof(double),
                            cudaMemcpyDeviceToHost, s->stream));
    HR_CUDA(cudaEventRecord(pin.ev[k & 1], s->stream));
    if (last) {
      HR_TRY(test_block(k));  // the residual of the final state closes the history
      break;
    }
    if (n > 1) HR_TRY(hr_step(s, n - 1));
    done += n;
    ++k;
  }
  // the last block's residual IS the residual of the returned state (its event has been waited for)
  int* flag = reinterpret_cast<int*>(s->pinned + 6);
  HR_CUDA(cudaMemcpyAsync(flag, s->plan.flag, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  HR_CUDA(cudaStreamSynchronize(s->stream));
  if (*flag) return fail(HR_ERR_NUMERIC, "psi_BL + u <= 0 or a non-finite value at an interior point");
  if (steps_done) *steps_done = done;
  if (n_history) *n_history = nh;
  if (final_residual) *final_residual = last_r;
  return HR_OK;
}

hr_status hr_residual(hr_solver* s, double* out) {
  if (!s || !out) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  double o3[3];
  hr_status st = hr_residual_ex(s, s->p.residual_mode, o3);
  if (st == HR_OK) *out = o3[0];
  return st;
}

// Copy one stored grid function out in the public layout.  A (stage buffer, free between steps)
// is the device staging area for host destinations.
static hr_status get_field(hr_solver* s, const void* src, void* dst, size_t bytes, int on_device) {
  if (!s || !dst) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  const size_t need = (size_t)s->g.ntot * s->scalar_bytes;
  if (bytes != need) return fail(HR_ERR_INVALID_ARG, "bytes = %zu, expected %zu", bytes, need);
  if (on_device) {
    HR_CUDA(hrk_pack(s, dst, src));
  } else {
    HR_CUDA(hrk_pack(s, s->a.A[0], src));
    HR_CUDA(cudaMemcpyAsync(dst, s->a.A[0], need, cudaMemcpyDeviceToHost, s->stream));
  }
  HR_CUDA(cudaStreamSynchronize(s->stream));
  return HR_OK;
}

hr_status hr_get_u(hr_solver* s, void* dst, size_t bytes, int32_t dst_on_device) {
  return get_field(s, s ? s->a.Y[0] : nullptr, dst, bytes, dst_on_device);
}

hr_status hr_get_v(hr_solver* s, void* dst, size_t bytes, int32_t dst_on_device) {
  return get_field(s, s ? s->a.Y[1] : nullptr, dst, bytes, dst_on_device);
}

hr_status hr_set_state(hr_solver* s, const void* u, const void* v, int32_t src_on_device) {
  if (!s || !u || !v) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  const size_t need = (size_t)s->g.ntot * s->scalar_bytes;
  if (src_on_device) {
    HR_CUDA(hrk_unpack(s, s->a.Y[0], u));
    HR_CUDA(hrk_unpack(s, s->a.Y[1], v));
  } else {
    HR_CUDA(cudaMemcpyAsync(s->a.A[0], u, need, cudaMemcpyHostToDevice, s->stream));
    HR_CUDA(cudaMemcpyAsync(s->a.A[1], v, need, cudaMemcpyHostToDevice, s->stream));
    HR_CUDA(hrk_unpack(s, s->a.Y[0], s->a.A[0]));
    HR_CUDA(hrk_unpack(s, s->a.Y[1], s->a.A[1]));
  }
  HR_CUDA(hrk_inner_fill(s, s->a.Y[0], s->a.Y[1]));
  HR_CUDA(cudaMemsetAsync(s->plan.flag, 0, sizeof(int), s->stream));  // a new state: the numeric flag starts clear
  if (!src_on_device) HR_CUDA(cudaStreamSynchronize(s->stream));
  return HR_OK;
}

hr_status hr_eval_rhs(hr_solver* s, void* ku_dev, void* kv_dev) {
  if (!s || !ku_dev || !kv_dev) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  // k is produced in the stored layout in B (free between steps), then packed out
  HR_CUDA(hrk_eval_rhs(s, s->a.B[0], s->a.B[1]));
  HR_CUDA(hrk_pack(s, ku_dev, s->a.B[0]));
  HR_CUDA(hrk_pack(s, kv_dev, s->a.B[1]));
  return HR_OK;
}

hr_status hr_get_source(hr_solver* s, void* psi_host, void* S_host) {
  if (!s) return fail(HR_ERR_INVALID_ARG, "solver is NULL");
  const size_t need = (size_t)s->g.ntot * s->scalar_bytes;
  if (psi_host) {
    HR_CUDA(hrk_pack(s, s->a.A[0], s->a.psi));
    HR_CUDA(cudaMemcpyAsync(psi_host, s->a.A[0], need, cudaMemcpyDeviceToHost, s->stream));
  }
  if (S_host) {
    HR_CUDA(hrk_pack(s, s->a.A[1], s->a.S));
    HR_CUDA(cudaMemcpyAsync(S_host, s->a.A[1], need, cudaMemcpyDeviceToHost, s->stream));
  }
  HR_CUDA(cudaStreamSynchronize(s->stream));
  return HR_OK;
}

hr_status hr_get_bc_lists(hr_solver* s, int32_t* inner_dst, int32_t* inner_src, int64_t* n_inner,
                          int32_t* outer_idx, int64_t* n_outer) {
  if (!s) return fail(HR_ERR_INVALID_ARG, "solver is NULL");
  if (n_inner) *n_inner = (int64_t)s->inner_dst.size();
  if (n_outer) *n_outer = (int64_t)s->outer_idx.size();
  if (inner_dst) memcpy(inner_dst, s->inner_dst.data(), s->inner_dst.size() * 4);
  if (inner_src) memcpy(inner_src, s->inner_src.data(), s->inner_src.size() * 4);
  if (outer_idx) memcpy(outer_idx, s->outer_idx.data(), s->outer_idx.size() * 4);
  return HR_OK;
}

hr_status hr_get_info(hr_solver* s, double* dt, double* dsmin, int32_t* nghosts, int32_t* T,
                      int64_t* total_pts) {
  if (!s) return fail(HR_ERR_INVALID_ARG, "solver is NULL");
  if (dt) *dt = s->dt;
  if (dsmin) *dsmin = s->dsmin;
  if (nghosts) *nghosts = s->g.ng;
  if (T) {
    T[0] = s->g.T0;
    T[1] = s->g.T1;
    T[2] = s->g.T2;
  }
  if (total_pts) *total_pts = s->g.ntot;
  return HR_OK;
}

hr_status hr_profile_step(hr_solver* s, int64_t n_steps, int32_t with_residual, double* ms6) {
  if (!s || !ms6) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  if (n_steps < 1 || n_steps > 4096) return fail(HR_ERR_INVALID_ARG, "n_steps must be in 1..4096");
  // one event pair per launch; elapsed times are read after a single synchronisation at the end
  const bool has_fill = hrk_launches_per_substep(s) >= 2;  // variants 1, 2: launches after the main kernel
  const int per_step = 4 + (has_fill ? 4 : 0) + (with_residual && (s->p.variant == 1 || s->p.variant == 2) ? 1 : 0);
  std::vector<cudaEvent_t> ev((size_t)n_steps * per_step * 2, nullptr);
  struct Cleanup {
    std::vector<cudaEvent_t>& ev;
    ~Cleanup() { for (cudaEvent_t e : ev) if (e) cudaEventDestroy(e); }
  } cleanup{ev};
  for (auto& e : ev) HR_CUDA(cudaEventCreate(&e));
  size_t k = 0;
  for (int64_t it = 0; it < n_steps; ++it) {
    const bool fused = with_residual && (s->p.variant == 0 || s->p.variant == 3);  // stage 1 carries it
    if (with_residual && !fused) {
      HR_CUDA(cudaEventRecord(ev[k++], s->stream));
      HR_CUDA(hrk_residual(s, s->p.residual_mode, s->a.result2));
      HR_CUDA(cudaEventRecord(ev[k++], s->stream));
    }
    for (int stage = 1; stage <= 4; ++stage) {
      HR_CUDA(cudaEventRecord(ev[k++], s->stream));
      if (fused && stage == 1) {
        HR_CUDA(hrk_fused_first(s, s->p.residual_mode, s->a.result2));
      } else {
        HR_CUDA(hrk_substep_main(s, stage));
      }
      HR_CUDA(cudaEventRecord(ev[k++], s->stream));
      if (has_fill) {
        HR_CUDA(cudaEventRecord(ev[k++], s->stream));
        HR_CUDA(hrk_substep_fill(s, stage));
        HR_CUDA(cudaEventRecord(ev[k++], s->stream));
      }
    }
  }
  HR_CUDA(cudaStreamSynchronize(s->stream));
  double acc[6] = {0, 0, 0, 0, 0, 0};
  k = 0;
  auto el = [&](size_t i, double& dst) -> cudaError_t {
    float ms = 0.f;
    cudaError_t e = cudaEventElapsedTime(&ms, ev[i], ev[i + 1]);
    dst += ms;
    return e;
  };
  const bool fused_r = with_residual && (s->p.variant == 0 || s->p.variant == 3);
  for (int64_t it = 0; it < n_steps; ++it) {
    if (with_residual && !fused_r) { HR_CUDA(el(k, acc[5])); k += 2; }
    for (int stage = 1; stage <= 4; ++stage) {
      HR_CUDA(el(k, acc[stage - 1])); k += 2;
      if (has_fill) { HR_CUDA(el(k, acc[4])); k += 2; }
    }
  }
  for (int i = 0; i < 6; ++i) ms6[i] = acc[i] / (double)n_steps;
  return HR_OK;
}

hr_status hr_query(hr_solver* s, int32_t what, int64_t* value) {
  if (!s || !value) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  switch (what) {
    case HR_Q_STEP_GRAPH: *value = s->step_graph != nullptr; return HR_OK;
    case HR_Q_RESID_GRAPH:
      *value = (s->step_resid_graph[0] ? 1 : 0) | (s->step_resid_graph[1] ? 2 : 0);
      return HR_OK;
    case HR_Q_PERSISTENT: *value = 0; return HR_OK;
    case HR_Q_NUMERIC_FLAG: {
      int* flag = reinterpret_cast<int*>(s->pinned + 6);
      HR_CUDA(cudaMemcpyAsync(flag, s->plan.flag, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
      HR_CUDA(cudaStreamSynchronize(s->stream));
      *value = *flag;
      return HR_OK;
    }
    case HR_Q_PLAN_ZC: *value = s->plan.zc; return HR_OK;
    case HR_Q_PLAN_ITEMS:  // long items (segments of plan.mseg chunks) + single chunks
      *value = s->plan.ncol + ((int64_t)s->plan.ntx * s->plan.nty * s->plan.nseg - s->plan.ncol) * s->plan.mseg;
      return HR_OK;
    case HR_Q_PLAN_GRID: *value = s->p.variant == 0 ? s->march_grid_lean[2] : s->march_grid[2]; return HR_OK;
  }
  return fail(HR_ERR_INVALID_ARG, "unknown query %d", what);
}

hr_status hr_measure_alu_peak(int32_t device, void* stream, int32_t dtype, int32_t packed, double* tflops) {
  if (!tflops || (dtype != HR_F64 && dtype != HR_F32)) return fail(HR_ERR_INVALID_ARG, "bad arguments");
  HR_CUDA(cudaSetDevice(device));
  HR_CUDA(hrk_measure_alu(static_cast<cudaStream_t>(stream), dtype, packed, tflops));
  return HR_OK;
}

hr_status hr_measure_launch_floor(int32_t device, void* stream, int32_t nodes, int32_t grid, int32_t block,
                                  int32_t reps, double* us_per_graph) {
  if (!us_per_graph || nodes < 1 || nodes > 64 || grid < 1 || block < 1 || block > 1024 || reps < 1 || !stream)
    return fail(HR_ERR_INVALID_ARG, "need 1 <= nodes <= 64, grid >= 1, 1 <= block <= 1024, reps >= 1, a non-default stream");
  HR_CUDA(cudaSetDevice(device));
  HR_CUDA(hrk_measure_launch_floor(static_cast<cudaStream_t>(stream), nodes, grid, block, reps, us_per_graph));
  return HR_OK;
}

hr_status hr_launches_per_step(hr_solver* s, int32_t* n) {
  if (!s || !n) return fail(HR_ERR_INVALID_ARG, "NULL argument");
  *n = s->launches_per_step;
  return HR_OK;
}

}  // extern "C"
