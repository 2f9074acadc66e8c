// hr_kernels.cu -- device code of the hyperbolic-relaxation hot path for sm_100a.
//
//   a0  k_source        psi_BL and S = (1/8) A~_ij A~^ij, once        (C1, C2)
//   a1  fused substep   RHS of Eq. 5 at interior points
//   a2  fused substep   radiation condition at the outer points       (C13)
//   a4  fused substep   RK4 combine (k never reaches HBM)              (C15)
//   a3  k_inner_fill    inner (parity) ghosts through the index map   (C14)
//   a5  k_residual      H and its grid L2 norm                        (C16)
//
// Product code: nothing here includes, links or calls oracle/.
#include <cuda_runtime.h>

#include <algorithm>

#include <cstdlib>
#include <mutex>
#include <type_traits>

#include "fd_tables.cuh"
#include "hr_internal.h"

namespace {

// ------------------------------------------------------------------------------------------
// arithmetic shared by the RHS and the residual
// ------------------------------------------------------------------------------------------

// 1/x for x = psi_BL + u, which is >= 1 - |u| and of order one (psi_BL > 1, C1): the hardware
// seed refined by Newton steps to full precision, without the denormal / overflow slow path a
// general division carries (two branches and a call per point).
__device__ __forceinline__ float rcp_near_one(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return fmaf(r, fmaf(-x, r, 1.0f), r);
}
__device__ __forceinline__ double rcp_near_one(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));  // ~20 good bits
  r = fma(r, fma(-x, r, 1.0), r);
  r = fma(r, fma(-x, r, 1.0), r);
  return fma(r, fma(-x, r, 1.0), r);
}

// (psi_BL + u)^-7 of Eq. 4/5: one reciprocal and four multiplies.
template <typename T>
__device__ __forceinline__ T pow_m7(T x) {
  const T t = rcp_near_one(x);
  const T t2 = t * t;
  const T t4 = t2 * t2;
  return t4 * t2 * t;
}

template <typename T>
struct StepArgs {
  const T* in_u;  // stage input (stencil source)
  const T* in_v;
  const T* y_u;  // Y (needed by stages 2, 3; stage 1 has in == Y)
  const T* y_v;
  T* out_u;  // stages 1-3: next stage input; stage 4: Y; eval mode: k_u
  T* out_v;
  T* acc_u;
  T* acc_v;
  const T* psi;
  const T* S;
  const T *L00, *L11, *L22, *L0, *L1, *C2;
  const T *RAD0, *RAD1, *RADI;
  const int32_t* OPOS;  // outer positions of the (i0,i1) plane with their stencil bits (C13)
  const T *Z22, *Z2, *ZC2, *AX;  // SinhCartesian (C25): per-plane factors and per-axis radiation tables
  int AXS;
  T eta;
  T dt;
};

// Classic RK4 (C15) in running-sum form.  STAGE 0 = "store k" (hr_eval_rhs).
//   1: out = Y + dt/2 k ; ACC  = Y + dt/6 k
//   2: out = Y + dt/2 k ; ACC += dt/3 k
//   3: out = Y + dt   k ; ACC += dt/3 k
//   4: Y   = ACC + dt/6 k
// (yu, yv) = Y and (au, av) = ACC at this point, loaded by the caller where the stage needs them;
// (wu, wv) returns what was stored to out (the value the point's ghost images take, C15).
// Arithmetic of one stage: (wu, wv) = what the stage stores to out, (nu, nv) = the new running
// sum ACC (stages 1-3).
template <typename T, int STAGE>
__device__ __forceinline__ void rk_values(T dt, T ku, T kv, T in_u, T in_v, T yu, T yv, T au, T av,
                                          T& wu, T& wv, T& nu, T& nv) {
  nu = T(0);
  nv = T(0);
  if constexpr (STAGE == 0) {
    wu = ku;
    wv = kv;
  } else if constexpr (STAGE == 1) {
    const T h = dt * T(0.5), s = dt / T(6);
    wu = in_u + h * ku;
    wv = in_v + h * kv;
    nu = in_u + s * ku;
    nv = in_v + s * kv;
  } else if constexpr (STAGE == 2 || STAGE == 3) {
    const T h = (STAGE == 2) ? dt * T(0.5) : dt;
    const T s = dt / T(3);
    wu = yu + h * ku;
    wv = yv + h * kv;
    nu = au + s * ku;
    nv = av + s * kv;
  } else {
    const T s = dt / T(6);
    wu = au + s * ku;
    wv = av + s * kv;
  }
}

template <typename T, int STAGE>
__device__ __forceinline__ void rk_combine_regs(const StepArgs<T>& a, int64_t c, T ku, T kv, T in_u,
                                                T in_v, T yu, T yv, T au, T av, T& wu, T& wv) {
  T nu, nv;
  rk_values<T, STAGE>(a.dt, ku, kv, in_u, in_v, yu, yv, au, av, wu, wv, nu, nv);
  if constexpr (STAGE >= 1 && STAGE <= 3) {
    a.acc_u[c] = nu;
    a.acc_v[c] = nv;
  }
  a.out_u[c] = wu;
  a.out_v[c] = wv;
}

template <typename T, int STAGE>
__device__ __forceinline__ void rk_combine(const StepArgs<T>& a, int64_t c, T ku, T kv, T in_u,
                                           T in_v, T& wu, T& wv) {
  T yu = T(0), yv = T(0), au = T(0), av = T(0);
  if constexpr (STAGE == 2 || STAGE == 3) {
    yu = a.y_u[c];
    yv = a.y_v[c];
  }
  if constexpr (STAGE >= 2) {
    au = a.acc_u[c];
    av = a.acc_v[c];
  }
  rk_combine_regs<T, STAGE>(a, c, ku, kv, in_u, in_v, yu, yv, au, av, wu, wv);
}

// Expanded curvilinear Laplacian (C4, C11, C12) with direct global loads of the stencil.
template <typename T, int NG>
__device__ __forceinline__ T laplacian_direct(const T* __restrict__ u, int64_t c, int64_t s1,
                                              int64_t s2, T uc, T l00, T l11, T l22, T l0, T l1) {
  using F = FdTable<NG>;
  T d00 = T(F::d2(0)) * uc, d11 = d00, d22 = d00;
  T d0 = T(0), d1 = T(0);
#pragma unroll
  for (int k = 1; k <= NG; ++k) {
    const T a0 = u[c + k], b0 = u[c - k];
    const T a1 = u[c + k * s1], b1 = u[c - k * s1];
    const T a2 = u[c + k * s2], b2 = u[c - k * s2];
    d00 += T(F::d2(k)) * (a0 + b0);
    d11 += T(F::d2(k)) * (a1 + b1);
    d22 += T(F::d2(k)) * (a2 + b2);
    d0 += T(F::c1(k)) * (a0 - b0);
    d1 += T(F::c1(k)) * (a1 - b1);
  }
  return l00 * d00 + l11 * d11 + l22 * d22 + l0 * d0 + l1 * d1;
}

// Radiation condition (C13) at an outer point c = (i0,i1,i2), j = i0 - (n0+ng):
//   k_f = -c [ rad0 (3 f_i - 4 f_{i-1} + f_{i-2})/(2 dx0) + rad1 (f_{i1+1} - f_{i1-1})/(2 dx1) + f/r ]
// Each derivative is second order: one-sided, pointing into the grid, along an axis in which the point lies
// beyond the interior (bits: 1 beyond x0 -> backward d_0; 2 beyond the high end of x1 -> backward d_1; 4 beyond
// its low end -> forward d_1), centred otherwise.  Spherical-like systems: bits = 1 at every outer point.
template <typename T>
__device__ __forceinline__ T radiation_k(const T* __restrict__ f, int64_t c, int64_t s1, T r0,
                                         T r1, T ri, int bits = 1) {
  const T fc = f[c];
  T d0, d1;
  if (bits & 1) d0 = T(3) * fc - T(4) * f[c - 1] + f[c - 2];
  else d0 = f[c + 1] - f[c - 1];
  if (bits & 2) d1 = T(3) * fc - T(4) * f[c - s1] + f[c - 2 * s1];
  else if (bits & 4) d1 = T(4) * f[c + s1] - T(3) * fc - f[c + 2 * s1];
  else d1 = f[c + s1] - f[c - s1];
  return -(r0 * d0 + r1 * d1 + ri * fc);
}

// ------------------------------------------------------------------------------------------
// a1 + a2 + a4, direct-load arrangement: one thread per point, i0 along threadIdx.x
// ------------------------------------------------------------------------------------------
constexpr int DBX = 64, DBY = 4;

template <typename T, int NG, int STAGE>
__global__ void __launch_bounds__(DBX* DBY)
    k_substep_direct(const __grid_constant__ HrGrid g, const __grid_constant__ StepArgs<T> a) {
  const int i0 = NG + blockIdx.x * DBX + threadIdx.x;
  const int i1 = NG + blockIdx.y * DBY + threadIdx.y;
  const int i2 = NG + blockIdx.z;
  if (i0 >= g.T0 || i1 >= g.n1 + NG) return;
  const int64_t c = g.off0 + i0 + g.s1 * i1 + g.s2 * i2;
  const T uc = a.in_u[c], vc = a.in_v[c];
  T ku, kv;
  if (i0 < g.n0 + NG) {
    const int64_t q = i0 + (int64_t)g.T0 * i1;
    const T lap = laplacian_direct<T, NG>(a.in_u, c, g.s1, g.s2, uc, a.L00[q], a.L11[q], a.L22[q],
                                          a.L0[q], a.L1[q]);
    ku = vc - a.eta * uc;
    kv = a.C2[q] * (lap + a.S[c] * pow_m7(a.psi[c] + uc));
  } else {
    const int qo = (i0 - (g.n0 + NG)) + NG * (i1 - NG);  // position in the outer list (HrArrays::OPOS order)
    const T r0 = a.RAD0[qo], r1 = a.RAD1[qo], ri = a.RADI[qo];
    ku = radiation_k(a.in_u, c, g.s1, r0, r1, ri);
    kv = radiation_k(a.in_v, c, g.s1, r0, r1, ri);
  }
  T wu, wv;
  rk_combine<T, STAGE>(a, c, ku, kv, uc, vc, wu, wv);
}

// ------------------------------------------------------------------------------------------
// Variant 1, the paper's arrangement as an ablation: one thread
// per point with block (32, NGHOSTS, 1), no shared memory, RHS -> BC -> RK as separate kernels
// with k stored in HBM (buffer B) and re-read by the RK kernel.  (The reference-metric factors
// still come from the (i0,i1) planes; the paper evaluates CSE'd expressions instead.)
// ------------------------------------------------------------------------------------------
template <typename T, int NG>
__global__ void __launch_bounds__(32 * NG)
    k_paper_rhs(const __grid_constant__ HrGrid g, const __grid_constant__ StepArgs<T> a) {
  const int i0 = NG + blockIdx.x * 32 + threadIdx.x;
  const int i1 = NG + blockIdx.y * NG + threadIdx.y;
  const int i2 = NG + blockIdx.z;
  if (i0 >= g.n0 + NG || i1 >= g.n1 + NG) return;
  const int64_t c = g.off0 + i0 + g.s1 * i1 + g.s2 * i2;
  const int64_t q = i0 + (int64_t)g.T0 * i1;
  const T uc = a.in_u[c], vc = a.in_v[c];
  const T lap = laplacian_direct<T, NG>(a.in_u, c, g.s1, g.s2, uc, a.L00[q], a.L11[q], a.L22[q],
                                        a.L0[q], a.L1[q]);
  a.out_u[c] = vc - a.eta * uc;
  a.out_v[c] = a.C2[q] * (lap + a.S[c] * pow_m7(a.psi[c] + uc));
}

template <typename T, int NG>
__global__ void __launch_bounds__(256)
    k_paper_bc_outer(const __grid_constant__ HrGrid g, const __grid_constant__ StepArgs<T> a) {
  const int m = blockIdx.x * 256 + threadIdx.x;
  if (m >= NG * g.n1 * g.n2) return;
  const int j = m % NG;
  const int r = m / NG;
  const int i1 = NG + r % g.n1, i2 = NG + r / g.n1;
  const int64_t c = g.off0 + (g.n0 + NG + j) + g.s1 * i1 + g.s2 * i2;
  const int qo = j + NG * (i1 - NG);  // position in the outer list (HrArrays::OPOS order)
  const T r0 = a.RAD0[qo], r1 = a.RAD1[qo], ri = a.RADI[qo];
  a.out_u[c] = radiation_k(a.in_u, c, g.s1, r0, r1, ri);
  a.out_v[c] = radiation_k(a.in_v, c, g.s1, r0, r1, ri);
}

// RK combine over all stored points (ghosts included, as Alg. 1 l.15 has it): k = (ku, kv) from
// HBM; stage 1-3 write the next stage state (in place in A) and the running sum, stage 4 writes Y.
template <typename T, int STAGE>
__global__ void __launch_bounds__(256)
    k_paper_rk(int64_t n, T dt, const T* __restrict__ ku, const T* __restrict__ kv,
               T* __restrict__ y_u, T* __restrict__ y_v, T* __restrict__ st_u,
               T* __restrict__ st_v, T* __restrict__ acc_u, T* __restrict__ acc_v) {
  const int64_t c = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (c >= n) return;
  T yu = T(0), yv = T(0), au = T(0), av = T(0);
  if constexpr (STAGE <= 3) {
    yu = y_u[c];
    yv = y_v[c];
  }
  if constexpr (STAGE >= 2) {
    au = acc_u[c];
    av = acc_v[c];
  }
  T wu, wv, nu, nv;
  rk_values<T, STAGE>(dt, ku[c], kv[c], yu, yv, yu, yv, au, av, wu, wv, nu, nv);
  if constexpr (STAGE <= 3) {
    st_u[c] = wu;
    st_v[c] = wv;
    acc_u[c] = nu;
    acc_v[c] = nv;
  } else {
    y_u[c] = wu;
    y_v[c] = wv;
  }
}

// ------------------------------------------------------------------------------------------
// a3: inner ghosts through the precomputed index map (C14), parity +1
// ------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
    k_inner_fill(T* __restrict__ fu, T* __restrict__ fv, const int32_t* __restrict__ dst,
                 const int32_t* __restrict__ src, int64_t n) {
  const int64_t m = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n) return;
  const int32_t d = dst[m], s = src[m];
  fu[d] = fu[s];
  if (fv) fv[d] = fv[s];
}

// ------------------------------------------------------------------------------------------
// a5: H at interior points, weighted squares reduced warp -> block -> one partial per block
// ------------------------------------------------------------------------------------------
constexpr int RBX = 64, RBY = 4;

template <typename T, int NG>
__global__ void __launch_bounds__(RBX* RBY)
    k_residual(const __grid_constant__ HrGrid g, const T* __restrict__ u,
               const T* __restrict__ psi, const T* __restrict__ S, const T* __restrict__ L00,
               const T* __restrict__ L11, const T* __restrict__ L22, const T* __restrict__ L0,
               const T* __restrict__ L1, const double* __restrict__ W, int mode,
               double* __restrict__ partials) {
  const int i0 = NG + blockIdx.x * RBX + threadIdx.x;
  const int i1 = NG + blockIdx.y * RBY + threadIdx.y;
  const int i2 = NG + blockIdx.z;
  double num = 0.0, den = 0.0;
  if (i0 < g.n0 + NG && i1 < g.n1 + NG) {
    const int64_t c = g.off0 + i0 + g.s1 * i1 + g.s2 * i2;
    const int64_t q = i0 + (int64_t)g.T0 * i1;
    const T uc = u[c];
    const T lap =
        laplacian_direct<T, NG>(u, c, g.s1, g.s2, uc, L00[q], L11[q], L22[q], L0[q], L1[q]);
    const T H = lap + S[c] * pow_m7(psi[c] + uc);
    const double w = (mode == 0) ? W[q] : 1.0;
    num = w * (double)H * (double)H;
    den = w;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    num += __shfl_down_sync(0xffffffffu, num, o);
    den += __shfl_down_sync(0xffffffffu, den, o);
  }
  __shared__ double sh[2][RBX * RBY / 32];
  const int tid = threadIdx.y * RBX + threadIdx.x;
  if ((tid & 31) == 0) {
    sh[0][tid >> 5] = num;
    sh[1][tid >> 5] = den;
  }
  __syncthreads();
  if (tid == 0) {
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int w = 0; w < RBX * RBY / 32; ++w) {
      a += sh[0][w];
      b += sh[1][w];
    }
    const int64_t bid = blockIdx.x + (int64_t)gridDim.x * (blockIdx.y + (int64_t)gridDim.y * blockIdx.z);
    partials[2 * bid] = a;
    partials[2 * bid + 1] = b;
  }
}

// Final pass: one block, fixed order (thread t sums partials t, t+1024, ...; then a tree).
__global__ void __launch_bounds__(1024)
    k_residual_final(const double* __restrict__ partials, int64_t nblocks, double* __restrict__ out2) {
  __shared__ double sh[2][1024];
  double a = 0.0, b = 0.0;
  for (int64_t i = threadIdx.x; i < nblocks; i += 1024) {
    a += partials[2 * i];
    b += partials[2 * i + 1];
  }
  sh[0][threadIdx.x] = a;
  sh[1][threadIdx.x] = b;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      sh[0][threadIdx.x] += sh[0][threadIdx.x + o];
      sh[1][threadIdx.x] += sh[1][threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    out2[0] = sh[0][0];
    out2[1] = sh[1][0];
  }
}

// ------------------------------------------------------------------------------------------
// a0: constant source terms, fp64 arithmetic, stored in the working precision (C1, C2, C19)
// ------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
    k_source(const __grid_constant__ HrGrid g, const double* __restrict__ rho,
             const double* __restrict__ rhoz, const double* __restrict__ sinth,
             const double* __restrict__ costh, const double* __restrict__ sinph,
             const double* __restrict__ cosph, const double* __restrict__ punct, int npunct,
             double ox, double oy, double oz, T* __restrict__ psi_out, T* __restrict__ S_out,
             int* __restrict__ bad_flag, int cart) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.ntot) return;
  const int i0 = (int)(c % g.T0);
  const int i1 = (int)((c / g.T0) % g.T1);
  const int i2 = (int)(c / ((int64_t)g.T0 * g.T1));
  const int64_t cs = g.off0 + i0 + g.s1 * i1 + g.s2 * i2;  // stored index
  // grid point in Cartesian coordinates (C4) + grid centre (C6)
  const double rs = rho[i0] * sinth[i1];
  // (C25, SinhCartesian: the three tables hold X0(i0), X1(i1), X2(i2))
  const double x = (cart ? rho[i0] : rs * cosph[i2]) + ox;
  const double y = (cart ? costh[i1] : rs * sinph[i2]) + oy;
  const double z = (cart ? cosph[i2] : rhoz[i0] * costh[i1]) + oz;
  double psi = 1.0;
  double axx = 0, ayy = 0, azz = 0, axy = 0, axz = 0, ayz = 0;
  for (int p = 0; p < npunct; ++p) {
    const double* pp = punct + 10 * p;
    const double m = pp[0];
    const double dx = x - pp[1], dy = y - pp[2], dz = z - pp[3];
    const double Px = pp[4], Py = pp[5], Pz = pp[6];
    const double Sx = pp[7], Sy = pp[8], Sz = pp[9];
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double r = sqrt(r2);
    const double ir = 1.0 / r;
    psi += 0.5 * m * ir;  // Brandt-Bruegmann psi_BL = 1 + sum m/(2r)
    const double nx = dx * ir, ny = dy * ir, nz = dz * ir;
    const double Pn = Px * nx + Py * ny + Pz * nz;
    // (S x n)
    const double cx = Sy * nz - Sz * ny, cy = Sz * nx - Sx * nz, cz = Sx * ny - Sy * nx;
    const double fP = 1.5 * ir * ir;       // 3 / (2 r^2)
    const double fS = 3.0 * ir * ir * ir;  // 3 / r^3
    // Bowen-York: fP [P^i n^j + P^j n^i - (delta^ij - n^i n^j) P.n] + fS [(Sxn)^i n^j + (Sxn)^j n^i]
    axx += fP * (2.0 * Px * nx - (1.0 - nx * nx) * Pn) + fS * (2.0 * cx * nx);
    ayy += fP * (2.0 * Py * ny - (1.0 - ny * ny) * Pn) + fS * (2.0 * cy * ny);
    azz += fP * (2.0 * Pz * nz - (1.0 - nz * nz) * Pn) + fS * (2.0 * cz * nz);
    axy += fP * (Px * ny + Py * nx + nx * ny * Pn) + fS * (cx * ny + cy * nx);
    axz += fP * (Px * nz + Pz * nx + nx * nz * Pn) + fS * (cx * nz + cz * nx);
    ayz += fP * (Py * nz + Pz * ny + ny * nz * Pn) + fS * (cy * nz + cz * ny);
  }
  const double AA = axx * axx + ayy * ayy + azz * azz + 2.0 * (axy * axy + axz * axz + ayz * ayz);
  const double Sval = 0.125 * AA;
  if (!isfinite(psi) || !isfinite(Sval)) atomicOr(bad_flag, 1);
  psi_out[cs] = (T)psi;
  S_out[cs] = (T)Sval;
}

// ------------------------------------------------------------------------------------------
// public layout <-> stored (padded) layout
// ------------------------------------------------------------------------------------------
template <typename T, bool TO_PUBLIC>
__global__ void __launch_bounds__(256)
    k_repack(const __grid_constant__ HrGrid g, T* __restrict__ dst, const T* __restrict__ src) {
  const int i0 = blockIdx.y * 256 + threadIdx.x;
  if (i0 >= g.T0) return;
  const int64_t row = blockIdx.x;  // i1 + T1 i2
  const int64_t pub = i0 + (int64_t)g.T0 * row;
  const int64_t sto = g.off0 + i0 + g.s1 * row;
  if (TO_PUBLIC)
    dst[pub] = src[sto];
  else
    dst[sto] = src[pub];
}


#include "hr_march.cuh"

// ------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------
template <typename T>
StepArgs<T> make_args(const hr_solver* s, int stage, void* ku, void* kv) {
  const HrArrays& a = s->a;
  StepArgs<T> r{};
  auto P = [](void* p) { return static_cast<T*>(p); };
  switch (stage) {
    case 0:  // eval: in = Y, out = k
      r.in_u = P(a.Y[0]); r.in_v = P(a.Y[1]); r.out_u = P(ku); r.out_v = P(kv);
      break;
    case 1:
    case 6:  // stage 1 fused with the residual of its input state
      r.in_u = P(a.Y[0]); r.in_v = P(a.Y[1]); r.out_u = P(a.A[0]); r.out_v = P(a.A[1]);
      break;
    case 2:
      r.in_u = P(a.A[0]); r.in_v = P(a.A[1]); r.out_u = P(a.B[0]); r.out_v = P(a.B[1]);
      break;
    case 3:
      r.in_u = P(a.B[0]); r.in_v = P(a.B[1]); r.out_u = P(a.A[0]); r.out_v = P(a.A[1]);
      break;
    case 4:
      r.in_u = P(a.A[0]); r.in_v = P(a.A[1]); r.out_u = P(a.Y[0]); r.out_v = P(a.Y[1]);
      break;
    case 11:
    case 16:  // lean: Y -> Y1 (A)
      r.in_u = P(a.Y[0]); r.in_v = P(a.Y[1]); r.out_u = P(a.A[0]); r.out_v = P(a.A[1]);
      break;
    case 12:
    case 22:  // lean: Y1 (A) -> Y2 (B)
      r.in_u = P(a.A[0]); r.in_v = P(a.A[1]); r.out_u = P(a.B[0]); r.out_v = P(a.B[1]);
      break;
    case 13:  // lean: Y2 (B) -> Y3 (A again: Y1 is no longer needed)
      r.in_u = P(a.B[0]); r.in_v = P(a.B[1]); r.out_u = P(a.A[0]); r.out_v = P(a.A[1]);
      break;
    case 14:
    case 24:  // lean: Y3 (A) -> Y, reading Q (the ACC buffer); 24 also reads Y
      r.in_u = P(a.A[0]); r.in_v = P(a.A[1]); r.out_u = P(a.Y[0]); r.out_v = P(a.Y[1]);
      break;
    default:  // 5, residual: the stencil source is the state
      r.in_u = P(a.Y[0]); r.in_v = P(a.Y[1]);
      break;
  }
  r.y_u = P(a.Y[0]); r.y_v = P(a.Y[1]);
  r.acc_u = P(a.ACC[0]); r.acc_v = P(a.ACC[1]);
  if (stage == 14) {  // Q rides in the Y slots (stage 24 keeps Y there and reads Qd from the ACC slots)
    r.y_u = P(a.ACC[0]); r.y_v = P(a.ACC[1]);
  }
  r.psi = P(a.psi); r.S = P(a.S);
  r.L00 = P(a.L00); r.L11 = P(a.L11); r.L22 = P(a.L22); r.L0 = P(a.L0); r.L1 = P(a.L1);
  r.C2 = P(a.C2); r.RAD0 = P(a.RAD0); r.RAD1 = P(a.RAD1); r.RADI = P(a.RADI);
  r.OPOS = a.OPOS;
  r.Z22 = P(a.Z22); r.Z2 = P(a.Z2); r.ZC2 = P(a.ZC2); r.AX = P(a.AX); r.AXS = a.AXS;
  r.eta = (T)s->p.eta;
  r.dt = (T)s->dt;
  return r;
}

// ---- direct-load arrangement (variant 2) ----
template <typename T, int NG>
cudaError_t launch_substep_direct(const hr_solver* s, int stage, void* ku, void* kv) {
  const HrGrid& g = s->g;
  const StepArgs<T> a = make_args<T>(s, stage, ku, kv);
  const dim3 block(DBX, DBY, 1);
  const dim3 grid((g.n0 + NG + DBX - 1) / DBX, (g.n1 + DBY - 1) / DBY, g.n2);
  switch (stage) {
    case 0: k_substep_direct<T, NG, 0><<<grid, block, 0, s->stream>>>(g, a); break;
    case 1: k_substep_direct<T, NG, 1><<<grid, block, 0, s->stream>>>(g, a); break;
    case 2: k_substep_direct<T, NG, 2><<<grid, block, 0, s->stream>>>(g, a); break;
    case 3: k_substep_direct<T, NG, 3><<<grid, block, 0, s->stream>>>(g, a); break;
    default: k_substep_direct<T, NG, 4><<<grid, block, 0, s->stream>>>(g, a); break;
  }
  return cudaGetLastError();
}

// ---- paper arrangement (variant 1) ----
// stage s: k = RHS(in) into B (in = Y for stage 1, else the stage state A); (ku, kv) given for eval
template <typename T>
StepArgs<T> make_args_paper(const hr_solver* s, int stage, void* ku, void* kv) {
  StepArgs<T> r = make_args<T>(s, 0, ku ? ku : s->a.B[0], kv ? kv : s->a.B[1]);
  if (stage >= 2) {
    r.in_u = static_cast<T*>(s->a.A[0]);
    r.in_v = static_cast<T*>(s->a.A[1]);
  }
  return r;
}

template <typename T, int NG>
cudaError_t launch_paper_rhs(const hr_solver* s, int stage, void* ku, void* kv) {
  const HrGrid& g = s->g;
  const StepArgs<T> a = make_args_paper<T>(s, stage, ku, kv);
  const dim3 block(32, NG, 1);
  const dim3 grid((g.n0 + 31) / 32, (g.n1 + NG - 1) / NG, g.n2);
  k_paper_rhs<T, NG><<<grid, block, 0, s->stream>>>(g, a);
  return cudaGetLastError();
}

template <typename T, int NG>
cudaError_t launch_paper_bc_outer(const hr_solver* s, int stage, void* ku, void* kv) {
  const HrGrid& g = s->g;
  const StepArgs<T> a = make_args_paper<T>(s, stage, ku, kv);
  const int n = NG * g.n1 * g.n2;
  k_paper_bc_outer<T, NG><<<(n + 255) / 256, 256, 0, s->stream>>>(g, a);
  return cudaGetLastError();
}

template <typename T>
cudaError_t launch_paper_rk(const hr_solver* s, int stage) {
  const HrArrays& a = s->a;
  auto P = [](void* p) { return static_cast<T*>(p); };
  const int64_t n = s->g.npad;
  const int blocks = (int)((n + 255) / 256);
  const T dt = (T)s->dt;
#define HR_RK(ST)                                                                                \
  k_paper_rk<T, ST><<<blocks, 256, 0, s->stream>>>(n, dt, P(a.B[0]), P(a.B[1]), P(a.Y[0]),      \
                                                    P(a.Y[1]), P(a.A[0]), P(a.A[1]), P(a.ACC[0]), \
                                                    P(a.ACC[1]))
  switch (stage) {
    case 1: HR_RK(1); break;
    case 2: HR_RK(2); break;
    case 3: HR_RK(3); break;
    default: HR_RK(4); break;
  }
#undef HR_RK
  return cudaGetLastError();
}

template <typename T>
cudaError_t dispatch_paper(const hr_solver* s, int what, int stage, void* ku, void* kv) {
#define HR_NGCASE(N)                                                          \
  case N:                                                                     \
    return what == 0 ? launch_paper_rhs<T, N>(s, stage, ku, kv)               \
                     : launch_paper_bc_outer<T, N>(s, stage, ku, kv);
  switch (s->g.ng) {
    HR_NGCASE(1) HR_NGCASE(2) HR_NGCASE(3) HR_NGCASE(4) HR_NGCASE(5) HR_NGCASE(6)
  }
#undef HR_NGCASE
  return cudaErrorInvalidValue;
}

// ---- marching arrangement (variant 0: ACC-free RK4; variant 3: running-sum RK4) ----
// Tile shape per dtype: TW x BY points, VX points per thread (16-byte vectors along i0 are
// double2 / float4; fp64 keeps one point per thread for register room), D planes of look-ahead.
template <typename T>
struct MarchCfg;
template <>
struct MarchCfg<double> {
  static constexpr int TW = HR_TW_F64, BY = HR_BY_F64, VX = HR_VX_F64, D = HR_MARCH_D_F64;
};
template <>
struct MarchCfg<float> {
  static constexpr int TW = HR_TW_F32, BY = HR_BY_F32, VX = HR_VX_F32, D = HR_MARCH_D_F32;
};

// Planes of look-ahead.  D = 2 everywhere by default (D = 1: -7 %).  HR_MARCH_D_EXTRA_LIGHT adds
// planes for the fp64 kernels other than the heaviest: with the running-sum arrangement
// (variant 3) one more plane gained 1-3 % on the 8 w kernels; with the default arrangement, whose
// kernels are all bound by the plane loop, it costs 1 % (shared memory -> occupancy), so it is 0.
template <typename T, int STAGE>
constexpr int march_depth() {
  // (the heavy kernels: stages 2, 3 of the running-sum form, 12 w; stage 2 = code 12 of the
  // ACC-free form, 10 w)
  return MarchCfg<T>::D +
         ((STAGE == 2 || STAGE == 3 || STAGE == 12 || sizeof(T) != 8) ? 0 : HR_MARCH_D_EXTRA_LIGHT);
}

// Stage codes of the default arrangement's stages 2 and 4 per dtype: fp32 takes the increment-preserving
// forms 22 / 24 (hr_march.cuh: rk_prec_q, rk_prec_4), fp64 the plain ACC-free forms 12 / 14.
template <typename T>
struct LeanCode {
  static constexpr bool PREC = sizeof(T) == 4 && HR_F32_PRECISE_RK;
  static constexpr int S2 = PREC ? 22 : 12, S4 = PREC ? 24 : 14;
};

#define HR_MARCH_KERNEL(T, NG, STAGE, CART) \
  k_march<T, NG, STAGE, MarchCfg<T>::TW, MarchCfg<T>::BY, MarchCfg<T>::VX, march_depth<T, STAGE>(), CART>
#define HR_MARCH_SMEM(T, NG, STAGE) \
  march_smem_bytes<T, NG, STAGE, MarchCfg<T>::TW, MarchCfg<T>::BY, march_depth<T, STAGE>()>()

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

cudaError_t encode_box(const hr_solver* s, CUtensorMap* map, void* base, int bw, int bh) {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q);
    if (e != cudaSuccess) return e;
    if (!p || q != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  const HrGrid& g = s->g;
  const cuuint64_t w = s->scalar_bytes;
  const cuuint64_t dims[3] = {(cuuint64_t)g.P0, (cuuint64_t)g.T1, (cuuint64_t)g.T2};
  const cuuint64_t strides[2] = {(cuuint64_t)g.P0 * w, (cuuint64_t)g.P0 * g.T1 * w};
  const cuuint32_t box[3] = {(cuuint32_t)bw, (cuuint32_t)bh, 1u};
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  const CUresult r = fn(map, w == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                        3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

// Planes per chunk.  Work items = tiles x chunks are handed out dynamically to `slots` persistent
// CTAs.  Measured on config 3 and on configs[4]'s sweep grids (profiles/r1c.md): chunks of 6-10
// planes are best or within 1-2 % of best everywhere -- short items keep the hand-out balanced and
// neighbouring tiles in step, and priming an item's 2NG-plane window costs about one plane --
// while 32-64 planes lose up to 30 %.  So: 8 planes, shorter (down to 2) only while the grid
// has fewer items than CTA slots (small grids, latency regime), evened out over n2.
static void choose_chunks(MarchPlan& m, int n2, int ng, int slots, bool f64) {
  (void)ng;
  const char* zc_env = std::getenv("HR_TUNE_ZC");  // tuning knob: planes per chunk
  int zc = 8;
  if (zc_env && std::atoi(zc_env) > 0) {
    zc = std::atoi(zc_env);
  } else {
    const long long ntiles = (long long)m.ntx * m.nty;
    // fp64 with plenty of items (>= 4 rounds): 12 planes amortise the window priming better
    // (config 3: +1.5 %, 512x256x256: +3 %; on 128^3 8 planes stay ahead)
    if (f64 && ntiles * ((n2 + 11) / 12) >= 4LL * slots) zc = 12;
    if (ntiles * ((n2 + 7) / 8) < 4LL * slots) {
      // Few waves of CTAs (L2-resident grids): a launch lasts waves x (planes per item + ~2 planes to prime the
      // window and start the pipeline), each plane a ~1.2 us latency chain, so the item length is chosen to
      // minimise that -- in particular never "just over one wave".  Ties go to the shorter item.  (Measured,
      // config 2: fp64 4 planes 79.5 us per step against 84.6 at 8; config 0 / 1: 1 / 2 planes, one wave;
      // the table of 16 grid / dtype cases x 7 lengths is in profiles/r2b.md.)
      long long best = -1;
      for (int c = 1; c <= 16 && c <= n2; ++c) {
        const int nz = (n2 + c - 1) / c, ce = (n2 + nz - 1) / nz;
        const long long waves = (ntiles * nz + slots - 1) / slots;
        // one wave of LONG items leaves the SMs with 3-4 CTAs each running a long serial chain: measured 12-14 %
        // behind two waves of shorter items (config 2 fp32: 7 planes 72.1 us against 3 planes 63.1; 256x128x64 fp32:
        // 13 planes 108 us against 6 planes 93), so a single wave is only taken with items of <= 4 planes
        if (waves == 1 && ce > 4) continue;
        const long long cost = waves * (ce + 2);
        if (best < 0 || cost < best) {
          best = cost;
          zc = c;
        }
      }
    }
  }
  if (zc > n2) zc = n2;
  m.nzc = (n2 + zc - 1) / zc;
  m.zc = (n2 + m.nzc - 1) / m.nzc;
  m.gt = m.ntx * m.nty;  // (round 1's groups of tile rows are gone: long items took over their job)
}

// Persistent grid of one stage's kernel: resident CTAs per SM x SMs (never more than the work).
template <typename T, int NG, int STAGE>
cudaError_t prepare_march_stage(const hr_solver* s, int* grid_out) {
  using C = MarchCfg<T>;
  auto kern = s->plan.cart ? HR_MARCH_KERNEL(T, NG, STAGE, true) : HR_MARCH_KERNEL(T, NG, STAGE, false);
  constexpr size_t smem = HR_MARCH_SMEM(T, NG, STAGE);
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, (C::TW / C::VX) * C::BY, smem);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) return cudaErrorLaunchOutOfResources;
  *grid_out = per_sm * s->num_sms;
  return cudaSuccess;
}

template <typename T, int NG>
cudaError_t prepare_march(hr_solver* s) {
  using C = MarchCfg<T>;
  using G = MarchGeom<T, NG, C::TW, C::BY>;
  cudaError_t e;
  const HrArrays& a = s->a;
  void* fields[10] = {a.Y[0], a.Y[1], a.A[0], a.A[1], a.B[0], a.B[1], a.ACC[0], a.ACC[1], a.psi, a.S};
  for (int f = 0; f < 10; ++f)
    if ((e = encode_box(s, &s->tm_box[f], fields[f], C::TW, C::BY)) != cudaSuccess) return e;
  for (int f = 0; f < 3; ++f)  // stencil sources: Y_u, A_u, B_u
    if ((e = encode_box(s, &s->tm_tile[f], fields[2 * f], G::SWA, G::SH)) != cudaSuccess) return e;
  if ((e = prepare_march_stage<T, NG, 0>(s, &s->march_grid[0])) != cudaSuccess) return e;
  if ((e = prepare_march_stage<T, NG, 1>(s, &s->march_grid[1])) != cudaSuccess) return e;
  if ((e = prepare_march_stage<T, NG, 2>(s, &s->march_grid[2])) != cudaSuccess) return e;
  if ((e = prepare_march_stage<T, NG, 3>(s, &s->march_grid[3])) != cudaSuccess) return e;
  if ((e = prepare_march_stage<T, NG, 4>(s, &s->march_grid[4])) != cudaSuccess) return e;
  if ((e = prepare_march_stage<T, NG, 5>(s, &s->march_grid[5])) != cudaSuccess) return e;
  if ((e = prepare_march_stage<T, NG, 6>(s, &s->march_grid[6])) != cudaSuccess) return e;
  if (s->p.variant == 0) {  // the ACC-free arrangement's kernels, grid sizes indexed by stage % 10
    if ((e = prepare_march_stage<T, NG, 11>(s, &s->march_grid_lean[1])) != cudaSuccess) return e;
    if ((e = prepare_march_stage<T, NG, LeanCode<T>::S2>(s, &s->march_grid_lean[2])) != cudaSuccess) return e;
    if ((e = prepare_march_stage<T, NG, 13>(s, &s->march_grid_lean[3])) != cudaSuccess) return e;
    if ((e = prepare_march_stage<T, NG, LeanCode<T>::S4>(s, &s->march_grid_lean[4])) != cudaSuccess) return e;
    if ((e = prepare_march_stage<T, NG, 16>(s, &s->march_grid_lean[6])) != cudaSuccess) return e;
  }
  for (int st = 0; st < 7; ++st) {
    s->march_slots[st] = s->march_grid[st];
    s->march_slots_lean[st] = s->march_grid_lean[st];
  }
  hrk_replan(s, 1);
  return cudaSuccess;
}

template <typename T>
cudaError_t prepare_march_ng(hr_solver* s) {
  switch (s->g.ng) {
    case 1: return prepare_march<T, 1>(s);
    case 2: return prepare_march<T, 2>(s);
    case 3: return prepare_march<T, 3>(s);
    case 4: return prepare_march<T, 4>(s);
    case 5: return prepare_march<T, 5>(s);
    case 6: return prepare_march<T, 6>(s);
  }
  return cudaErrorInvalidValue;
}

// Tensor maps of one stage: stencil source = Y (stages 0, 1, residual), A (2, 4), B (3).
MarchMaps make_maps(const hr_solver* s, int stage) {
  MarchMaps m;
  if (stage >= 10) {  // lean: front psi S v | Y (stages 2, 3) or Q = ACC (stage 4) | Y; sources Y, A, B, A
    const int st = stage % 10;
    const int in = (st == 2 || st == 4) ? 1 : (st == 3 ? 2 : 0);
    const int ys = st == 4 ? 6 : 0;
    m.tile = s->tm_tile[in];
    m.st[0] = s->tm_box[2 * in];
    m.st[1] = s->tm_box[8];
    m.st[2] = s->tm_box[9];
    m.st[3] = s->tm_box[2 * in + 1];
    m.st[4] = s->tm_box[ys];
    m.st[5] = s->tm_box[ys + 1];
    m.st[6] = s->tm_box[0];
    m.st[7] = s->tm_box[1];
    return m;
  }
  const int in = (stage == 2 || stage == 4) ? 1 : (stage == 3 ? 2 : 0);  // 0, 1, 5, 6: Y
  m.tile = s->tm_tile[in];
  m.st[ST_FRONT] = s->tm_box[2 * in];
  m.st[ST_V] = s->tm_box[2 * in + 1];
  m.st[ST_PSI] = s->tm_box[8];
  m.st[ST_S] = s->tm_box[9];
  m.st[ST_AU] = s->tm_box[6];
  m.st[ST_AV] = s->tm_box[7];
  m.st[ST_YU] = s->tm_box[0];
  m.st[ST_YV] = s->tm_box[1];
  return m;
}

template <typename T, int NG, int STAGE>
cudaError_t launch_march_stage(const hr_solver* s, const StepArgs<T>& a, const ResidArgs& ra) {
  using C = MarchCfg<T>;
  constexpr size_t smem = HR_MARCH_SMEM(T, NG, STAGE);
  const dim3 block(C::TW / C::VX, C::BY, 1);
  const dim3 grid(STAGE >= 10 ? s->march_grid_lean[STAGE % 10] : s->march_grid[STAGE], 1, 1);
  const MarchMaps mm = make_maps(s, STAGE);
  // Programmatic dependent launch: the kernel signals launch_dependents at once and waits (griddepcontrol.wait)
  // before it touches anything its predecessor wrote, so the launch latency, CTA start-up and barrier set-up of
  // substep s + 1 overlap the end of substep s (on L2-resident grids ~1 us of a 5-7 us launch).
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = HR_MARCH_PDL;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (s->plan.cart)
    return cudaLaunchKernelEx(&cfg, HR_MARCH_KERNEL(T, NG, STAGE, true), s->g, a, s->plan, ra, mm);
  return cudaLaunchKernelEx(&cfg, HR_MARCH_KERNEL(T, NG, STAGE, false), s->g, a, s->plan, ra, mm);
}

template <typename T, int NG>
cudaError_t launch_march(const hr_solver* s, int stage, void* ku, void* kv, int mode,
                         double* partials, double* out2 = nullptr) {
  if (stage == 12) stage = LeanCode<T>::S2;
  if (stage == 14) stage = LeanCode<T>::S4;
  const StepArgs<T> a = make_args<T>(s, stage, ku, kv);
  const ResidArgs ra{s->a.Wvol, partials, mode, out2, s->a.ZH};
  switch (stage) {
    case 0: return launch_march_stage<T, NG, 0>(s, a, ra);
    case 1: return launch_march_stage<T, NG, 1>(s, a, ra);
    case 2: return launch_march_stage<T, NG, 2>(s, a, ra);
    case 3: return launch_march_stage<T, NG, 3>(s, a, ra);
    case 4: return launch_march_stage<T, NG, 4>(s, a, ra);
    case 6: return launch_march_stage<T, NG, 6>(s, a, ra);
    case 11: return launch_march_stage<T, NG, 11>(s, a, ra);
    case 12:
    case 22: return launch_march_stage<T, NG, LeanCode<T>::S2>(s, a, ra);
    case 13: return launch_march_stage<T, NG, 13>(s, a, ra);
    case 14:
    case 24: return launch_march_stage<T, NG, LeanCode<T>::S4>(s, a, ra);
    case 16: return launch_march_stage<T, NG, 16>(s, a, ra);
    default: return launch_march_stage<T, NG, 5>(s, a, ra);
  }
}

template <typename T>
cudaError_t dispatch_substep(const hr_solver* s, int stage, void* ku, void* kv) {
  if (s->p.variant == 2) {
    switch (s->g.ng) {
      case 1: return launch_substep_direct<T, 1>(s, stage, ku, kv);
      case 2: return launch_substep_direct<T, 2>(s, stage, ku, kv);
      case 3: return launch_substep_direct<T, 3>(s, stage, ku, kv);
      case 4: return launch_substep_direct<T, 4>(s, stage, ku, kv);
      case 5: return launch_substep_direct<T, 5>(s, stage, ku, kv);
      case 6: return launch_substep_direct<T, 6>(s, stage, ku, kv);
    }
    return cudaErrorInvalidValue;
  }
  if (s->p.variant == 0 && stage >= 1 && stage <= 4) stage += 10;  // the ACC-free arrangement
  switch (s->g.ng) {
    case 1: return launch_march<T, 1>(s, stage, ku, kv, 0, nullptr);
    case 2: return launch_march<T, 2>(s, stage, ku, kv, 0, nullptr);
    case 3: return launch_march<T, 3>(s, stage, ku, kv, 0, nullptr);
    case 4: return launch_march<T, 4>(s, stage, ku, kv, 0, nullptr);
    case 5: return launch_march<T, 5>(s, stage, ku, kv, 0, nullptr);
    case 6: return launch_march<T, 6>(s, stage, ku, kv, 0, nullptr);
  }
  return cudaErrorInvalidValue;
}

template <typename T>
cudaError_t inner_fill_t(const hr_solver* s, void* fu, void* fv) {
  const int64_t n = s->g.n_inner;
  if (n == 0) return cudaSuccess;
  const int blocks = (int)((n + 255) / 256);
  k_inner_fill<T><<<blocks, 256, 0, s->stream>>>(static_cast<T*>(fu), static_cast<T*>(fv),
                                                  s->a.inner_dst, s->a.inner_src, n);
  return cudaGetLastError();
}

template <typename T, int NG>
cudaError_t launch_residual(const hr_solver* s, int mode, double* out2) {
  const HrGrid& g = s->g;
  const HrArrays& a = s->a;
  int64_t nb;
  cudaError_t e;
  if (s->p.variant == 1 || s->p.variant == 2) {
    auto P = [](void* p) { return static_cast<const T*>(p); };
    const dim3 block(RBX, RBY, 1);
    const dim3 grid((g.n0 + RBX - 1) / RBX, (g.n1 + RBY - 1) / RBY, g.n2);
    k_residual<T, NG><<<grid, block, 0, s->stream>>>(g, P(a.Y[0]), P(a.psi), P(a.S), P(a.L00),
                                                      P(a.L11), P(a.L22), P(a.L0), P(a.L1), a.Wvol,
                                                      mode, a.partials);
    e = cudaGetLastError();
    nb = (int64_t)grid.x * grid.y * grid.z;
  } else {
    // one partial pair per work item; the last CTA to finish sums them into out2
    return launch_march<T, NG>(s, 5, nullptr, nullptr, mode, a.partials, out2);
  }
  if (e != cudaSuccess) return e;
  k_residual_final<<<1, 1024, 0, s->stream>>>(a.partials, nb, out2);
  return cudaGetLastError();
}

template <typename T>
cudaError_t dispatch_residual(const hr_solver* s, int mode, double* out2) {
  switch (s->g.ng) {
    case 1: return launch_residual<T, 1>(s, mode, out2);
    case 2: return launch_residual<T, 2>(s, mode, out2);
    case 3: return launch_residual<T, 3>(s, mode, out2);
    case 4: return launch_residual<T, 4>(s, mode, out2);
    case 5: return launch_residual<T, 5>(s, mode, out2);
    case 6: return launch_residual<T, 6>(s, mode, out2);
  }
  return cudaErrorInvalidValue;
}

template <typename T>
cudaError_t dispatch_fused_first(const hr_solver* s, int mode, double* out2) {
  const int st = s->p.variant == 0 ? 16 : 6;
  switch (s->g.ng) {
    case 1: return launch_march<T, 1>(s, st, nullptr, nullptr, mode, s->a.partials, out2);
    case 2: return launch_march<T, 2>(s, st, nullptr, nullptr, mode, s->a.partials, out2);
    case 3: return launch_march<T, 3>(s, st, nullptr, nullptr, mode, s->a.partials, out2);
    case 4: return launch_march<T, 4>(s, st, nullptr, nullptr, mode, s->a.partials, out2);
    case 5: return launch_march<T, 5>(s, st, nullptr, nullptr, mode, s->a.partials, out2);
    case 6: return launch_march<T, 6>(s, st, nullptr, nullptr, mode, s->a.partials, out2);
  }
  return cudaErrorInvalidValue;
}

// hr_residual_static: the stand-alone residual launch of launch_march_stage<T, NG, 5> with the work-item
// partials and the {next item, CTAs done} counter pair in `scratch` (the file-scope array below) instead of
// the solver's workspace.  The numeric flag stays the solver's.  No programmatic launch: the clear of the
// counters that precedes it in the stream is complete when the kernel starts.
template <typename T, int NG>
cudaError_t launch_residual_static(const hr_solver* s, int mode, unsigned char* scratch, double* out2) {
  using C = MarchCfg<T>;
  constexpr size_t smem = HR_MARCH_SMEM(T, NG, 5);
  const dim3 block(C::TW / C::VX, C::BY, 1);
  const dim3 grid(s->march_grid[5], 1, 1);
  const MarchMaps mm = make_maps(s, 5);
  const StepArgs<T> a = make_args<T>(s, 5, nullptr, nullptr);
  MarchPlan plan = s->plan;
  plan.counters = reinterpret_cast<int*>(scratch);
  const ResidArgs ra{s->a.Wvol, reinterpret_cast<double*>(scratch + HR_STATIC_COUNTER_BYTES), mode, out2, s->a.ZH};
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s->stream;
  if (s->plan.cart) return cudaLaunchKernelEx(&cfg, HR_MARCH_KERNEL(T, NG, 5, true), s->g, a, plan, ra, mm);
  return cudaLaunchKernelEx(&cfg, HR_MARCH_KERNEL(T, NG, 5, false), s->g, a, plan, ra, mm);
}

template <typename T>
cudaError_t dispatch_residual_static(const hr_solver* s, int mode, unsigned char* scratch, double* out2) {
  switch (s->g.ng) {
    case 1: return launch_residual_static<T, 1>(s, mode, scratch, out2);
    case 2: return launch_residual_static<T, 2>(s, mode, scratch, out2);
    case 3: return launch_residual_static<T, 3>(s, mode, scratch, out2);
    case 4: return launch_residual_static<T, 4>(s, mode, scratch, out2);
    case 5: return launch_residual_static<T, 5>(s, mode, scratch, out2);
    case 6: return launch_residual_static<T, 6>(s, mode, scratch, out2);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

// Scratch of hr_residual_static: HR_STATIC_COUNTER_BYTES of launch counters, then HR_STATIC_MAX_PARTIALS pairs
// of doubles.  One copy per GPU that loads the library, held until the process exits.  In host code the name
// below is a host-side stand-in, not a device address: the launcher gets the address once per device from
// cudaGetSymbolAddress, with that device current, and hands it to the kernel.
static __device__ __align__(256) unsigned char hr_static_scratch[HR_STATIC_COUNTER_BYTES +
                                                                  (size_t)HR_STATIC_MAX_PARTIALS * 16];

cudaError_t hrk_residual_static(const hr_solver* s, int mode, double* out2_dev) {
  static std::mutex mu;
  static unsigned char* addr[HR_STATIC_MAX_DEVICES] = {};  // per device, filled on first use
  const int dev = s->p.device;
  if (dev < 0 || dev >= HR_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
  unsigned char* scratch;
  {
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
      int cur = -1;
      cudaError_t e = cudaGetDevice(&cur);
      if (e != cudaSuccess) return e;
      if (cur != dev && (e = cudaSetDevice(dev)) != cudaSuccess) return e;
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, hr_static_scratch);
      if (cur != dev) cudaSetDevice(cur);
      if (e != cudaSuccess) return e;
      addr[dev] = static_cast<unsigned char*>(p);
    }
    scratch = addr[dev];
  }
  // the array keeps the last call's contents: the counters must start at zero (the partials are all written
  // before they are read)
  cudaError_t e = cudaMemsetAsync(scratch, 0, HR_STATIC_COUNTER_BYTES, s->stream);
  if (e != cudaSuccess) return e;
  return s->p.dtype == HR_F64 ? dispatch_residual_static<double>(s, mode, scratch, out2_dev)
                              : dispatch_residual_static<float>(s, mode, scratch, out2_dev);
}

// Tiling of the marching kernels for a grid.  The chunk length is fixed later (hrk_prepare),
// once the persistent grid size is known.
MarchPlan hrk_make_plan(const int32_t n[3], int ng, int coord, int dtype) {
  MarchPlan m{};
  const int tw = dtype == HR_F64 ? MarchCfg<double>::TW : MarchCfg<float>::TW;
  const int by = dtype == HR_F64 ? MarchCfg<double>::BY : MarchCfg<float>::BY;
  m.ntx = (n[0] + tw - 1) / tw;
  m.nty = (n[1] + by - 1) / by;
  m.sph = coord == HR_SINHSPHERICAL ? 1 : 0;
  m.cyl = coord == HR_SINHCYLINDRICAL ? 1 : 0;
  m.cart = coord == HR_SINHCARTESIAN ? 1 : 0;
  m.zc = n[2];
  m.nzc = 1;
  m.gt = m.ntx * m.nty;
  m.mseg = 1;
  m.nseg = 1;
  m.ncol = 0;
  (void)ng;
  return m;
}

// Division of 0 <= n < 2^31 by a launch-invariant d >= 1 as a multiplication (Granlund & Montgomery 1994):
// p = 31 + ceil(log2 d), mul = ceil(2^p / d), n / d = umulhi(n, mul) >> (p - 32).  The item decode runs before a
// CTA's first loads are issued: three hardware divisions there are ~120 instructions in a dependent chain.
static void set_fast_div(uint32_t out[2], long long d) {
  out[0] = 0;
  out[1] = 0;
  if (d <= 1) return;  // mul = 0: the kernel takes n itself
  int lg = 0;
  while ((1ll << lg) < d) ++lg;
  const int p = 31 + lg;
  out[0] = (uint32_t)((((unsigned long long)1 << p) + (unsigned long long)d - 1) / (unsigned long long)d);
  out[1] = (uint32_t)(p - 32);
}

void hrk_replan(hr_solver* s, int share) {
  if (s->p.variant == 1 || s->p.variant == 2) return;
  if (share < 1) share = 1;
  // one chunking for all stages, balanced for the RK stage kernels (stages 2, 3 dominate)
  const int slots = s->march_slots[2] / share > 0 ? s->march_slots[2] / share : 1;
  choose_chunks(s->plan, s->g.n2, s->g.ng, slots, s->p.dtype == HR_F64);
  MarchPlan& m = s->plan;
  const long long ntiles = (long long)m.ntx * m.nty;
  m.mseg = 1;
  m.nseg = m.nzc;
  m.ncol = 0;
  // CTAs of the next launch that move in early wait in slots that the kernels of the other solvers could run in
  const char* pdl_env = std::getenv("HR_TUNE_PDL");  // tuning knob: 0 / 1 / 2, see MarchPlan::pdl
  m.pdl = pdl_env ? std::atoi(pdl_env) : (share == 1 ? 1 : 0);
  const char* col_env = std::getenv("HR_TUNE_COL");  // tuning knob: 0 = chunks only
  // Long items = whole columns, for the first whole waves of CTAs, where a column is short enough for window
  // priming to matter (<= 12 chunks) and there is at least one column per CTA; the remaining tiles' chunks are
  // handed out one by one and absorb the CTAs whose tiles cost more (ghost images at the axis and the poles).
  // Measured (burst, G point-substeps/s, columns / chunks only): config 3 fp64 73.9 / 70.2, 512x256x128 fp64 76.3 /
  // 75.3, 512x256x256 fp64 85.9 / 87.0; segments shorter than a column, or columns on grids with fewer tiles than
  // CTAs (every fp32 grid of the sweep: 256^3 fp32 100 against 130), never beat single chunks.
  const bool want = col_env ? std::atoi(col_env) != 0 : true;
  if (want && ntiles >= slots && m.nzc > 1 && m.nzc <= 12) {
    m.mseg = m.nzc;
    m.nseg = 1;
    m.ncol = (int)((ntiles / slots) * slots);
  }
  set_fast_div(m.dv_tiles, ntiles);
  set_fast_div(m.dv_ntx, m.ntx);
  set_fast_div(m.dv_rem, ntiles * m.nseg - m.ncol);
  set_fast_div(m.dv_o2, s->g.n_o2);
  set_fast_div(m.dv_T0, s->g.T0);
  const long long items = m.ncol + (ntiles * m.nseg - m.ncol) * m.mseg;
  for (int st = 0; st < 7; ++st) {
    s->march_grid[st] = (int)std::min<long long>(s->march_slots[st], items);
    s->march_grid_lean[st] = (int)std::min<long long>(s->march_slots_lean[st], items);
  }
}

cudaError_t hrk_prepare(hr_solver* s) {
  if (s->p.variant == 1 || s->p.variant == 2) return cudaSuccess;
  return s->p.dtype == HR_F64 ? prepare_march_ng<double>(s) : prepare_march_ng<float>(s);
}

int hrk_max_partials(const int32_t n[3], int ng, int dtype) {
  (void)ng;
  const int direct = ((n[0] + RBX - 1) / RBX) * ((n[1] + RBY - 1) / RBY) * n[2];
  // marching kernels: one partial pair per work item; a work item has at least one plane
  const MarchPlan m = hrk_make_plan(n, ng, 0, dtype);
  const long long march = (long long)m.ntx * m.nty * n[2];
  return direct > march ? direct : (int)march;
}

int hrk_launches_per_substep(const hr_solver* s) {
  if (s->p.variant == 1) return 4;  // RHS, BC outer, BC inner, RK
  if (s->p.variant == 2) return s->g.n_inner > 0 ? 2 : 1;
  return 1;
}

void hrk_row_geometry(int T0, int ng, size_t scalar_bytes, int* P0, int* off0) {
  const int line = (int)(128 / scalar_bytes);  // scalars per 128-byte line
  const int lead = (ng + line - 1) / line * line;  // first interior point starts a line
  *off0 = lead - ng;
  *P0 = (*off0 + T0 + line - 1) / line * line;
}

template <typename T>
cudaError_t repack_t(const hr_solver* s, void* dst, const void* src, bool to_public) {
  const HrGrid& g = s->g;
  const dim3 grid(g.T1 * g.T2, (g.T0 + 255) / 256, 1);
  if (to_public)
    k_repack<T, true><<<grid, 256, 0, s->stream>>>(g, static_cast<T*>(dst), static_cast<const T*>(src));
  else
    k_repack<T, false><<<grid, 256, 0, s->stream>>>(g, static_cast<T*>(dst), static_cast<const T*>(src));
  return cudaGetLastError();
}

cudaError_t hrk_pack(const hr_solver* s, void* dst_public, const void* src_stored) {
  return s->p.dtype == HR_F64 ? repack_t<double>(s, dst_public, src_stored, true)
                              : repack_t<float>(s, dst_public, src_stored, true);
}

cudaError_t hrk_unpack(const hr_solver* s, void* dst_stored, const void* src_public) {
  return s->p.dtype == HR_F64 ? repack_t<double>(s, dst_stored, src_public, false)
                              : repack_t<float>(s, dst_stored, src_public, false);
}

cudaError_t hrk_inner_fill(const hr_solver* s, void* fu, void* fv) {
  return s->p.dtype == HR_F64 ? inner_fill_t<double>(s, fu, fv) : inner_fill_t<float>(s, fu, fv);
}

cudaError_t hrk_substep_main(const hr_solver* s, int stage) {
  if (s->p.variant == 1)  // the RHS kernel alone; BC and RK follow in hrk_substep_fill
    return s->p.dtype == HR_F64 ? dispatch_paper<double>(s, 0, stage, nullptr, nullptr)
                                : dispatch_paper<float>(s, 0, stage, nullptr, nullptr);
  return s->p.dtype == HR_F64 ? dispatch_substep<double>(s, stage, nullptr, nullptr)
                              : dispatch_substep<float>(s, stage, nullptr, nullptr);
}

cudaError_t hrk_substep_fill(const hr_solver* s, int stage) {
  if (s->p.variant == 1) {  // Alg. 1 l.14-15 as separate kernels: BC (outer, inner) on k, then RK
    cudaError_t e = s->p.dtype == HR_F64 ? dispatch_paper<double>(s, 1, stage, nullptr, nullptr)
                                         : dispatch_paper<float>(s, 1, stage, nullptr, nullptr);
    if (e != cudaSuccess) return e;
    if ((e = hrk_inner_fill(s, s->a.B[0], s->a.B[1])) != cudaSuccess) return e;
    return s->p.dtype == HR_F64 ? launch_paper_rk<double>(s, stage) : launch_paper_rk<float>(s, stage);
  }
  if (s->p.variant != 2) return cudaSuccess;  // the marching kernel writes the ghost images itself
  // a3 on the array this stage wrote (bitwise equivalent to filling k, C15)
  void* const* out = (stage == 1 || stage == 3) ? s->a.A : (stage == 2 ? s->a.B : s->a.Y);
  return hrk_inner_fill(s, out[0], out[1]);
}

cudaError_t hrk_substep(const hr_solver* s, int stage) {
  cudaError_t e = hrk_substep_main(s, stage);
  if (e != cudaSuccess) return e;
  return hrk_substep_fill(s, stage);
}

cudaError_t hrk_eval_rhs(const hr_solver* s, void* ku, void* kv) {
  if (s->p.variant == 1) {
    cudaError_t e1 = s->p.dtype == HR_F64 ? dispatch_paper<double>(s, 0, 1, ku, kv)
                                          : dispatch_paper<float>(s, 0, 1, ku, kv);
    if (e1 != cudaSuccess) return e1;
    e1 = s->p.dtype == HR_F64 ? dispatch_paper<double>(s, 1, 1, ku, kv)
                              : dispatch_paper<float>(s, 1, 1, ku, kv);
    if (e1 != cudaSuccess) return e1;
    return hrk_inner_fill(s, ku, kv);
  }
  cudaError_t e = s->p.dtype == HR_F64 ? dispatch_substep<double>(s, 0, ku, kv)
                                       : dispatch_substep<float>(s, 0, ku, kv);
  if (e != cudaSuccess) return e;
  if (s->p.variant != 2) return cudaSuccess;
  return hrk_inner_fill(s, ku, kv);
}

// Alg. 1 l.9-16 in four launches: stage 1 also accumulates the residual of the state it starts
// from and its last CTA reduces the item partials into out2_dev (variant 0 only).
cudaError_t hrk_step_with_residual(const hr_solver* s, int mode, double* out2_dev) {
  if (s->p.variant == 1 || s->p.variant == 2) {
    cudaError_t e0 = hrk_residual(s, mode, out2_dev);
    for (int stage = 1; stage <= 4 && e0 == cudaSuccess; ++stage) e0 = hrk_substep(s, stage);
    return e0;
  }
  cudaError_t e = hrk_fused_first(s, mode, out2_dev);
  for (int stage = 2; stage <= 4 && e == cudaSuccess; ++stage) e = hrk_substep(s, stage);
  return e;
}

cudaError_t hrk_fused_first(const hr_solver* s, int mode, double* out2_dev) {
  return s->p.dtype == HR_F64 ? dispatch_fused_first<double>(s, mode, out2_dev)
                              : dispatch_fused_first<float>(s, mode, out2_dev);
}

cudaError_t hrk_residual(const hr_solver* s, int mode, double* out2_dev) {
  return s->p.dtype == HR_F64 ? dispatch_residual<double>(s, mode, out2_dev)
                              : dispatch_residual<float>(s, mode, out2_dev);
}

cudaError_t hrk_source(const hr_solver* s) {
  const HrGrid& g = s->g;
  const HrArrays& a = s->a;
  const int blocks = (int)((g.ntot + 255) / 256);
  int* flag = reinterpret_cast<int*>(a.result2);  // reused as the bad-point flag during create
  cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int), s->stream);
  if (e != cudaSuccess) return e;
  if (s->p.dtype == HR_F64)
    k_source<double><<<blocks, 256, 0, s->stream>>>(
        g, a.rho, a.rhoz, a.sinth, a.costh, a.sinph, a.cosph, a.punct, s->p.n_punctures,
        s->p.origin[0], s->p.origin[1], s->p.origin[2], static_cast<double*>(a.psi),
        static_cast<double*>(a.S), flag, s->p.coord == HR_SINHCARTESIAN);
  else
    k_source<float><<<blocks, 256, 0, s->stream>>>(
        g, a.rho, a.rhoz, a.sinth, a.costh, a.sinph, a.cosph, a.punct, s->p.n_punctures,
        s->p.origin[0], s->p.origin[1], s->p.origin[2], static_cast<float*>(a.psi),
        static_cast<float*>(a.S), flag, s->p.coord == HR_SINHCARTESIAN);
  return cudaGetLastError();
}
