// hr_march.cuh -- the default arrangement of the fused substep and of the residual on sm_100a:
// 2.5-D blocking.  One CTA owns a BX x BY tile of (i0, i1) and marches along i2 over a chunk of
// planes.
//   * the (i0, i1) halo tile of the stage's u lives in shared memory, double buffered: the halo
//     ring of plane z+1 is fetched with cp.async (LDGSTS) while plane z is being computed, the
//     tile centre is stored from registers; one __syncthreads per plane;
//   * the i2 stencil is a register pipeline of 2 NG + 1 values per thread, fed by one coalesced
//     load per plane issued a full iteration before it is consumed;
//   * the reference-metric factors depend on (i0, i1) only (reading C4), so each thread loads its
//     six coefficients once and keeps them in registers for the whole column;
//   * the RK combine (a4) happens in the same thread, so k never reaches HBM, and the thread that
//     produces a point also writes that point's inner-ghost images (a3, reading C14/C15) --
//     closed-form integer arithmetic, the inverse of the host's inner map -- so a substep is
//     one launch;
//   * the outer (radiation) points are handled by extra CTAs at the end of the same grid.
// Included by hr_kernels.cu only.
#pragma once

struct ResidArgs {
  const double* W;   // |h0 h1 h2| plane (C16)
  double* partials;  // 2 doubles per marching CTA
  int mode;
};

__device__ __forceinline__ void cp_async_scalar(double* smem_dst, const double* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_scalar(float* smem_dst, const float* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// Inner-ghost images of the point (j0, j1, j2) that was just written (j0 >= NG, j1 and j2
// interior): every ghost point whose source under the host's inner map (hr_api.cu:
// inner_source, reading C14) is this point.  r0 = 2NG-1-j0 if j0 < 2NG else -1; cB / cC = the
// theta-low / theta-high reflections of j1 or -1.  Each flip shifts phi by pi; phi is periodic.
template <typename T>
__device__ __forceinline__ void scatter_images(const HrGrid& g, int sph, T* __restrict__ ou,
                                               T* __restrict__ ov, T vu, T vv, int j0, int j1,
                                               int j2, int r0, int cB, int cC) {
  const int ng = g.ng;
  const int kbase = j2 - ng;
  const int half = g.n2 >> 1;
  const int s2 = g.T0 * g.T1;
#pragma unroll
  for (int f0 = 0; f0 < 2; ++f0) {
    if (f0 && r0 < 0) continue;
    const int d0 = f0 ? r0 : j0;
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      const int c = m == 0 ? j1 : (m == 1 ? cB : cC);
      if (c < 0) continue;
      const int d1 = (f0 && sph) ? g.T1 - 1 - c : c;
      const int flips = f0 + (m != 0);
      int kd = kbase - ((flips & 1) ? half : 0);
      if (kd < 0) kd += g.n2;
      const int base = d0 + g.T0 * d1;
      if (f0 || m) {
        const int d = base + (kd + ng) * s2;
        ou[d] = vu;
        ov[d] = vv;
      }
      if (kd < ng) {
        const int d = base + (kd + ng + g.n2) * s2;
        ou[d] = vu;
        ov[d] = vv;
      }
      if (kd >= g.n2 - ng) {
        const int d = base + (kd + ng - g.n2) * s2;
        ou[d] = vu;
        ov[d] = vv;
      }
    }
  }
}

// STAGE 0: k -> out (hr_eval_rhs); 1..4: RK4 stages (rk_combine); 5: residual (a5).
template <typename T, int NG, int STAGE, int BX, int BY>
__global__ void __launch_bounds__(BX* BY)
    k_march(const __grid_constant__ HrGrid g, const __grid_constant__ StepArgs<T> a,
            const __grid_constant__ MarchPlan plan, const __grid_constant__ ResidArgs ra) {
  constexpr int NT = BX * BY;
  constexpr int SW = BX + 2 * NG, SH = BY + 2 * NG;
  constexpr int NHALO = SW * SH - NT;
  constexpr int NSLOT = (NHALO + NT - 1) / NT;
  using F = FdTable<NG>;
  const int tid = threadIdx.y * BX + threadIdx.x;
  const int s2 = g.T0 * g.T1;

  // ---------------- outer points: radiation condition (a2, C13) + RK combine ----------------
  if constexpr (STAGE != 5) {
    if ((int)blockIdx.x >= plan.n_items) {
      const int m = ((int)blockIdx.x - plan.n_items) * NT + tid;
      if (m >= NG * g.n1 * g.n2) return;
      const int j = m % NG;
      const int r = m / NG;
      const int i1 = NG + r % g.n1, i2 = NG + r / g.n1;
      const int i0 = g.n0 + NG + j;
      const int c = i0 + g.T0 * i1 + s2 * i2;
      const int qo = j + NG * i1;
      const T r0 = a.RAD0[qo], r1 = a.RAD1[qo], ri = a.RADI[qo];
      const T uc = a.in_u[c], vc = a.in_v[c];
      const T ku = radiation_k(a.in_u, c, g.T0, r0, r1, ri);
      const T kv = radiation_k(a.in_v, c, g.T0, r0, r1, ri);
      T wu, wv;
      rk_combine<T, STAGE>(a, c, ku, kv, uc, vc, wu, wv);
      const int cB = i1 < 2 * NG ? 2 * NG - 1 - i1 : -1;
      const int cC = i1 >= g.n1 ? 2 * (g.n1 + NG) - 1 - i1 : -1;
      if (cB >= 0 || cC >= 0 || i2 < 2 * NG || i2 >= g.n2)
        scatter_images<T>(g, plan.sph, a.out_u, a.out_v, wu, wv, i0, i1, i2, -1, cB, cC);
      return;
    }
  }

  // ---------------- marching CTAs ----------------
  __shared__ T sm[2][SH][SW];
  const int bid = blockIdx.x;
  const int tx = bid % plan.ntx;
  const int rest = bid / plan.ntx;
  const int ty = rest % plan.nty;
  const int zci = rest / plan.nty;
  const int lx = threadIdx.x, ly = threadIdx.y;
  const int i0 = NG + tx * BX + lx, i1 = NG + ty * BY + ly;
  const bool active = i0 < g.n0 + NG && i1 < g.n1 + NG;
  // inactive threads of edge tiles still feed the tile centre (their points are ghosts that the
  // neighbours' stencils read), so they load real grid values, clamped to the grid
  const int col = min(i0, g.T0 - 1) + g.T0 * min(i1, g.T1 - 1);
  const int z_begin = NG + zci * plan.zc;
  const int z_end = min(z_begin + plan.zc, g.n2 + NG);

  // halo ring slots of this thread: shared-memory offset and in-plane global offset (-1: outside)
  int h_s[NSLOT], h_g[NSLOT];
#pragma unroll
  for (int s = 0; s < NSLOT; ++s) {
    const int h = tid + s * NT;
    int r, c;
    if (h < 2 * NG * SW) {
      r = h / SW;
      c = h - r * SW;
      if (r >= NG) r += BY;
    } else {
      const int hh = h - 2 * NG * SW;
      r = NG + hh / (2 * NG);
      c = hh % (2 * NG);
      if (c >= NG) c += BX;
    }
    const int gi0 = tx * BX + c, gi1 = ty * BY + r;
    h_s[s] = r * SW + c;
    h_g[s] = (h < NHALO && gi0 < g.T0 && gi1 < g.T1) ? gi0 + g.T0 * gi1 : -1;
  }

  // per-column constants
  T l00 = T(0), l11 = T(0), l22 = T(0), l0 = T(0), l1 = T(0), c2 = T(0);
  double wq = 0.0;
  int r0 = -1, cB = -1, cC = -1;
  if (active) {
    const int q = i0 + g.T0 * i1;
    l00 = a.L00[q]; l11 = a.L11[q]; l22 = a.L22[q]; l0 = a.L0[q]; l1 = a.L1[q];
    if constexpr (STAGE == 5) {
      wq = ra.mode == 0 ? ra.W[q] : 1.0;
    } else {
      c2 = a.C2[q];
      r0 = i0 < 2 * NG ? 2 * NG - 1 - i0 : -1;
      cB = i1 < 2 * NG ? 2 * NG - 1 - i1 : -1;
      cC = i1 >= g.n1 ? 2 * (g.n1 + NG) - 1 - i1 : -1;
    }
  }
  const bool inplane_images = (r0 >= 0) || (cB >= 0) || (cC >= 0);

  // register pipeline: p[j] = u(i0, i1, z - NG + j)
  const T* __restrict__ uin = a.in_u;
  T p[2 * NG + 1];
#pragma unroll
  for (int j = 0; j <= 2 * NG; ++j) p[j] = uin[col + (z_begin - NG + j) * s2];

  // stage the first plane
  {
    T* buf = &sm[0][0][0];
#pragma unroll
    for (int s = 0; s < NSLOT; ++s)
      if (h_g[s] >= 0) cp_async_scalar(buf + h_s[s], uin + h_g[s] + z_begin * s2);
    cp_async_commit();
    sm[0][ly + NG][lx + NG] = p[NG];
    cp_async_wait_all();
    __syncthreads();
  }

  double num = 0.0, den = 0.0;
  int b = 0;
  for (int z = z_begin; z < z_end; ++z, b ^= 1) {
    T front = T(0);
    if (z + 1 < z_end) {
      T* buf = &sm[b ^ 1][0][0];
#pragma unroll
      for (int s = 0; s < NSLOT; ++s)
        if (h_g[s] >= 0) cp_async_scalar(buf + h_s[s], uin + h_g[s] + (z + 1) * s2);
      sm[b ^ 1][ly + NG][lx + NG] = p[NG + 1];
      front = uin[col + (z + 1 + NG) * s2];
    }
    cp_async_commit();

    if (active) {
      const int c = col + z * s2;
      const T uc = p[NG];
      if constexpr (STAGE == 5) {
        const T psi = a.psi[c], S = a.S[c];
        T d00 = T(F::d2(0)) * uc, d11 = d00, d22 = d00, d0 = T(0), d1 = T(0);
#pragma unroll
        for (int k = 1; k <= NG; ++k) {
          const T a0 = sm[b][ly + NG][lx + NG + k], b0 = sm[b][ly + NG][lx + NG - k];
          const T a1 = sm[b][ly + NG + k][lx + NG], b1 = sm[b][ly + NG - k][lx + NG];
          d00 += T(F::d2(k)) * (a0 + b0);
          d11 += T(F::d2(k)) * (a1 + b1);
          d22 += T(F::d2(k)) * (p[NG + k] + p[NG - k]);
          d0 += T(F::c1(k)) * (a0 - b0);
          d1 += T(F::c1(k)) * (a1 - b1);
        }
        const T lap = l00 * d00 + l11 * d11 + l22 * d22 + l0 * d0 + l1 * d1;
        const T H = lap + S * pow_m7(psi + uc);
        num += wq * (double)H * (double)H;
        den += wq;
      } else {
        // pointwise streams of this plane, issued before the stencil arithmetic
        const T vc = a.in_v[c], psi = a.psi[c], S = a.S[c];
        T yu = T(0), yv = T(0), au = T(0), av = T(0);
        if constexpr (STAGE == 2 || STAGE == 3) {
          yu = a.y_u[c]; yv = a.y_v[c];
        }
        if constexpr (STAGE >= 2) {
          au = a.acc_u[c]; av = a.acc_v[c];
        }
        T d00 = T(F::d2(0)) * uc, d11 = d00, d22 = d00, d0 = T(0), d1 = T(0);
#pragma unroll
        for (int k = 1; k <= NG; ++k) {
          const T a0 = sm[b][ly + NG][lx + NG + k], b0 = sm[b][ly + NG][lx + NG - k];
          const T a1 = sm[b][ly + NG + k][lx + NG], b1 = sm[b][ly + NG - k][lx + NG];
          d00 += T(F::d2(k)) * (a0 + b0);
          d11 += T(F::d2(k)) * (a1 + b1);
          d22 += T(F::d2(k)) * (p[NG + k] + p[NG - k]);
          d0 += T(F::c1(k)) * (a0 - b0);
          d1 += T(F::c1(k)) * (a1 - b1);
        }
        const T lap = l00 * d00 + l11 * d11 + l22 * d22 + l0 * d0 + l1 * d1;
        const T ku = vc - a.eta * uc;
        const T kv = c2 * (lap + S * pow_m7(psi + uc));
        T wu, wv;
        rk_combine_regs<T, STAGE>(a, c, ku, kv, uc, vc, yu, yv, au, av, wu, wv);
        if (inplane_images || z < 2 * NG || z >= g.n2)
          scatter_images<T>(g, plan.sph, a.out_u, a.out_v, wu, wv, i0, i1, z, r0, cB, cC);
      }
    }

    cp_async_wait_all();
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 2 * NG; ++j) p[j] = p[j + 1];
    p[2 * NG] = front;
  }

  if constexpr (STAGE == 5) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      num += __shfl_down_sync(0xffffffffu, num, o);
      den += __shfl_down_sync(0xffffffffu, den, o);
    }
    __shared__ double red[2][NT / 32];
    if ((tid & 31) == 0) {
      red[0][tid >> 5] = num;
      red[1][tid >> 5] = den;
    }
    __syncthreads();
    if (tid == 0) {
      double sa = 0.0, sb = 0.0;
#pragma unroll
      for (int w = 0; w < NT / 32; ++w) {
        sa += red[0][w];
        sb += red[1][w];
      }
      ra.partials[2 * bid] = sa;
      ra.partials[2 * bid + 1] = sb;
    }
  }
}
