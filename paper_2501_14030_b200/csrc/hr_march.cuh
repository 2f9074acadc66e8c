// hr_march.cuh -- the default arrangement of the fused substep and of the residual on sm_100a:
// 2.5-D blocking.  One CTA owns a BX x BY tile of (i0, i1) and marches along i2 over a chunk of
// planes.
//   * every global load of the loop is asynchronous (cp.async / LDGSTS into shared memory) and
//     issued D planes ahead of its use, so no memory round trip sits on an iteration's critical
//     path and the bytes in flight do not depend on occupancy: per plane a thread fetches its
//     share of the (i0, i1) halo ring of the stage's u, the next value of its i2 pipeline, and
//     its own pointwise inputs (v, psi_BL, S, Y, ACC) into private slots of a (D+1)-deep ring;
//   * the tile centre is stored from registers one plane ahead; one __syncthreads per plane;
//   * the i2 stencil is a register pipeline of 2 NG + 1 values per thread;
//   * CTAs are persistent: the (tile, plane) iterations are split evenly over the resident CTAs,
//     each CTA marching one or more column segments, so there is no wave-quantisation tail;
//   * the reference-metric factors depend on (i0, i1) only (reading C4), so each thread loads its
//     six coefficients once and keeps them in registers for the whole column;
//   * the RK combine (a4) happens in the same thread, so k never reaches HBM, and the thread that
//     produces a point also writes that point's inner-ghost images (a3, reading C14/C15) --
//     closed-form integer arithmetic, the inverse of the host's inner map -- so a substep is
//     one launch;
//   * the outer (radiation) points are a grid-stride loop at the end of the same kernel.
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
__device__ __forceinline__ void prefetch_l2(const void* p) {
  asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

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
  const int s2 = g.P0 * g.T1;
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
      const int base = g.off0 + d0 + g.P0 * d1;
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


// Slots of a thread's private stream ring, in the order the stages need them.
enum { ST_FRONT = 0, ST_PSI = 1, ST_S = 2, ST_V = 3, ST_AU = 4, ST_AV = 5, ST_YU = 6, ST_YV = 7 };

template <int STAGE>
__host__ __device__ constexpr int march_nstreams() {
  return STAGE == 5 ? 3 : (STAGE <= 1 ? 4 : (STAGE == 4 ? 6 : 8));
}

template <typename T, int NG, int STAGE, int BX, int BY, int D>
__host__ __device__ constexpr size_t march_smem_bytes() {
  return sizeof(T) * (size_t)(D + 1) *
         ((size_t)(BX + 2 * NG) * (BY + 2 * NG) + (size_t)march_nstreams<STAGE>() * BX * BY);
}

// STAGE 0: k -> out (hr_eval_rhs); 1..4: RK4 stages (rk_combine); 5: residual (a5).
// D = planes of asynchronous look-ahead.
template <typename T, int NG, int STAGE, int BX, int BY, int D>
__global__ void __launch_bounds__(BX* BY, sizeof(T) == 8 ? HR_MARCH_MINB_F64 : HR_MARCH_MINB_F32)
    k_march(const __grid_constant__ HrGrid g, const __grid_constant__ StepArgs<T> a,
            const __grid_constant__ MarchPlan plan, const __grid_constant__ ResidArgs ra) {
  constexpr int NT = BX * BY;
  constexpr int SW = BX + 2 * NG, SH = BY + 2 * NG;
  constexpr int TILE = SW * SH;
  constexpr int NHALO = TILE - NT;
  constexpr int NSLOT = (NHALO + NT - 1) / NT;
  constexpr int NS = march_nstreams<STAGE>();
  constexpr int RING = D + 1;
  using F = FdTable<NG>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* const tiles = reinterpret_cast<T*>(smem_raw);  // [RING][SH][SW]
  T* const strm = tiles + RING * TILE;              // [RING][NS][NT]

  const int lx = threadIdx.x, ly = threadIdx.y;
  const int tid = ly * BX + lx;
  const int s2 = g.P0 * g.T1;
  const T* __restrict__ uin = a.in_u;
  const int ctr = (ly + NG) * SW + lx + NG;  // this thread's point in a tile

  // work items = (chunk of planes, tile), chunk-major, so that the CTAs resident at any time work
  // on neighbouring tiles of the same planes (halo rows and partial lines meet in L2)
  const int ntiles = plan.ntx * plan.nty;
  const int n_items = ntiles * plan.nzc;

  double num = 0.0, den = 0.0;

  for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int chunk = item / ntiles;
    const int tile_id = item - chunk * ntiles;
    const int zi = chunk * plan.zc;
    const int seg = min(plan.zc, g.n2 - zi);
    const int tx = tile_id % plan.ntx, ty = tile_id / plan.ntx;
    const int z_begin = NG + zi, z_end = z_begin + seg;
    const int i0 = NG + tx * BX + lx, i1 = NG + ty * BY + ly;
    const bool active = i0 < g.n0 + NG && i1 < g.n1 + NG;
    // inactive threads of edge tiles still feed the tile centre (their points are ghosts that
    // the neighbours' stencils read), so they track real grid values, clamped to the grid
    const int col = g.off0 + min(i0, g.T0 - 1) + g.P0 * min(i1, g.T1 - 1);

    // halo ring slots of this thread: tile offset and in-plane global offset (-1: none)
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
      h_g[s] = (h < NHALO && gi0 < g.T0 && gi1 < g.T1) ? g.off0 + gi0 + g.P0 * gi1 : -1;
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

    // everything plane zz needs from global memory, as one cp.async group into ring slot sl
    auto issue = [&](int zz, int sl) {
      if (zz < z_end) {
        T* tl = tiles + sl * TILE;
        T* st = strm + sl * (NS * NT) + tid;
        const int pl = zz * s2;
#pragma unroll
        for (int s = 0; s < NSLOT; ++s)
          if (h_g[s] >= 0) cp_async_scalar(tl + h_s[s], uin + h_g[s] + pl);
        const int c = col + pl;
        cp_async_scalar(st + ST_FRONT * NT, uin + c + NG * s2);
        if (active) {
          cp_async_scalar(st + ST_PSI * NT, a.psi + c);
          cp_async_scalar(st + ST_S * NT, a.S + c);
          if constexpr (STAGE != 5) cp_async_scalar(st + ST_V * NT, a.in_v + c);
          if constexpr (STAGE >= 2 && STAGE <= 4) {
            cp_async_scalar(st + ST_AU * NT, a.acc_u + c);
            cp_async_scalar(st + ST_AV * NT, a.acc_v + c);
          }
          if constexpr (STAGE == 2 || STAGE == 3) {
            cp_async_scalar(st + ST_YU * NT, a.y_u + c);
            cp_async_scalar(st + ST_YV * NT, a.y_v + c);
          }
        }
      }
      cp_async_commit();
    };

    // prologue: look-ahead groups, then the register pipeline.  w(k) = u(i0, i1, z - NG + k),
    // k = 0..2NG, lives in p[(j + k) % U] where j = (z - z_begin) % U: the plane loop is unrolled
    // U = 2NG+1 times so the window rotates through the registers without moves.
#pragma unroll
    for (int d = 0; d < D; ++d) issue(z_begin + d, d);
    constexpr int U = 2 * NG + 1;
    T p[U];
#pragma unroll
    for (int k = 0; k < 2 * NG; ++k) p[k] = uin[col + (z_begin - NG + k) * s2];
    tiles[ctr] = p[NG];

    int sl = 0;  // ring slot of plane z
    for (int zb = z_begin; zb < z_end; zb += U) {
#pragma unroll
      for (int j = 0; j < U; ++j) {
        const int z = zb + j;
        if (z >= z_end) break;
#define HR_W(k) p[(j + (k)) % U]
        cp_async_wait_group<D - 1>();  // this thread's group of plane z has landed
        __syncthreads();               // everyone's has; slot of plane z-1 is free again
        {
          int sn = sl + D;
          if (sn >= RING) sn -= RING;
          issue(z + D, sn);
        }
        const T* tl = tiles + sl * TILE;
        const T* st = strm + sl * (NS * NT) + tid;
        HR_W(2 * NG) = st[ST_FRONT * NT];
        int sn1 = sl + 1;
        if (sn1 >= RING) sn1 = 0;
        if (z + 1 < z_end) tiles[sn1 * TILE + ctr] = HR_W(NG + 1);

        if (active) {
          const int c = col + z * s2;
          const T uc = HR_W(NG);
          T d00 = T(F::d2(0)) * uc, d11 = d00, d22 = d00, d0 = T(0), d1 = T(0);
#pragma unroll
          for (int k = 1; k <= NG; ++k) {
            const T a0 = tl[ctr + k], b0 = tl[ctr - k];
            const T a1 = tl[ctr + k * SW], b1 = tl[ctr - k * SW];
            d00 += T(F::d2(k)) * (a0 + b0);
            d11 += T(F::d2(k)) * (a1 + b1);
            d22 += T(F::d2(k)) * (HR_W(NG + k) + HR_W(NG - k));
            d0 += T(F::c1(k)) * (a0 - b0);
            d1 += T(F::c1(k)) * (a1 - b1);
          }
          const T lap = l00 * d00 + l11 * d11 + l22 * d22 + l0 * d0 + l1 * d1;
          const T H = lap + st[ST_S * NT] * pow_m7(st[ST_PSI * NT] + uc);
          if constexpr (STAGE == 5) {
            num += wq * (double)H * (double)H;
            den += wq;
          } else {
            const T vc = st[ST_V * NT];
            T yu = T(0), yv = T(0), au = T(0), av = T(0);
            if constexpr (STAGE >= 2 && STAGE <= 4) {
              au = st[ST_AU * NT];
              av = st[ST_AV * NT];
            }
            if constexpr (STAGE == 2 || STAGE == 3) {
              yu = st[ST_YU * NT];
              yv = st[ST_YV * NT];
            }
            const T ku = vc - a.eta * uc;
            const T kv = c2 * H;
            T wu, wv;
            rk_combine_regs<T, STAGE>(a, c, ku, kv, uc, vc, yu, yv, au, av, wu, wv);
            if (inplane_images || z < 2 * NG || z >= g.n2)
              scatter_images<T>(g, plan.sph, a.out_u, a.out_v, wu, wv, i0, i1, z, r0, cB, cC);
          }
        }
        if (++sl >= RING) sl = 0;
#undef HR_W
      }
    }
    cp_async_wait_all();
    __syncthreads();  // the ring is reused by the next segment
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
      ra.partials[2 * blockIdx.x] = sa;
      ra.partials[2 * blockIdx.x + 1] = sb;
    }
  } else {
    // ---------------- outer points: radiation condition (a2, C13) + RK combine ----------------
    const int n_outer = NG * g.n1 * g.n2;
    for (int m = blockIdx.x * NT + tid; m < n_outer; m += gridDim.x * NT) {
      const int j = m % NG;
      const int r = m / NG;
      const int i1 = NG + r % g.n1, i2 = NG + r / g.n1;
      const int i0 = g.n0 + NG + j;
      const int c = g.off0 + i0 + g.P0 * i1 + s2 * i2;
      const int qo = j + NG * i1;
      const T r0 = a.RAD0[qo], r1 = a.RAD1[qo], ri = a.RADI[qo];
      const T uc = a.in_u[c], vc = a.in_v[c];
      const T ku = radiation_k(a.in_u, c, g.P0, r0, r1, ri);
      const T kv = radiation_k(a.in_v, c, g.P0, r0, r1, ri);
      T wu, wv;
      rk_combine<T, STAGE>(a, c, ku, kv, uc, vc, wu, wv);
      const int cB = i1 < 2 * NG ? 2 * NG - 1 - i1 : -1;
      const int cC = i1 >= g.n1 ? 2 * (g.n1 + NG) - 1 - i1 : -1;
      if (cB >= 0 || cC >= 0 || i2 < 2 * NG || i2 >= g.n2)
        scatter_images<T>(g, plan.sph, a.out_u, a.out_v, wu, wv, i0, i1, i2, -1, cB, cC);
    }
  }
}
