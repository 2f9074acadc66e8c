// hr_march.cuh -- the default arrangement of the fused substep and of the residual on sm_100a:
// 2.5-D blocking with TMA.  One CTA owns a TW x BY tile of (i0, i1) and marches along i2.
//   * every load of the loop is a TMA box copy (cp.async.bulk.tensor.3d) issued by one thread D
//     planes ahead of its use into a (D+1)-deep shared-memory ring and completed on an mbarrier:
//     per plane the (i0, i1) halo tile of the stage's u, the next plane of the i2 window, and the
//     tile's pointwise inputs (v, psi_BL, S, Y, ACC).  No memory round trip sits on an
//     iteration's critical path, the bytes in flight do not depend on occupancy, and the
//     compute threads spend no instructions on load addresses;
//   * a thread owns VX consecutive points along i0 and reads / writes them as one vector
//     (rows of the stored layout start on 128-byte lines, hr_internal.h);
//   * the i2 stencil is a register window of 2 NG + 1 planes per point; the plane loop is
//     unrolled twice over a window one plane longer, which is shifted by two planes per pass
//     (HR_MARCH_ROTATE = 1 unrolls 2 NG + 1 times instead so the window rotates without moves;
//     that copy of the loop no longer fits the 32 KB instruction cache and measured no faster);
//   * fp32: a thread owns two points and does the i1 / i2 stencils, the metric combination, the
//     source term and the RK combine on packed pairs (fma/add/mul.f32x2 -> FFMA2 / FADD2 / FMUL2);
//   * CTAs are persistent over work items: whole columns of a tile for the first whole waves of
//     CTAs where a column is short (config 3), then (chunk of planes, tile) items, chunk-major, so the
//     CTAs resident at any time work on neighbouring tiles of the same planes (halo rows meet in
//     L2); after its first item a CTA takes the next one from an atomic counter, unless there are
//     no more items than CTAs;
//   * the reference-metric factors depend on (i0, i1) only (reading C4), so each thread loads its
//     six coefficients once per column and keeps them in registers;
//   * the RK combine (a4) happens in the same thread, so k never reaches HBM (default: classic RK4
//     without a running sum, STAGE codes 11-14 and 16, 32w bytes per point and step; STAGE 1-4
//     and 6: the running-sum form, variant 3, 40w; fp32 takes the increment-preserving stages 22 / 24,
//     34w), and the thread that
//     produces a point also writes that point's inner-ghost images (a3, reading C14/C15) --
//     closed-form integer arithmetic, the inverse of the host's inner map -- so a substep is
//     one launch;
//   * the outer (radiation) points are a grid-stride loop of the same kernel, run by every CTA once
//     the first loads of its first item are in flight; CART = the SinhCartesian instantiation (C25);
//   * launched with programmatic stream serialization: launch_dependents at entry where every CTA has one
//     item (small grids), after the item loop where items are handed out; griddepcontrol.wait before the
//     first access to what the previous substep wrote.
// Included by hr_kernels.cu only.
#pragma once

struct ResidArgs {
  const double* W;   // |h0 h1 h2| plane (C16)
  double* partials;  // 2 doubles per work item
  int mode;
  double* out2;      // { sum w H^2, sum w }, written by the last CTA to finish
  const double* ZH;  // SinhCartesian (C25): h2 per plane, the x2 factor of the weight
};

template <typename T, int VX>
struct alignas(sizeof(T) * VX) Vec {
  T v[VX];
};

// Two fp32 values in one 64-bit register pair and the sm_100 packed arithmetic on them
// (add/sub/mul/fma.f32x2 -> FADD2 / FMUL2 / FFMA2: one issue slot for two points).  lo = point 0.
struct F2 {
  unsigned long long r;
};
__device__ __forceinline__ F2 f2_pack(float lo, float hi) {
  F2 x;
  asm("mov.b64 %0, {%1, %2};" : "=l"(x.r) : "f"(lo), "f"(hi));
  return x;
}
__device__ __forceinline__ void f2_unpack(F2 x, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x.r));
}
__device__ __forceinline__ F2 f2_bc(float w) { return f2_pack(w, w); }
__device__ __forceinline__ F2 f2_add(F2 a, F2 b) {
  F2 d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.r) : "l"(a.r), "l"(b.r));
  return d;
}
__device__ __forceinline__ F2 f2_sub(F2 a, F2 b) {
  F2 d;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d.r) : "l"(a.r), "l"(b.r));
  return d;
}
__device__ __forceinline__ F2 f2_mul(F2 a, F2 b) {
  F2 d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.r) : "l"(a.r), "l"(b.r));
  return d;
}
__device__ __forceinline__ F2 f2_fma(F2 a, F2 b, F2 c) {
  F2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.r) : "l"(a.r), "l"(b.r), "l"(c.r));
  return d;
}
// the RK combine of rk_values on two points at once (same formulas, same order)
template <int RK>
__device__ __forceinline__ void rk_values_f2(float dt, F2 ku, F2 kv, F2 in_u, F2 in_v, F2 yu, F2 yv,
                                             F2 au, F2 av, F2& wu, F2& wv, F2& nu, F2& nv) {
  nu = f2_bc(0.f);
  nv = nu;
  if constexpr (RK == 0) {
    wu = ku;
    wv = kv;
  } else if constexpr (RK == 1) {
    const F2 h = f2_bc(dt * 0.5f), s = f2_bc(dt / 6.f);
    wu = f2_fma(h, ku, in_u);
    wv = f2_fma(h, kv, in_v);
    nu = f2_fma(s, ku, in_u);
    nv = f2_fma(s, kv, in_v);
  } else if constexpr (RK == 2 || RK == 3) {
    const F2 h = f2_bc(RK == 2 ? dt * 0.5f : dt), s = f2_bc(dt / 3.f);
    wu = f2_fma(h, ku, yu);
    wv = f2_fma(h, kv, yv);
    nu = f2_fma(s, ku, au);
    nv = f2_fma(s, kv, av);
  } else {
    const F2 s = f2_bc(dt / 6.f);
    wu = f2_fma(s, ku, au);
    wv = f2_fma(s, kv, av);
  }
}

// The ACC-free arrangement (k_march, STAGE >= 10), one field at a time: `in` is the stage's own
// input (Y, Y1, Y2 or Y3); y is Y for stages 2 and 3 and Q = (Y1 - Y) + 2 Y2 for stage 4.
template <typename T, int RK>
__device__ __forceinline__ T rk_lean(T dt, T k, T in, T y) {
  if constexpr (RK == 0) return k;
  if constexpr (RK == 1) return in + dt * T(0.5) * k;
  if constexpr (RK == 2) return y + dt * T(0.5) * k;
  if constexpr (RK == 3) return y + dt * k;
  return (T(1) / T(3)) * (y + in) + dt / T(6) * k;  // Y_new = (1/3)(Q + Y3) + dt/6 k4
}
template <int RK>
__device__ __forceinline__ F2 rk_lean_f2(float dt, F2 k, F2 in, F2 y) {
  if constexpr (RK == 0) return k;
  if constexpr (RK == 1) return f2_fma(f2_bc(dt * 0.5f), k, in);
  if constexpr (RK == 2) return f2_fma(f2_bc(dt * 0.5f), k, y);
  if constexpr (RK == 3) return f2_fma(f2_bc(dt), k, y);
  return f2_fma(f2_bc(dt / 6.f), k, f2_mul(f2_bc(1.f / 3.f), f2_add(y, in)));
}

// The increment-preserving form of the same arrangement (STAGE >= 20; the fp32 default): stage 2 keeps
// Qd = (Y1 - Y) + dt k2 -- an increment, so its rounding error is relative to dt k, not to Y -- and
// stage 4 adds increments to Y:  Y_new = Y + [ (1/3)(Qd + (Y3 - Y)) + dt/6 k4 ].  One rounding at the
// size of Y per step, like the textbook k-sum form, at the price of reading Y in stage 4 (10w instead
// of 8w in that stage).  In the plain ACC-free form the roundings of Q = (Y1 - Y) + 2 Y2, of Q + Y3
// and of the product by 1/3 are each of the size of ulp(Y): twice the per-step noise in the state,
// which the residual amplifies by 1/ds^2 (fp32: visible against the 1e-4 bar of reading C21).
template <typename T>
__device__ __forceinline__ T rk_prec_q(T dt, T k, T in, T y) {
  return (in - y) + dt * k;
}
template <typename T>
__device__ __forceinline__ T rk_prec_4(T dt, T k, T in, T q, T y) {
  return y + ((T(1) / T(3)) * (q + (in - y)) + dt / T(6) * k);
}
__device__ __forceinline__ F2 rk_prec_q_f2(float dt, F2 k, F2 in, F2 y) {
  return f2_fma(f2_bc(dt), k, f2_sub(in, y));
}
__device__ __forceinline__ F2 rk_prec_4_f2(float dt, F2 k, F2 in, F2 q, F2 y) {
  const F2 t = f2_mul(f2_bc(1.f / 3.f), f2_add(q, f2_sub(in, y)));
  return f2_add(y, f2_fma(f2_bc(dt / 6.f), k, t));
}

// Tensor maps of one launch: the halo-tile box of the stage's u and the TW x BY box of every
// pointwise input, indexed by ST_*.
struct alignas(64) MarchMaps {
  CUtensorMap tile;
  CUtensorMap st[8];
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
// n / d for 0 <= n < 2^31 with the multiplier and shift the host derived from d (MarchPlan::dv_*)
__device__ __forceinline__ int fast_div(int n, const uint32_t dv[2]) {
  return dv[0] ? (int)(__umulhi((uint32_t)n, dv[0]) >> dv[1]) : n;
}
// one lane of a converged warp (the TMA issue then compiles to straight-line uniform-datapath code instead of a
// loop over the active lanes of a divergent branch)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}\n" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes)
               : "memory");
}
// A lost TMA transaction must fail loudly, not hang -- but a long stall (compute-sanitizer, a debugger,
// time-slicing, an ncu replay) is not a lost transaction: the watchdog is wall-clock based
// (HR_MBAR_TIMEOUT_NS of %globaltimer, default 20 s; 0 compiles it out), looked at every 4096 failed polls.
#ifndef HR_MBAR_TIMEOUT_NS
#define HR_MBAR_TIMEOUT_NS 20000000000ull
#endif
__device__ __forceinline__ unsigned long long global_timer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t bar, uint32_t phase) {
  uint32_t ok;
  asm volatile(
      "{\n.reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n}\n"
      : "=r"(ok)
      : "r"(bar), "r"(phase)
      : "memory");
  return ok;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t phase) {
  if (mbar_try_wait(bar, phase)) return;  // the common case costs one instruction and a branch
  [[maybe_unused]] uint32_t spins = 0;
  [[maybe_unused]] unsigned long long t0 = 0;
  do {
#if HR_MBAR_TIMEOUT_NS
    if ((++spins & 4095u) == 0) {
      const unsigned long long now = global_timer_ns();
      if (t0 == 0) t0 = now;
      else if (now - t0 > HR_MBAR_TIMEOUT_NS) __trap();
    }
#endif
  } while (!mbar_try_wait(bar, phase));
}
// L2 eviction policies for the loads: the pointwise inputs are read once per substep
// (evict first), u is read again by the neighbouring tiles and, NG planes later, as a halo tile
// (evict last).
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(p));
  return p;
}
__device__ __forceinline__ void tma_load_3d_hint(uint32_t dst, const CUtensorMap* map, int x, int y,
                                                 int z, uint32_t bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
      "[%0], [%1, {%2, %3, %4}], [%5], %6;\n" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int x, int y, int z,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%2, %3, %4}], [%5];\n" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar)
      : "memory");
}

// Inner-ghost images of the point (j0, j1, j2) that was just written (j0 >= NG, j1 and j2
// interior): every ghost point whose source under the host's inner map (hr_api.cu:
// inner_source, reading C14) is this point.  r0 = 2NG-1-j0 if j0 < 2NG else -1; cB / cC = the
// theta-low / theta-high reflections of j1 or -1.  Each flip shifts phi by pi; phi is periodic.
// Not inlined: few points have images, and inlining this into the plane loop pushed the stage
// kernels out of the instruction cache.
struct ImgGeom {
  int ng, n2, T1, P0, off0, sph;
};
template <typename T>
__device__ __noinline__ void scatter_images(ImgGeom g, T* __restrict__ ou, T* __restrict__ ov, T vu,
                                            T vv, int j0, int j1, int j2, int r0, int cB, int cC) {
  const int ng = g.ng;
  const int kbase = j2 - ng;
  const int half = g.n2 >> 1;
  const int s2 = g.P0 * g.T1;
#pragma unroll 1
  for (int f0 = 0; f0 < 2; ++f0) {
    if (f0 && r0 < 0) continue;
    const int d0 = f0 ? r0 : j0;
#pragma unroll 1
    for (int m = 0; m < 3; ++m) {
      const int c = m == 0 ? j1 : (m == 1 ? cB : cC);
      if (c < 0) continue;
      const int d1 = (f0 && g.sph) ? g.T1 - 1 - c : c;
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

// The same for the VX points (i0 .. i0+VX-1, i1, z) a marching thread has just written, with the
// common cases first: the phi-periodic images of the points themselves and the theta-reflected
// rows are whole-vector stores; only the rho -> -rho reflections (first 2NG points of a row) go
// point by point.  Not inlined (see above); called for boundary planes / boundary threads only.
template <typename T, int VX>
__device__ __noinline__ void scatter_vec(ImgGeom g, T* __restrict__ ou, T* __restrict__ ov,
                                         Vec<T, VX> wu, Vec<T, VX> wv, int i0, int i1, int z,
                                         int nact, int cB, int cC) {
  const int ng = g.ng, n2 = g.n2;
  const int s2 = g.P0 * g.T1;
  const int k0 = z - ng;  // phi index of the source
  int k1 = k0 - (n2 >> 1);  // after an odd number of flips
  if (k1 < 0) k1 += n2;
  auto store_v = [&](int d) {
    if (nact == VX) {
      *reinterpret_cast<Vec<T, VX>*>(ou + d) = wu;
      *reinterpret_cast<Vec<T, VX>*>(ov + d) = wv;
    } else {
#pragma unroll
      for (int j = 0; j < VX; ++j)
        if (j < nact) {
          ou[d + j] = wu.v[j];
          ov[d + j] = wv.v[j];
        }
    }
  };
  auto put_v = [&](int rowbase, int k, bool main) {
    if (main) store_v(rowbase + (k + ng) * s2);
    if (k < ng) store_v(rowbase + (k + ng + n2) * s2);
    if (k >= n2 - ng) store_v(rowbase + (k + ng - n2) * s2);
  };
  const int rb = g.off0 + i0;
  put_v(rb + g.P0 * i1, k0, false);
  if (cB >= 0) put_v(rb + g.P0 * cB, k1, true);
  if (cC >= 0) put_v(rb + g.P0 * cC, k1, true);
  if (i0 < 2 * ng) {
#pragma unroll
    for (int j = 0; j < VX; ++j) {
      if (j >= nact || i0 + j >= 2 * ng) continue;
      const int rr = g.off0 + 2 * ng - 1 - (i0 + j);
      const T vu = wu.v[j], vv = wv.v[j];
#pragma unroll 1
      for (int m = 0; m < 3; ++m) {
        const int c = m == 0 ? i1 : (m == 1 ? cB : cC);
        if (c < 0) continue;
        const int d1 = g.sph ? g.T1 - 1 - c : c;
        const int k = m == 0 ? k1 : k0;  // one flip, or two
        const int rowbase = rr + g.P0 * d1;
        {
          const int d = rowbase + (k + ng) * s2;
          ou[d] = vu;
          ov[d] = vv;
        }
        if (k < ng) {
          const int d = rowbase + (k + ng + n2) * s2;
          ou[d] = vu;
          ov[d] = vv;
        }
        if (k >= n2 - ng) {
          const int d = rowbase + (k + ng - n2) * s2;
          ou[d] = vu;
          ov[d] = vv;
        }
      }
    }
  }
}

// Boxes of a ring slot, in the order the stages need them.
enum { ST_FRONT = 0, ST_PSI = 1, ST_S = 2, ST_V = 3, ST_AU = 4, ST_AV = 5, ST_YU = 6, ST_YV = 7 };

template <int STAGE>
__host__ __device__ constexpr int march_nstreams() {
  if (STAGE >= 10) {  // ACC-free stages 11..14, 16: front psi S v | Y (stages 2, 3) or Q (stage 4)
    if (STAGE == 24) return 8;  // increment-preserving stage 4: ... | Qd | Y
    return (STAGE % 10 == 1 || STAGE % 10 == 6) ? 4 : 6;
  }
  return STAGE == 5 ? 3 : ((STAGE <= 1 || STAGE == 6) ? 4 : (STAGE == 4 ? 6 : 8));
}

// Geometry shared by the kernel and the host (tensor-map boxes, shared-memory size).
//   NGA  halo width of the tile along i0, NG rounded up so that box rows are whole 16-byte units
//   SWA  tile row length, SH tile rows
template <typename T, int NG, int TW, int BY>
struct MarchGeom {
  static constexpr int Q = 16 / (int)sizeof(T);
  static constexpr int NGA = (NG + Q - 1) / Q * Q;
  static constexpr int SWA = TW + 2 * NGA;
  static constexpr int SH = BY + 2 * NG;
  static constexpr int TILE_BYTES = (SWA * SH * (int)sizeof(T) + 127) / 128 * 128;
  static constexpr int BOX_BYTES = TW * BY * (int)sizeof(T);
  static_assert(BOX_BYTES % 128 == 0, "stream boxes must keep 128-byte alignment");
};

template <typename T, int NG, int STAGE, int TW, int BY, int D>
__host__ __device__ constexpr size_t march_smem_bytes() {
  using G = MarchGeom<T, NG, TW, BY>;
  return 128 + (size_t)(D + 1) * (G::TILE_BYTES + march_nstreams<STAGE>() * G::BOX_BYTES);
}

// STAGE 0: k -> out (hr_eval_rhs); 1..4: RK4 stages (rk_combine); 5: residual (a5);
// 6: RK4 stage 1 that also accumulates the residual of its input state -- the bracket of Eq. 5 at
// the state Y is exactly H of Eq. 4, so Alg. 1 l.9-11 followed by l.12-16 needs no pass of its own.
// TW x BY points per tile, VX points per thread along i0, D planes of look-ahead.
// CART: the SinhCartesian (C25) instantiation -- a u_2 term, per-plane factors, six outer faces, no ghost images.
// A template parameter because even uniform branches on it in the plane loop cost the other systems 4 %.
template <typename T, int NG, int STAGE, int TW, int BY, int VX, int D, bool CART>
__global__ void __launch_bounds__((TW / VX) * BY,
                                  sizeof(T) == 8 ? HR_MARCH_MINB_F64 : HR_MARCH_MINB_F32)
    k_march(const __grid_constant__ HrGrid g, const __grid_constant__ StepArgs<T> a,
            const __grid_constant__ MarchPlan plan, const __grid_constant__ ResidArgs ra,
            const __grid_constant__ MarchMaps mm) {
  using G = MarchGeom<T, NG, TW, BY>;
  using V = Vec<T, VX>;
  using F = FdTable<NG>;
  constexpr int BXT = TW / VX;  // threads along i0
  constexpr int NT = BXT * BY;
  constexpr int NGA = G::NGA, SWA = G::SWA;
  constexpr int NGV = (NG + VX - 1) / VX * VX;  // halo rounded to whole vectors
  constexpr int NS = march_nstreams<STAGE>();
  // STAGE >= 10: the ACC-free ("lean") arrangement of the same RK4 (the default): stage 1 writes
  // Y1 = Y + dt/2 k1 (buffer A); stage 2 writes Y2 = Y + dt/2 k2 (B) and Q = (Y1 - Y) + 2 Y2 (the
  // ACC buffer); stage 3 writes Y3 = Y + dt k3 (A again, Y1 is no longer needed); stage 4 forms
  // Y_new = (1/3)(Q + Y3) + dt/6 k4 = Y + dt/6 (k1 + 2 k2 + 2 k3 + k4).  Bytes per point:
  // 6w, 10w, 8w, 8w = 32w per step instead of 8w, 12w, 12w, 8w = 40w.
  constexpr bool LEAN = STAGE >= 10;
  // the numeric guard (psi_BL + u <= 0 or NaN -> plan.flag) looks at the state a step starts from and at the
  // residual's / hr_eval_rhs's input: stages 2-4 of a step that goes wrong feed a stage 1 that reports it
  constexpr bool GUARD = STAGE % 10 == 0 || STAGE % 10 == 1 || STAGE % 10 == 5 || STAGE % 10 == 6;
  constexpr bool PREC = STAGE >= 20;  // increment-preserving stages 22 and 24 (rk_prec_q, rk_prec_4)
  constexpr int ST = STAGE % 10;
  constexpr int RK = ST == 6 ? 1 : ST;                  // which RK combine (0 = store k)
  constexpr bool RESID = ST == 5 || ST == 6;            // accumulate sum w H^2, sum w
  constexpr bool ADVANCE = ST != 5;                     // write stage outputs and ghost images
  // slots of the pointwise boxes (lean: Y right after v, then Y1, then Y2)
  constexpr int S_YU = LEAN ? 4 : ST_YU, S_YV = LEAN ? 5 : ST_YV;
  constexpr int S_AU = LEAN ? 6 : ST_AU, S_AV = LEAN ? 7 : ST_AV;
  constexpr bool NEED_Y = (RK == 2 || RK == 3) || (LEAN && RK == 4);  // lean stage 4: the Y slot is Q
  constexpr bool NEED_A = (!LEAN && RK >= 2 && RK <= 4) || (PREC && RK == 4);  // PREC stage 4: the A slot is Y
  constexpr bool WRITE_ACC = LEAN ? RK == 2 : (RK >= 1 && RK <= 3);   // lean stage 2: ACC <- Q
  constexpr bool PACKED = HR_MARCH_F32X2 && sizeof(T) == 4 && VX == 2;  // FFMA2 / FADD2 path
  constexpr int RING = D + 1;
  constexpr int SLOT_BYTES = G::TILE_BYTES + NS * G::BOX_BYTES;
  constexpr int U = 2 * NG + 1;
  // UR = U: the plane loop is unrolled U times and the i2 window rotates through the registers
  // without moves; UR = 1: one copy of the body (fits the 32 KB instruction cache) and the
  // window is shifted with register moves.
  // Otherwise the loop is unrolled HR_MARCH_UNROLL times over a window of U + UR - 1 planes that
  // is shifted by UR planes once per unrolled block (2NG register moves per block, not per plane).
  constexpr int UR = HR_MARCH_ROTATE ? U : HR_MARCH_UNROLL;
  constexpr int WS = HR_MARCH_ROTATE ? U : U + UR - 1;  // window registers (planes)
  static_assert(NGA % VX == 0 && TW % VX == 0, "vector alignment");

  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* const bars = reinterpret_cast<uint64_t*>(smem_raw);  // [RING] "slot is full"
  unsigned char* const ring = smem_raw + 128;

  const int lx = threadIdx.x, ly = threadIdx.y;
  const int tid = ly * BXT + lx;
  const bool warp0 = __shfl_sync(0xffffffffu, tid >> 5, 0) == 0;  // warp-uniform, and known to be
  constexpr bool is_cart = CART;  // SinhCartesian (C25)
  const int s2 = g.P0 * g.T1;
  const ImgGeom ig{NG, g.n2, g.T1, g.P0, g.off0, plan.sph};

  // work items = (chunk of planes, tile), chunk-major
  const int ntiles = plan.ntx * plan.nty;
  const int n_long = ntiles * plan.nseg;                              // segments of plan.mseg chunks
  const int n_items = plan.ncol + (n_long - plan.ncol) * plan.mseg;   // long items, then single chunks
  const int n_part = ntiles * plan.nzc;                               // residual partials: one per (tile, chunk)
  // no more items than CTAs (small grids): every CTA has exactly one item, nothing is handed out, and
  // no atomic round trip sits at the end of the CTA's (short) life
  const bool dynamic = n_items > (int)gridDim.x;
#if HR_MARCH_PDL
  // PDL: let the next launch of the stream start its own set-up now ... -- on small grids only, where a CTA
  // lives for one short item and the next launch's start-up is worth hiding.  Where items are handed out, the
  // CTAs of the next launch would sit in the slots of those that are done while the last ones still march:
  // measured up to 30 % slower per step (profiles/r2c.md), so there the trigger is left to the end of the grid.
  const bool pdl_early = plan.pdl == 2 || (plan.pdl == 1 && !dynamic);
  if (pdl_early) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
  if (tid == 0) {
#pragma unroll
    for (int r = 0; r < RING; ++r) mbar_init(&bars[r], 1);
    mbar_fence_init();
  }
  __syncthreads();
#if HR_MARCH_PDL
  // ... and do not read or write anything the previous launch touches before it has completed
  asm volatile("griddepcontrol.wait;" ::: "memory");
#endif


  double num = 0.0, den = 0.0;
  bool bad = false;  // psi_BL + u <= 0 or NaN met at an interior point (the device flag)
  // ring position of the next plane to consume, and the parity its mbarrier completes with
  int sl = 0;
  uint32_t par = 0;
  const uint32_t bars_u32 = smem_u32(bars), ring_u32 = smem_u32(ring);
#if HR_MARCH_L2_HINTS
  const uint64_t pol_keep = l2_policy_evict_last(), pol_stream = l2_policy_evict_first();
#endif

  // ---------------- outer points: radiation condition (a2, C13) + RK combine ----------------
  // A grid-stride loop over the NG n1 n2 outer points, run by every CTA right after it has issued the
  // first TMA loads of its first item, so that its load latency hides behind theirs (on L2-resident
  // grids a CTA lives for one short item: anything serial at its end is on the critical path).
  [[maybe_unused]] auto outer_tail = [&]() {
    const int n_outer = is_cart ? g.T0 * g.T1 * g.T2 - g.n0 * g.n1 * g.n2 : g.n_o2 * g.n2;
    for (int m = blockIdx.x * NT + tid; m < n_outer; m += gridDim.x * NT) {
      int i0, i1, i2, c;
      T uc, vc, ku, kv;
      if (is_cart) {
        // C25: every ghost point is an outer point.  Shell enumeration: the 2 NG ghost planes of x2 in full,
        // then per interior plane the 2 NG ghost rows of x1 in full and the 2 NG ghost columns of x0.
        const int A = g.T0 * g.T1, ring = A - g.n0 * g.n1, nzg = 2 * NG * A;
        if (m < nzg) {
          const int pz = m / A, q = m - pz * A;
          i2 = pz < NG ? pz : g.n2 + pz;
          i1 = fast_div(q, plan.dv_T0);
          i0 = q - i1 * g.T0;
        } else {
          const int mm2 = m - nzg, pz = mm2 / ring, r = mm2 - pz * ring;
          i2 = NG + pz;
          if (r < 2 * NG * g.T0) {
            const int pr = fast_div(r, plan.dv_T0);
            i1 = pr < NG ? pr : g.n1 + pr;
            i0 = r - pr * g.T0;
          } else {
            const int r2 = r - 2 * NG * g.T0, row = r2 / (2 * NG), pc = r2 - row * (2 * NG);
            i1 = NG + row;
            i0 = pc < NG ? pc : g.n0 + pc;
          }
        }
        c = g.off0 + i0 + g.P0 * i1 + s2 * i2;
        // r = |X|, d_r f = sum_a (X_a / r) (1/h_a) d_a f, c = c_min min_a(h_a dx_a) / ds_min, from the nine
        // per-axis tables {X_a, 1/(2 dx_a h_a), c_min h_a dx_a / ds_min} (C13 on six faces)
        const int ia[3] = {i0, i1, i2};
        const int na[3] = {g.n0, g.n1, g.n2};
        const int sa[3] = {1, g.P0, s2};
        T X[3], rh[3], cw = T(0);
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
          X[ax] = a.AX[(3 * ax + 0) * a.AXS + ia[ax]];
          rh[ax] = a.AX[(3 * ax + 1) * a.AXS + ia[ax]];
          const T ca = a.AX[(3 * ax + 2) * a.AXS + ia[ax]];
          cw = (ax == 0 || ca < cw) ? ca : cw;
        }
        const T ir = T(1) / sqrt(X[0] * X[0] + X[1] * X[1] + X[2] * X[2]);
        uc = a.in_u[c];
        vc = a.in_v[c];
        T au = T(0), av = T(0);
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
          const int st = sa[ax];
          T du, dv;
          if (ia[ax] >= na[ax] + NG) {
            du = T(3) * uc - T(4) * a.in_u[c - st] + a.in_u[c - 2 * st];
            dv = T(3) * vc - T(4) * a.in_v[c - st] + a.in_v[c - 2 * st];
          } else if (ia[ax] < NG) {
            du = T(4) * a.in_u[c + st] - T(3) * uc - a.in_u[c + 2 * st];
            dv = T(4) * a.in_v[c + st] - T(3) * vc - a.in_v[c + 2 * st];
          } else {
            du = a.in_u[c + st] - a.in_u[c - st];
            dv = a.in_v[c + st] - a.in_v[c - st];
          }
          const T rad = X[ax] * ir * rh[ax];
          au += rad * du;
          av += rad * dv;
        }
        ku = -cw * (au + uc * ir);
        kv = -cw * (av + vc * ir);
      } else {
        const int pz = fast_div(m, plan.dv_o2), qo = m - pz * g.n_o2;
        i2 = NG + pz;
        const T r0 = a.RAD0[qo], r1 = a.RAD1[qo], ri = a.RADI[qo];
        if (plan.cyl) {  // C24: the list of outer positions of the plane with their stencil bits
          const int po = a.OPOS[qo];
          const int q = po & 0x0fffffff;
          const int bits = po >> 28;
          i1 = fast_div(q, plan.dv_T0);
          i0 = q - i1 * g.T0;
          c = g.off0 + i0 + g.P0 * i1 + s2 * i2;
          uc = a.in_u[c];
          vc = a.in_v[c];
          ku = radiation_k(a.in_u, c, g.P0, r0, r1, ri, bits);
          kv = radiation_k(a.in_v, c, g.P0, r0, r1, ri, bits);
        } else {
          // spherical-like: the NG columns beyond x0 at interior rows, in list order; backward d_0, centred d_1
          // (constant stencil bits: no dependent load and no branch between the loads -- on L2-resident grids
          // this loop is on the critical path of the launch)
          const int row = qo / NG;
          i0 = g.n0 + NG + (qo - row * NG);
          i1 = NG + row;
          c = g.off0 + i0 + g.P0 * i1 + s2 * i2;
          uc = a.in_u[c];
          vc = a.in_v[c];
          ku = radiation_k(a.in_u, c, g.P0, r0, r1, ri, 1);
          kv = radiation_k(a.in_v, c, g.P0, r0, r1, ri, 1);
        }
      }
      T wu, wv;
      if constexpr (LEAN) {
        T yu = T(0), yv = T(0);
        if constexpr (NEED_Y) { yu = a.y_u[c]; yv = a.y_v[c]; }  // lean stage 4: y_u / y_v point at Q
        if constexpr (PREC && RK == 4) {  // Qd from the ACC buffer, Y through y_u / y_v
          wu = rk_prec_4<T>(a.dt, ku, uc, a.acc_u[c], yu);
          wv = rk_prec_4<T>(a.dt, kv, vc, a.acc_v[c], yv);
        } else {
          wu = rk_lean<T, RK>(a.dt, ku, uc, yu);
          wv = rk_lean<T, RK>(a.dt, kv, vc, yv);
        }
        a.out_u[c] = wu;
        a.out_v[c] = wv;
        if constexpr (RK == 2 && PREC) {
          a.acc_u[c] = rk_prec_q<T>(a.dt, ku, uc, yu);
          a.acc_v[c] = rk_prec_q<T>(a.dt, kv, vc, yv);
        } else if constexpr (RK == 2) {
          a.acc_u[c] = (uc - yu) + (wu + wu);
          a.acc_v[c] = (vc - yv) + (wv + wv);
        }
      } else {
        rk_combine<T, RK>(a, c, ku, kv, uc, vc, wu, wv);
      }
      // theta reflections (spherical-like systems); rho -> -rho images of the end-face points near the axis (C24)
      const int cB = (!plan.cyl && i1 < 2 * NG) ? 2 * NG - 1 - i1 : -1;
      const int cC = (!plan.cyl && i1 >= g.n1) ? 2 * (g.n1 + NG) - 1 - i1 : -1;
      const int rr = i0 < 2 * NG ? 2 * NG - 1 - i0 : -1;
      if (!is_cart && (cB >= 0 || cC >= 0 || rr >= 0 || i2 < 2 * NG || i2 >= g.n2))
        scatter_images<T>(ig, a.out_u, a.out_v, wu, wv, i0, i1, i2, rr, cB, cC);
    }
  };
  [[maybe_unused]] bool tail_done = false;
  // The first item of a CTA is its block index; further items are handed out by an atomic counter
  // (items differ in cost: boundary tiles also write ghost images), except for the residual,
  // whose per-CTA partial sums must not depend on timing (C16: fixed reduction order).
  __shared__ int s_item;
  __shared__ double red[2][NT / 32];
  int item = blockIdx.x;
  while (item < n_items) {
    // item -> (tile, first chunk, number of chunks).  The first plan.ncol items are whole segments of
    // plan.mseg chunks, segment-major over the tiles: neighbouring tiles march up the same planes together
    // (halo rows meet in L2) and a segment primes its i2 window and starts its TMA pipeline once.  The
    // chunks of the remaining segments follow one by one, chunk-major, to even out the end of the launch.
    int tile_id, ch0, nch;
    if (item < plan.ncol) {
      const int sgi = fast_div(item, plan.dv_tiles);
      tile_id = item - sgi * ntiles;
      ch0 = sgi * plan.mseg;
      nch = min(plan.mseg, plan.nzc - ch0);
    } else {
      const int nrem = n_long - plan.ncol;
      const int rem = item - plan.ncol;
      const int cpos = fast_div(rem, plan.dv_rem);
      const int sid = plan.ncol + (rem - cpos * nrem);
      const int sgi = fast_div(sid, plan.dv_tiles);
      tile_id = sid - sgi * ntiles;
      ch0 = sgi * plan.mseg + cpos;
      nch = ch0 < plan.nzc ? 1 : 0;  // the last segment of a tile may be shorter: an empty item
      if (nch == 0) ch0 = 0;
    }
    const int zi = ch0 * plan.zc;
    const int seg = nch > 0 ? min(nch * plan.zc, g.n2 - zi) : 0;
    const int ty = fast_div(tile_id, plan.dv_ntx), tx = tile_id - ty * plan.ntx;
    const int z_begin = NG + zi, z_end = z_begin + seg;
    const int x0 = NG + tx * TW, y0 = NG + ty * BY;  // first point of the tile
    const int i0 = x0 + VX * lx, i1 = y0 + ly;
    // number of this thread's points that are interior (0..VX)
    const int nact = (i1 < g.n1 + NG && nch > 0) ? max(0, min(VX, g.n0 + NG - i0)) : 0;
    const int col = g.off0 + i0 + g.P0 * i1;  // only dereferenced if nact > 0

    // one thread feeds the ring: everything plane zz needs, into ring slot sl
    auto issue = [&](int zz, int sl) {
      const uint32_t base = ring_u32 + sl * SLOT_BYTES;
      const uint32_t bar = bars_u32 + sl * 8;
      mbar_expect_tx(bar, (uint32_t)(SWA * G::SH * sizeof(T) + NS * G::BOX_BYTES));
      const int xs = g.off0 + x0;
#if HR_MARCH_L2_HINTS
      tma_load_3d_hint(base, &mm.tile, xs - NGA, y0 - NG, zz, bar, pol_keep);
      const uint32_t sb = base + G::TILE_BYTES;
      tma_load_3d_hint(sb + ST_FRONT * G::BOX_BYTES, &mm.st[ST_FRONT], xs, y0, zz + NG, bar, pol_keep);
#pragma unroll
      for (int q = 1; q < NS; ++q)
        tma_load_3d_hint(sb + q * G::BOX_BYTES, &mm.st[q], xs, y0, zz, bar, pol_stream);
#else
      tma_load_3d(base, &mm.tile, xs - NGA, y0 - NG, zz, bar);
      const uint32_t sb = base + G::TILE_BYTES;
      tma_load_3d(sb + ST_FRONT * G::BOX_BYTES, &mm.st[ST_FRONT], xs, y0, zz + NG, bar);
#pragma unroll
      for (int q = 1; q < NS; ++q) tma_load_3d(sb + q * G::BOX_BYTES, &mm.st[q], xs, y0, zz, bar);
#endif
    };
    if (warp0 && elect_one()) {
      int sd = sl;
#pragma unroll
      for (int d = 0; d < D; ++d) {
        if (z_begin + d < z_end) issue(z_begin + d, sd);
        if (++sd == RING) sd = 0;
      }
    }
    // per-column constants
    T l00[VX], l11[VX], l22[VX], l0[VX], l1[VX], c2[VX];
    double wq[VX];
    int cB = -1, cC = -1;
    bool inplane_images = false;
#pragma unroll
    for (int j = 0; j < VX; ++j) {
      l00[j] = l11[j] = l22[j] = l0[j] = l1[j] = c2[j] = T(0);
      wq[j] = 0.0;
      if (j < nact) {
        const int q = i0 + j + g.T0 * i1;
        l00[j] = a.L00[q]; l11[j] = a.L11[q]; l22[j] = a.L22[q]; l0[j] = a.L0[q]; l1[j] = a.L1[q];
        if constexpr (RESID) wq[j] = ra.mode == 0 ? ra.W[q] : 1.0;
        if constexpr (ADVANCE) {
          c2[j] = a.C2[q];
          inplane_images |= !is_cart && i0 + j < 2 * NG;
        }
      }
    }
    if (ADVANCE && nact > 0 && !plan.cyl) {
      cB = i1 < 2 * NG ? 2 * NG - 1 - i1 : -1;
      cC = i1 >= g.n1 ? 2 * (g.n1 + NG) - 1 - i1 : -1;
      inplane_images |= (cB >= 0) || (cC >= 0);
    }

    // register window: w(k)[j] = u(i0 + j, i1, z - NG + k), k = 0..2NG, kept in p[(r + k) % U]
    // with r = (z - z_begin) % U (the plane loop is unrolled U times)
    // (packed fp32 path: one 64-bit element holds both points, so that the pair stays in an aligned
    // register pair and FFMA2 / FADD2 take it without repacking moves)
    using WT = typename std::conditional<PACKED, unsigned long long, T>::type;
    constexpr int WJ = PACKED ? 1 : VX;
    WT p[WS][WJ];
    if (nact > 0) {
#pragma unroll
      for (int k = 0; k < 2 * NG; ++k) {
        const T* src = a.in_u + col + (z_begin - NG + k) * s2;
        if constexpr (PACKED) {
          p[k][0] = *reinterpret_cast<const unsigned long long*>(src);
        } else {
          const V t = *reinterpret_cast<const V*>(src);
#pragma unroll
          for (int j = 0; j < VX; ++j) p[k][j] = t.v[j];
        }
      }
    }
    // The outer-point loop runs once per CTA, here: after the first TMA copies, the per-column factors and the
    // window priming loads have been ISSUED and before anything waits for them, so that its own load latency
    // overlaps theirs (on L2-resident grids a CTA's life is one short item: serial latencies add up to the launch).
    if constexpr (ADVANCE) {
      if (!tail_done) {
        outer_tail();
        tail_done = true;
      }
    }
    [[maybe_unused]] F2 l00p{}, l11p{}, l22p{}, l0p{}, l1p{}, c2p{};
    if constexpr (PACKED) {
      l00p = f2_pack((float)l00[0], (float)l00[VX - 1]);
      l11p = f2_pack((float)l11[0], (float)l11[VX - 1]);
      l22p = f2_pack((float)l22[0], (float)l22[VX - 1]);
      l0p = f2_pack((float)l0[0], (float)l0[VX - 1]);
      l1p = f2_pack((float)l1[0], (float)l1[VX - 1]);
      c2p = f2_pack((float)c2[0], (float)c2[VX - 1]);
    }

    const int so = ly * TW + VX * lx;                                     // in a TW x BY box
    const int to = (ly + NG) * SWA + NGA + VX * lx;                       // in the halo tile
    constexpr int NE = 2 * NGV + VX;                                      // row values a thread reads
    // Residual partials: one pair per (tile, chunk), flushed at every chunk boundary of the item and summed in
    // a fixed order (thread: planes in order; then lanes, then warps), so the result does not depend on which
    // CTA ran the chunk, when, or as part of how long an item (C16)
    [[maybe_unused]] auto flush_partial = [&](int slot) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        num += __shfl_down_sync(0xffffffffu, num, o);
        den += __shfl_down_sync(0xffffffffu, den, o);
      }
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
        ra.partials[2 * slot] = sa;
        ra.partials[2 * slot + 1] = sb;
      }
      num = 0.0;
      den = 0.0;
    };
    int cz = col + z_begin * s2;  // stored index of this thread's first point in plane z
    [[maybe_unused]] int zleft = plan.zc, pslot = tile_id * plan.nzc + ch0;  // planes left in the chunk, its partial slot
    for (int zb = z_begin; zb < z_end; zb += UR) {
#pragma unroll
      for (int r = 0; r < UR; ++r) {
        const int z = zb + r;
        if (z >= z_end) break;
#define HR_W(k) p[HR_MARCH_ROTATE ? (r + (k)) % U : r + (k)]
        __syncthreads();  // every thread is done with plane z-1: its slot can be refilled
        if (warp0 && z + D < z_end) {
          if (elect_one()) issue(z + D, sl == 0 ? RING - 1 : sl - 1);  // (sl + D) % RING
        }
        mbar_wait(bars_u32 + sl * 8, par);  // the boxes of plane z have landed
        const T* tl = reinterpret_cast<const T*>(ring + sl * SLOT_BYTES);
        const T* sb = reinterpret_cast<const T*>(ring + sl * SLOT_BYTES + G::TILE_BYTES);
        if (++sl == RING) {
          sl = 0;
          par ^= 1u;
        }
        // C25 (SinhCartesian): what depends on x2 is uniform over the plane
        T z22 = T(0), z2v = T(0), zc2 = T(0);
        double zh = 1.0;
        if (is_cart) {
          z22 = a.Z22[z];
          z2v = a.Z2[z];
          zc2 = a.ZC2[z];
          if constexpr (RESID) zh = ra.ZH[z];
        }
        if (nact > 0) {
          if constexpr (PACKED) {
            HR_W(2 * NG)[0] = *reinterpret_cast<const unsigned long long*>(sb + ST_FRONT * (TW * BY) + so);
          } else {
            const V fr = *reinterpret_cast<const V*>(sb + ST_FRONT * (TW * BY) + so);
#pragma unroll
            for (int j = 0; j < VX; ++j) HR_W(2 * NG)[j] = fr.v[j];
          }
          T e[NE];  // tile row of this thread: e[NGV + j + m] = u(i0 + j + m, i1, z)
#pragma unroll
          for (int m = 0; m < NE / VX; ++m) {
            const V t = *reinterpret_cast<const V*>(tl + to - NGV + m * VX);
#pragma unroll
            for (int j = 0; j < VX; ++j) e[m * VX + j] = t.v[j];
          }
          const V psi = *reinterpret_cast<const V*>(sb + ST_PSI * (TW * BY) + so);
          const V Ss = *reinterpret_cast<const V*>(sb + ST_S * (TW * BY) + so);
          T H[VX];
          [[maybe_unused]] F2 H2{}, uc2{};
          if constexpr (PACKED) {
            // fp32, two points per thread: the i1 and i2 stencils, the combination with the metric
            // factors, the source term and (below) the RK combine on packed pairs; the i0 stencil
            // stays per point (its neighbour pairs straddle the register pairs)
            auto L2 = [](const T* q) { return F2{*reinterpret_cast<const unsigned long long*>(q)}; };
            uc2 = F2{(unsigned long long)HR_W(NG)[0]};
            float uc_lo, uc_hi;
            f2_unpack(uc2, uc_lo, uc_hi);
            float d00s[2] = {(float)F::d2(0) * uc_lo, (float)F::d2(0) * uc_hi}, d0s[2] = {0.f, 0.f};
            F2 d11 = f2_mul(f2_bc((float)F::d2(0)), uc2), d22 = d11, d1 = f2_bc(0.f);
#pragma unroll
            for (int k = 1; k <= NG; ++k) {
              const F2 up2 = L2(tl + to + k * SWA), dn2 = L2(tl + to - k * SWA);
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                const float a0 = (float)e[NGV + j + k], b0 = (float)e[NGV + j - k];
                d00s[j] += (float)F::d2(k) * (a0 + b0);
                d0s[j] += (float)F::c1(k) * (a0 - b0);
              }
              d11 = f2_fma(f2_bc((float)F::d2(k)), f2_add(up2, dn2), d11);
              d22 = f2_fma(f2_bc((float)F::d2(k)),
                           f2_add(F2{(unsigned long long)HR_W(NG + k)[0]}, F2{(unsigned long long)HR_W(NG - k)[0]}),
                           d22);
              d1 = f2_fma(f2_bc((float)F::c1(k)), f2_sub(up2, dn2), d1);
            }
            F2 lap = f2_mul(l00p, f2_pack(d00s[0], d00s[1]));
            lap = f2_fma(l11p, d11, lap);
            lap = f2_fma(l22p, d22, lap);
            lap = f2_fma(l0p, f2_pack(d0s[0], d0s[1]), lap);
            lap = f2_fma(l1p, d1, lap);
            if (is_cart) {  // C25: the u_22 factor belongs to the plane, and there is a u_2 term
              F2 d2p = f2_bc(0.f);
#pragma unroll
              for (int k = 1; k <= NG; ++k)
                d2p = f2_fma(f2_bc((float)F::c1(k)),
                             f2_sub(F2{(unsigned long long)HR_W(NG + k)[0]}, F2{(unsigned long long)HR_W(NG - k)[0]}),
                             d2p);
              lap = f2_mul(l00p, f2_pack(d00s[0], d00s[1]));
              lap = f2_fma(l11p, d11, lap);
              lap = f2_fma(f2_bc((float)z22), d22, lap);
              lap = f2_fma(l0p, f2_pack(d0s[0], d0s[1]), lap);
              lap = f2_fma(l1p, d1, lap);
              lap = f2_fma(f2_bc((float)z2v), d2p, lap);
            }
            // (psi + u)^-7: hardware reciprocal seed per lane, Newton step and powers packed
            const F2 x = f2_add(L2(sb + ST_PSI * (TW * BY) + so), uc2);
            float x0, x1, r0, r1;
            f2_unpack(x, x0, x1);
            if constexpr (GUARD) bad |= !(x0 > 0.f) | (nact == VX & !(x1 > 0.f));
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r0) : "f"(x0));
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r1) : "f"(x1));
            F2 rr = f2_pack(r0, r1);
            const F2 nx = f2_sub(f2_bc(0.f), x);
            rr = f2_fma(rr, f2_fma(nx, rr, f2_bc(1.f)), rr);
            const F2 t2 = f2_mul(rr, rr), t4 = f2_mul(t2, t2);
            H2 = f2_fma(L2(sb + ST_S * (TW * BY) + so), f2_mul(f2_mul(t4, t2), rr), lap);
            float h0, h1;
            f2_unpack(H2, h0, h1);
            H[0] = (T)h0;
            H[VX - 1] = (T)h1;
          } else {
          T d00[VX], d11[VX], d22[VX], d0[VX], d1[VX];
#pragma unroll
          for (int j = 0; j < VX; ++j) {
            d00[j] = T(F::d2(0)) * HR_W(NG)[j];
            d11[j] = d00[j];
            d22[j] = d00[j];
            d0[j] = T(0);
            d1[j] = T(0);
          }
#pragma unroll
          for (int k = 1; k <= NG; ++k) {
            const V up = *reinterpret_cast<const V*>(tl + to + k * SWA);
            const V dn = *reinterpret_cast<const V*>(tl + to - k * SWA);
#pragma unroll
            for (int j = 0; j < VX; ++j) {
              const T a0 = e[NGV + j + k], b0 = e[NGV + j - k];
              d00[j] += T(F::d2(k)) * (a0 + b0);
              d11[j] += T(F::d2(k)) * (up.v[j] + dn.v[j]);
              d22[j] += T(F::d2(k)) * (HR_W(NG + k)[j] + HR_W(NG - k)[j]);
              d0[j] += T(F::c1(k)) * (a0 - b0);
              d1[j] += T(F::c1(k)) * (up.v[j] - dn.v[j]);
            }
          }
#pragma unroll
          for (int j = 0; j < VX; ++j) {
            T lap = l00[j] * d00[j] + l11[j] * d11[j] + l22[j] * d22[j] + l0[j] * d0[j] +
                    l1[j] * d1[j];
            if (is_cart) {  // C25: the u_22 factor belongs to the plane, and there is a u_2 term
              T d2 = T(0);
#pragma unroll
              for (int k = 1; k <= NG; ++k) d2 += T(F::c1(k)) * (HR_W(NG + k)[j] - HR_W(NG - k)[j]);
              lap = l00[j] * d00[j] + l11[j] * d11[j] + z22 * d22[j] + l0[j] * d0[j] + l1[j] * d1[j] +
                    z2v * d2;
            }
            const T x = psi.v[j] + HR_W(NG)[j];
            if constexpr (GUARD) bad |= j < nact & !(x > T(0));
            H[j] = lap + Ss.v[j] * pow_m7(x);
          }
          }
          if constexpr (RESID) {
#pragma unroll
            for (int j = 0; j < VX; ++j)
              if (j < nact) {
                const double wj = (is_cart && ra.mode == 0) ? wq[j] * zh : wq[j];
                num += wj * (double)H[j] * (double)H[j];
                den += wj;
              }
          }
          if constexpr (ADVANCE) {
            const V vin = *reinterpret_cast<const V*>(sb + ST_V * (TW * BY) + so);
            [[maybe_unused]] V yu{}, yv{}, au{}, av{};
            if constexpr (NEED_A && !PACKED) {
              au = *reinterpret_cast<const V*>(sb + S_AU * (TW * BY) + so);
              av = *reinterpret_cast<const V*>(sb + S_AV * (TW * BY) + so);
            }
            if constexpr (NEED_Y && !PACKED) {
              yu = *reinterpret_cast<const V*>(sb + S_YU * (TW * BY) + so);
              yv = *reinterpret_cast<const V*>(sb + S_YV * (TW * BY) + so);
            }

            V wu, wv, nu, nv;  // stage output and the new running sum
            if constexpr (PACKED) {
              auto L2 = [](const T* q) { return F2{*reinterpret_cast<const unsigned long long*>(q)}; };
              auto toV = [](F2 x) {
                V v;
                float lo, hi;
                f2_unpack(x, lo, hi);
                v.v[0] = (T)lo;
                v.v[VX - 1] = (T)hi;
                return v;
              };
              const F2 vin2 = L2(sb + ST_V * (TW * BY) + so);
              const F2 ku = f2_fma(f2_bc(-(float)a.eta), uc2, vin2);
              const F2 kv = f2_mul(is_cart ? f2_pack(fminf((float)c2[0], (float)zc2), fminf((float)c2[VX - 1], (float)zc2))
                                             : c2p, H2);
              F2 yu2{}, yv2{}, au2{}, av2{};
              if constexpr (NEED_A) {
                au2 = L2(sb + S_AU * (TW * BY) + so);
                av2 = L2(sb + S_AV * (TW * BY) + so);
              }
              if constexpr (NEED_Y) {
                yu2 = L2(sb + S_YU * (TW * BY) + so);
                yv2 = L2(sb + S_YV * (TW * BY) + so);
              }
              F2 wu2, wv2, nu2{}, nv2{};
              if constexpr (LEAN) {
                if constexpr (PREC && RK == 4) {
                  wu2 = rk_prec_4_f2((float)a.dt, ku, uc2, yu2, au2);
                  wv2 = rk_prec_4_f2((float)a.dt, kv, vin2, yv2, av2);
                } else {
                  wu2 = rk_lean_f2<RK>((float)a.dt, ku, uc2, yu2);
                  wv2 = rk_lean_f2<RK>((float)a.dt, kv, vin2, yv2);
                }
                if constexpr (RK == 2 && PREC) {  // Qd = (Y1 - Y) + dt k2
                  nu2 = rk_prec_q_f2((float)a.dt, ku, uc2, yu2);
                  nv2 = rk_prec_q_f2((float)a.dt, kv, vin2, yv2);
                } else if constexpr (RK == 2) {  // Q = (Y1 - Y) + 2 Y2
                  nu2 = f2_add(f2_sub(uc2, yu2), f2_add(wu2, wu2));
                  nv2 = f2_add(f2_sub(vin2, yv2), f2_add(wv2, wv2));
                }
              } else {
                rk_values_f2<RK>((float)a.dt, ku, kv, uc2, vin2, yu2, yv2, au2, av2, wu2, wv2, nu2, nv2);
              }
              wu = toV(wu2);
              wv = toV(wv2);
              nu = toV(nu2);
              nv = toV(nv2);
            } else {
#pragma unroll
              for (int j = 0; j < VX; ++j) {
                const T uc = HR_W(NG)[j];
                const T ku = vin.v[j] - a.eta * uc;
                const T kv = (is_cart ? (c2[j] < zc2 ? c2[j] : zc2) : c2[j]) * H[j];
                if constexpr (LEAN) {
                  if constexpr (PREC && RK == 4) {
                    wu.v[j] = rk_prec_4<T>(a.dt, ku, uc, yu.v[j], au.v[j]);
                    wv.v[j] = rk_prec_4<T>(a.dt, kv, vin.v[j], yv.v[j], av.v[j]);
                  } else {
                    wu.v[j] = rk_lean<T, RK>(a.dt, ku, uc, yu.v[j]);
                    wv.v[j] = rk_lean<T, RK>(a.dt, kv, vin.v[j], yv.v[j]);
                  }
                  if constexpr (RK == 2 && PREC) {  // Qd = (Y1 - Y) + dt k2
                    nu.v[j] = rk_prec_q<T>(a.dt, ku, uc, yu.v[j]);
                    nv.v[j] = rk_prec_q<T>(a.dt, kv, vin.v[j], yv.v[j]);
                  } else if constexpr (RK == 2) {  // Q = (Y1 - Y) + 2 Y2
                    nu.v[j] = (uc - yu.v[j]) + (wu.v[j] + wu.v[j]);
                    nv.v[j] = (vin.v[j] - yv.v[j]) + (wv.v[j] + wv.v[j]);
                  }
                } else {
                  rk_values<T, RK>(a.dt, ku, kv, uc, vin.v[j], yu.v[j], yv.v[j], au.v[j], av.v[j],
                                   wu.v[j], wv.v[j], nu.v[j], nv.v[j]);
                }
              }
            }
            const int c = cz;
            if (nact == VX) {
              *reinterpret_cast<V*>(a.out_u + c) = wu;
              *reinterpret_cast<V*>(a.out_v + c) = wv;
              if constexpr (WRITE_ACC) {
                *reinterpret_cast<V*>(a.acc_u + c) = nu;
                *reinterpret_cast<V*>(a.acc_v + c) = nv;
              }
            } else {
#pragma unroll
              for (int j = 0; j < VX; ++j)
                if (j < nact) {
                  a.out_u[c + j] = wu.v[j];
                  a.out_v[c + j] = wv.v[j];
                  if constexpr (WRITE_ACC) {
                    a.acc_u[c + j] = nu.v[j];
                    a.acc_v[c + j] = nv.v[j];
                  }
                }
            }
            if (!is_cart && (inplane_images || z < 2 * NG || z >= g.n2))
              scatter_vec<T, VX>(ig, a.out_u, a.out_v, wu, wv, i0, i1, z, nact, cB, cC);
          }
        }
        cz += s2;
        if constexpr (RESID) {  // a chunk of the item is complete: its partial pair
          if (--zleft == 0 || z + 1 == z_end) {
            flush_partial(pslot++);
            zleft = plan.zc;
          }
        }
#undef HR_W
      }
      if constexpr (!HR_MARCH_ROTATE) {  // shift the window by the UR planes just done
#pragma unroll
        for (int k = 0; k < 2 * NG; ++k)
#pragma unroll
          for (int j = 0; j < WJ; ++j) p[k][j] = p[k + UR][j];
      }
    }
    if (bad) *plan.flag = 1;
    if constexpr (ST == 5) {
      __syncthreads();  // red is reused by the next item
      item += gridDim.x;
    } else {
      if (!dynamic) break;
      __syncthreads();  // all threads are done with this item (and with s_item, red)
      if (tid == 0) s_item = (int)gridDim.x + atomicAdd(plan.counters + 2 * STAGE, 1);
      __syncthreads();
      item = s_item;
    }
  }
#if HR_MARCH_PDL
  // (dynamic hand-out, shared GPU) this CTA marches no more: once all have said so the next launch may move in
  if (!pdl_early) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
  // The last CTA to leave the item loop re-arms the counters for the next launch of this stage
  // and, for the residual stages, sums the item partials in a fixed order (thread t takes items
  // t, t + NT, ...; then a fixed tree), so the reduction needs no launch of its own and its
  // result does not depend on which CTA happens to be last (C16).
  if (RESID || (ST != 5 && dynamic)) {
    __shared__ int s_last;
    if (tid == 0) {
      if constexpr (RESID) __threadfence();  // this CTA's partials before its "done" tick
      s_last = atomicAdd(plan.counters + 2 * STAGE + 1, 1) == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (s_last) {
      if constexpr (RESID) {
        __threadfence();
        double sa = 0.0, sb = 0.0;
        // batches of 8 independent 16-byte loads, added in index order (latency-bound otherwise)
        const double2* pp = reinterpret_cast<const double2*>(ra.partials);
        int i = tid;
        for (; i + 7 * NT < n_part; i += 8 * NT) {
          double2 v[8];
#pragma unroll
          for (int q = 0; q < 8; ++q) v[q] = __ldcg(pp + i + q * NT);
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            sa += v[q].x;
            sb += v[q].y;
          }
        }
        for (; i < n_part; i += NT) {
          const double2 v = __ldcg(pp + i);
          sa += v.x;
          sb += v.y;
        }
        __shared__ double fin[2][NT];
        fin[0][tid] = sa;
        fin[1][tid] = sb;
        __syncthreads();
#pragma unroll
        for (int o = NT / 2; o > 0; o >>= 1) {
          if (tid < o) {
            fin[0][tid] += fin[0][tid + o];
            fin[1][tid] += fin[1][tid + o];
          }
          __syncthreads();
        }
        if (tid == 0) {
          ra.out2[0] = fin[0][0];
          ra.out2[1] = fin[1][0];
        }
      }
      if (tid == 0) {
        plan.counters[2 * STAGE] = 0;
        plan.counters[2 * STAGE + 1] = 0;
      }
    }
  }


}
