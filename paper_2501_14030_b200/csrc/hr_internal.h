// hr_internal.h -- solver object and the launcher interface between hr_api.cu (host logic) and
// hr_kernels.cu (device code).  Product code: shares nothing with oracle/.
#pragma once

#include <cuda.h>  // CUtensorMap (types only; the driver is reached through the runtime)
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/hr.h"

#define HR_MAX_NG 6

// Device-side view of one solver: everything a kernel needs, passed by value (__grid_constant__).
// The PUBLIC layout of a grid function is idx = i0 + T0 (i1 + T1 i2) (reading C8).  In HBM the
// library keeps a padded copy of that layout: point (i0,i1,i2) sits at
//     off0 + i0 + P0 (i1 + T1 i2),   P0 = row pitch >= off0 + T0,
// with P0 and off0 + NG multiples of 128 bytes, so that the first interior point of every row
// starts a 128-byte line (full-sector warp stores, aligned vector loads, TMA-legal strides).
// hr_get_u / hr_set_state / hr_eval_rhs convert between the two with k_pack / k_unpack.
struct HrGrid {
  int32_t n0, n1, n2;  // interior points
  int32_t ng;          // ghost layers = FD radius (C7)
  int32_t T0, T1, T2;  // points per axis incl. ghosts
  int32_t P0, off0;    // padded row pitch and offset of i0 = 0 within a row, in scalars
  int64_t s1, s2;      // strides of i1 and i2 in scalars (P0, P0*T1)
  int64_t npad;        // scalars per stored grid function (P0*T1*T2)
  int64_t ntot;
  int64_t n_inner;
  int32_t n_outer_cols;  // = ng: outer layers i0 in [n0+ng, T0)
  int32_t n_o2;          // outer positions of the (i0,i1) plane (HrArrays::OPOS); outer points = n_o2 * n2
};

// Pointers into the caller's workspace.  `void*` scalars are double or float per dtype.
struct HrArrays {
  void* Y[2];    // state (u, v)
  void* A[2];    // stage buffer A
  void* B[2];    // stage buffer B
  void* ACC[2];  // running RK4 sum  Y + dt/6 k1 + dt/3 k2 + dt/3 k3
  void* psi;     // psi_BL (C1)
  void* S;       // (1/8) A~_ij A~^ij (C2)
  // (i0,i1) planes, index i0 + T0 i1, working dtype (reading C4, C9, C12); FD weights are for
  // unit spacing, so the 1/dx^a and 1/(dx^a)^2 factors are folded in here.
  void* L00;  // g00 / dx0^2
  void* L11;  // g11 / dx1^2
  void* L22;  // g22 / dx2^2
  void* L0;   // g0 / dx0
  void* L1;   // g1 / dx1
  void* C2;   // c^2
  // outer radiation condition (C13), compact (ng x T1) arrays, index j + ng*i1, j = i0-(n0+ng):
  void* RAD0;  // c * rad0 / (2 dx0)
  void* RAD1;  // c * rad1 / (2 dx1)
  void* RADI;  // c / r
  // the outer positions themselves: i0 + T0 i1 in the low 28 bits, stencil bits above (hr_api.cu: HostSetup::opos);
  // RAD0 / RAD1 / RADI are indexed like this list
  int32_t* OPOS;
  // SinhCartesian (C25) only.  Per plane i2 (T2 each): Z22 = 1/(h2 dx2)^2, Z2 = -X2''/X2'^3 / dx2, ZC2 =
  // (c_min h2 dx2 / ds_min)^2 in the working dtype, ZH = h2 in fp64.  AX: nine tables of AXS scalars (working
  // dtype), for a = 0, 1, 2: X_a(i), 1/(2 dx_a h_a(i)), c_min h_a(i) dx_a / ds_min (radiation on six faces).
  void *Z22, *Z2, *ZC2, *AX;
  double* ZH;
  int32_t AXS;
  double* Wvol;  // |h0 h1 h2| plane, always fp64 (C16)
  int32_t* inner_dst;
  int32_t* inner_src;
  double* partials;  // residual partial sums: 2 doubles per block
  double* result2;   // {sum w H^2, sum w}
  // 1-D coordinate tables for the source kernel, fp64 (host libm values)
  double *rho, *rhoz;          // T0: rho(x0); sqrt(rho^2 + b^2) (SymTP) or rho (spherical)
  double *sinth, *costh;       // T1
  double *sinph, *cosph;       // T2
  double* punct;               // n_punctures x 10
};

// Tiles of the marching arrangement (hr_march.cuh): TW x BY points, VX points per thread.
// Measured on config 3 (profiles/r1b.md, r1c.md): 4-row tiles (128 threads, 5 CTAs per SM) beat
// 8-row tiles (256 threads, 2-3 CTAs) by 3-4 % -- the per-plane barrier spans fewer warps.  The
// fp64 kernels fit 96 registers without spills, so 5 CTAs per SM (4: -1 %, 6: -1 %).
#ifndef HR_TW_F64
#define HR_TW_F64 32
#define HR_BY_F64 4
#define HR_VX_F64 1
#endif
#ifndef HR_TW_F32
#define HR_TW_F32 64
#define HR_BY_F32 4
#define HR_VX_F32 2
#endif

// Minimum resident CTAs per SM the marching kernels are compiled for (register cap).
#ifndef HR_MARCH_MINB_F64
#define HR_MARCH_MINB_F64 5
#endif
#ifndef HR_MARCH_MINB_F32
#define HR_MARCH_MINB_F32 5
#endif

// 1: unroll the plane loop 2NG+1 times (rotating register window); 0: single copy + moves.
#ifndef HR_MARCH_ROTATE
#define HR_MARCH_ROTATE 0
#endif

// 1: L2 eviction hints on the TMA loads (u: evict last, pointwise inputs: evict first).  Measured
// on config 3: no gain (fp64 0.703 vs 0.706, fp32 0.611 vs 0.632), so off.
#ifndef HR_MARCH_L2_HINTS
#define HR_MARCH_L2_HINTS 0
#endif

// 1: fp32 with two points per thread uses the sm_100 packed fp32x2 instructions (FFMA2, FADD2).
#ifndef HR_MARCH_F32X2
#define HR_MARCH_F32X2 1
#endif

// 1: fp32 takes the increment-preserving ACC-free RK4 (stage codes 22 / 24: one rounding of the size of Y
// per step, stage 4 reads Y as well: 34w instead of 32w bytes per point and step); 0: the plain form.
#ifndef HR_F32_PRECISE_RK
#define HR_F32_PRECISE_RK 1
#endif

// Copies of the plane-loop body per window shift (HR_MARCH_ROTATE = 0).
#ifndef HR_MARCH_UNROLL
#define HR_MARCH_UNROLL 2
#endif

// 1: the marching kernels are launched with programmatic stream serialization (PDL) and order themselves after
// their predecessor with griddepcontrol.wait.
#ifndef HR_MARCH_PDL
#define HR_MARCH_PDL 1
#endif

// Planes of asynchronous look-ahead in the marching kernels.
#ifndef HR_MARCH_D_F64
#define HR_MARCH_D_F64 2
#endif
#ifndef HR_MARCH_D_EXTRA_LIGHT
#define HR_MARCH_D_EXTRA_LIGHT 0
#endif
#ifndef HR_MARCH_D_F32
#define HR_MARCH_D_F32 2
#endif

// hr_residual_static's scratch (a static __device__ array, one per GPU that loads the library): room for the
// launch counters and for HR_STATIC_MAX_PARTIALS work-item partial pairs = 1 MiB + 256 bytes.
#define HR_STATIC_COUNTER_BYTES 256
#define HR_STATIC_MAX_PARTIALS 65536
#define HR_STATIC_MAX_DEVICES 64

// Tiling of the marching kernels (hr_march.cuh).
struct MarchPlan {
  int ntx, nty;  // tiles along i0, i1
  int zc, nzc;   // planes per chunk, chunks along i2
  int gt;        // tiles per group (whole tile rows); items are chunk-major within a group (unused since r2)
  // Long items: a tile's column of chunks is cut into nseg segments of mseg chunks; the first ncol segments
  // (segment-major over the tiles, a whole number of waves of CTAs) are marched in one go -- one window
  // priming and one pipeline start per segment instead of per chunk -- and the chunks of the remaining
  // segments are handed out one by one, chunk-major, to even out the end.  ncol = 0, mseg = 1: chunks only.
  int mseg, nseg, ncol;
  int* counters; // device: {next item, CTAs done} per stage kernel, zero between launches
  int sph;       // 1 = SinhSpherical inner map (theta -> pi - theta under rho -> -rho)
  int cart;      // 1 = SinhCartesian (C25): u_2 term, x2-dependent factors, six outer faces, no images
  int cyl;       // 1 = SinhCylindrical (C24): x1 is axial, no theta reflections, outer points beyond its ends
  int* flag;     // device: set non-zero by a kernel that meets psi_BL + u <= 0 or NaN at an interior point
  // quotients of the work-item decode by multiplication: q = umulhi(n, mul) >> shr for 0 <= n < 2^31 (mul = 0: the
  // divisor is 1 or unused), for the divisors ntx * nty, ntx and ntx * nty * nseg - ncol; set by hrk_replan
  uint32_t dv_tiles[2], dv_ntx[2], dv_rem[2];
  uint32_t dv_o2[2], dv_T0[2];  // the same for the outer-point loop: by g.n_o2 and g.T0
  int pdl;       // programmatic-launch trigger: 1 = at entry where every CTA has one item, 0 = always after the
                 // item loop (solvers that share the GPU in hr_step_many), 2 = always at entry (HR_TUNE_PDL)
};

struct hr_solver {
  hr_params p;
  MarchPlan plan;
  int num_sms;
  int march_grid_lean[7] = {0, 0, 0, 0, 0, 0, 0};  // variant 0: the ACC-free stages, by stage % 10
  int march_grid[7];  // persistent grid size per stage kernel (0 = eval, 1..4, 5 = residual, 6 = 1 + residual)
  int march_slots[7] = {0, 0, 0, 0, 0, 0, 0};       // resident CTAs per SM x SMs, before the clamp to the work
  int march_slots_lean[7] = {0, 0, 0, 0, 0, 0, 0};
  // TMA descriptors of the ten stored grid functions (Y, A, B, ACC (u, v), psi, S): the TW x BY
  // box of each, and the halo-tile box of the three stencil sources Y_u, A_u, B_u
  CUtensorMap tm_box[10];
  CUtensorMap tm_tile[3];
  std::vector<hr_puncture> punctures;
  HrGrid g;
  HrArrays a;
  double dx[3];
  double dt, dsmin;
  int64_t n_outer;
  std::vector<int32_t> inner_dst, inner_src, outer_idx;  // host copies (hr_get_bc_lists)
  size_t scalar_bytes;
  int max_partials;
  cudaStream_t stream;
  cudaGraphExec_t step_graph;  // one RK4 step = 4 x (fused kernel, inner fill)
  cudaGraphExec_t step_resid_graph[2];  // the same with the residual fused into stage 1, per mode
  bool step_resid_tried[2] = {false, false};
  int launches_per_step;
  void* workspace;
  size_t workspace_bytes;
  // hr_relax: two pinned {num, den} slots and two events (the host tests block k-1 while block k runs),
  // and the pinned word the numeric flag is read into; created once in hr_create
  double* pinned = nullptr;
  cudaEvent_t relax_ev[2] = {nullptr, nullptr};
};

// ---- hr_kernels.cu ----
// All launchers return the cudaError_t of the launch (cudaGetLastError).
cudaError_t hrk_source(const hr_solver* s);
// stage = 1..4: fused [RHS at interior + radiation at outer] + RK combine, then inner fill of
// the array written by that stage.
cudaError_t hrk_substep(const hr_solver* s, int stage);
// the two launches of hrk_substep, separately (hr_profile_step times them one by one)
cudaError_t hrk_substep_main(const hr_solver* s, int stage);
cudaError_t hrk_substep_fill(const hr_solver* s, int stage);
// k = full Alg. 1 l.13-14 evaluation of the current state into ku, kv (N_tot each).
cudaError_t hrk_eval_rhs(const hr_solver* s, void* ku, void* kv);
// inner fill (C14) of the pair (fu, fv), stored layout
cudaError_t hrk_inner_fill(const hr_solver* s, void* fu, void* fv);
// public layout (N_tot scalars, device) <-> stored layout
cudaError_t hrk_pack(const hr_solver* s, void* dst_public, const void* src_stored);
cudaError_t hrk_unpack(const hr_solver* s, void* dst_stored, const void* src_public);
// padded row geometry for a dtype: pitch and offset in scalars
void hrk_row_geometry(int T0, int ng, size_t scalar_bytes, int* P0, int* off0);
// residual partial sums + final deterministic pass into out2_dev
cudaError_t hrk_residual(const hr_solver* s, int mode, double* out2_dev);
// hr_residual_static: the same launch (marching arrangements only) with its scratch -- the work-item partials and
// the launch counters -- in a file-scope __device__ array of hr_kernels.cu; enqueues a clear of the counters and
// the kernel, allocates nothing.  The caller has checked that the plan has at most HR_STATIC_MAX_PARTIALS items.
cudaError_t hrk_residual_static(const hr_solver* s, int mode, double* out2_dev);
// one RK4 step whose first substep also reduces the residual of the state it starts from
cudaError_t hrk_step_with_residual(const hr_solver* s, int mode, double* out2_dev);
// its first launch alone (hr_profile_step): stage 1 + residual, reduced into out2_dev
cudaError_t hrk_fused_first(const hr_solver* s, int mode, double* out2_dev);
MarchPlan hrk_make_plan(const int32_t n[3], int ng, int coord, int dtype);
// shared-memory opt-in and persistent grid sizes of the marching kernels; before graph capture
cudaError_t hrk_prepare(hr_solver* s);
int hrk_max_partials(const int32_t n[3], int ng, int dtype);
// Re-chunk the marching plan for a solver that shares the device with `share` - 1 others running at the same
// time (hr_step_many): chunk lengths and persistent grids as if 1/share of the CTA slots were its own.  share = 1
// restores the stand-alone plan.  Kernels already captured in a graph keep the plan they were captured with.
void hrk_replan(hr_solver* s, int share);
int hrk_launches_per_substep(const hr_solver* s);

// ---- hr_measure.cu ----
cudaError_t hrk_measure_alu(cudaStream_t st, int dtype, int packed, double* tflops);
cudaError_t hrk_measure_launch_floor(cudaStream_t st, int nodes, int grid, int block, int reps,
                                     double* us_per_graph);
