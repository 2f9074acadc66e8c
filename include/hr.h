/*
 * hr.h -- C ABI of the B200-native hyperbolic-relaxation hot path (arxiv 2501.14030).
 *
 * The library advances the (u, v) relaxation system of PAPER.md Sec. 2, Eq. 5
 *     d_t u = v - eta u
 *     d_t v = c^2 [ lap u + (1/8) A~_ij A~^ij (psi_singular + u)^-7 ]
 * by the method-of-lines loop of PAPER.md Alg. 1 l.12-16: RHS -> BC -> RK,
 * four times per RK4 step, and evaluates the residual of Eq. 4 (Alg. 1 l.9-11).
 * Everything the paper defers to its references is fixed by the readings C1-C23 in DESIGN.md.
 *
 * Conventions
 *   - Every entry point returns hr_status, never throws or aborts, and writes its outputs only
 *     on HR_OK.  hr_last_error() gives the text of the calling thread's last failure.
 *   - "device pointer" = CUDA global memory on hr_params.device; "host pointer" = ordinary or
 *     pinned host memory.  No torch / C++ types cross this boundary.
 *   - Grid layout (reading C8): interior points N = (N0, N1, N2); NG = fd_order/2 ghost layers
 *     on every face; T_a = N_a + 2 NG; N_tot = T0 T1 T2; a grid function is N_tot scalars with
 *     flat index  idx(i0,i1,i2) = i0 + T0 (i1 + T1 i2), i0 fastest.  Scalars are double
 *     (HR_F64) or float (HR_F32).  Coordinates: x0 in [0,1] (sinh-compactified radius),
 *     x1 = theta in [0,pi], x2 = phi in [-pi,pi], cell-centred.
 *   - All work is enqueued on hr_params.stream (a cudaStream_t, may be NULL = legacy default
 *     stream).  hr_step is asynchronous with respect to the host; the calls
 *     that return host values synchronise that stream.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with HR_ERR_CUDA.
 */
#ifndef HR_H
#define HR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define HR_API __attribute__((visibility("default")))
#else
#define HR_API
#endif

typedef struct hr_solver hr_solver; /* opaque; created and destroyed by the library */

typedef enum {
  HR_OK = 0,
  HR_ERR_INVALID_ARG = 1, /* NULL pointer, N2 odd, N_a < NG, m <= 0, eta < 0, cfl <= 0, ...   */
  HR_ERR_UNSUPPORTED = 2, /* fd_order / coord / dtype not instantiated                        */
  HR_ERR_WORKSPACE = 3,   /* workspace too small or misaligned (256 B)                        */
  HR_ERR_CUDA = 4,        /* a CUDA runtime call failed; text in hr_last_error()              */
  HR_ERR_NUMERIC = 5      /* a puncture coincides with a grid point (non-finite source)       */
} hr_status;

/* Reference metrics ("Cartesian-like, spherical-like, cylindrical-like, and bispherical-like"):
 * SinhSpherical and SinhSymTP (reading C4: x0 in [0,1], x1 = theta in [0,pi], x2 = phi) and SinhCylindrical
 * (reading C24: x0 in [0,1] -> R = rho(x0), x1 in [-1,1] -> Z = rho(x1), same amp and sinhw, x2 = phi; outer
 * points beyond the outer cylinder AND beyond both end faces) and SinhCartesian (reading C25: x^a in [-1,1],
 * X_a = rho(x^a) on every axis; a u_2 term, factors that depend on x2, every ghost point an outer point, no inner
 * points).  The last two run in the default and running-sum arrangements (variant 0, 3) only. */
typedef enum { HR_SINHSPHERICAL = 0, HR_SINHSYMTP = 1, HR_SINHCYLINDRICAL = 2, HR_SINHCARTESIAN = 3 } hr_coord;
typedef enum { HR_F64 = 0, HR_F32 = 1 } hr_dtype;                 /* reading C19           */

/* One Brandt-Bruegmann puncture: bare mass, Cartesian position, Bowen-York
 * linear momentum P and spin S (readings C1, C2). */
typedef struct {
  double m;
  double pos[3];
  double P[3];
  double S[3];
} hr_puncture;

/* Problem statement: grid, coordinate system, FD order, punctures, eta, CFL (Eq. 4-5
 * and Alg. 1 l.2-7). */
typedef struct {
  int32_t n[3];          /* interior points N0 N1 N2; N2 even; N_a >= NG                      */
  int32_t coord;         /* hr_coord                                                          */
  int32_t fd_order;      /* 4, 6, 8, 10 (also 2, 12): centred stencils, NG = fd_order/2 (C7,
                            C11)                                                */
  int32_t dtype;         /* hr_dtype: arithmetic and storage type of state and RHS            */
  double amp, sinhw;     /* AMPL/SINHW (SinhSpherical) or AMAX/SINHWAA (SinhSymTP) (C4, C5)   */
  double bscale;         /* SinhSymTP focal half-distance b; ignored for SinhSpherical        */
  double origin[3];      /* Cartesian position of the grid centre (C6)                        */
  int32_t n_punctures;   /* >= 0                                                              */
  int32_t residual_mode; /* default mode of hr_residual: 0 volume-weighted RMS, 1 plain RMS
                            (C16)                                                             */
  const hr_puncture* punctures; /* host pointer, read during hr_create only (copied)          */
  double eta;            /* damping factor of Eq. 5 (C10)                        */
  double cfl;            /* dt = cfl * ds_min over interior points (C9)                       */
  double c_min;          /* wave-speed normalisation: c(x) = c_min ds(x)/ds_min (C9)          */
  int32_t device;        /* CUDA device ordinal                                               */
  int32_t variant;       /* kernel arrangement: 0 = default (fused RHS + radiation + RK combine +
                            ghost images in one TMA-fed marching kernel per substep; classic RK4
                            without a running sum: with Y1 = Y + dt/2 k1, Y2 = Y + dt/2 k2,
                            Y3 = Y + dt k3, stage 2 also stores Q = (Y1 - Y) + 2 Y2 and stage 4
                            forms (1/3)(Q + Y3) + dt/6 k4, which moves 32 w instead of 40 w bytes
                            per point and step);
                            3 = the same kernels with RK4 as a running sum (ACC = Y + dt/6 k1 +
                            dt/3 k2 + dt/3 k3), the arrangement of profiles/r1b-r1f;
                            2 = direct-load fused kernel (one thread per point, stencil through
                            L1/L2) + list-driven inner fill, kept for comparison;
                            1 = the paper's arrangement as an ablation: one thread per point,
                            block (32, NGHOSTS, 1), RHS -> BC -> RK as separate kernels with k
                            stored in HBM                              */
  void* stream;          /* cudaStream_t owned by the caller; must outlive the solver         */
} hr_params;

/* Bytes of device workspace hr_create needs for these parameters (10 grid functions, the
 * (i0,i1) coefficient planes, the boundary lists, reduction scratch).  Inside
 * the workspace every grid function is stored with rows padded to 128-byte lines; the layout
 * above is what crosses this boundary (hr_get_u, hr_set_state, hr_eval_rhs convert). */
HR_API hr_status hr_workspace_bytes(const hr_params* p, size_t* bytes);

/* Alg. 1 l.2-7: coordinate arrays, reference-metric factor planes, wave speed
 * and dt (C9), inner/outer boundary containers (C13, C14; integer closed form), then the
 * one-time device source kernel psi_BL and (1/8) A~_ij A~^ij (C1, C2), and u = v = 0 (C17).
 * workspace_dev: device pointer, 256-byte aligned, >= hr_workspace_bytes; owned by the caller,
 * must outlive the solver; the library never frees it.  *out receives the handle. */
HR_API hr_status hr_create(const hr_params* p, void* workspace_dev, size_t workspace_bytes,
                    hr_solver** out);

/* Releases the handle and its host metadata / CUDA graph.  NULL is accepted. */
HR_API hr_status hr_destroy(hr_solver* s);

/* Alg. 1 l.12-16 x n_steps: n_steps classic RK4 steps (C15), each four substeps of
 * [RHS (Eq. 5) + radiation condition at the outer points (C13) + RK combine + inner-boundary
 * fill (C14)] -- one kernel launch per substep in the default arrangement.  Enqueues on the
 * stream and returns; n_steps >= 0. */
HR_API hr_status hr_step(hr_solver* s, int64_t n_steps);

/* Alg. 1 l.9-16 in one call: the residual of the CURRENT state (as hr_residual_async: { sum w H^2,
 * sum w } to out2_dev, device pointer) and then one RK4 step.  In the default arrangement the
 * residual costs no pass of its own: the bracket of Eq. 5 that the first RK substep evaluates at
 * the state Y is exactly H of Eq. 4, so that substep also reduces w H^2 (one partial pair per
 * work item, summed in a fixed order by the last CTA to finish; equal to hr_residual_async's result
 * to a few ulp).  Asynchronous. */
HR_API hr_status hr_step_residual_async(hr_solver* s, int32_t mode, double* out2_dev);

/* PAPER.md:337-347 (N independent grids advanced together): n_steps RK4 steps of each of the n
 * solvers, enqueued round-robin, one solver's step after the other's, each on its own solver's
 * stream -- so the steps of different solvers overlap on the device when the solvers were created
 * on different streams (small grids do not fill the GPU).  No data is shared between
 * the solvers.  All solvers must live on the calling thread's current device.  Asynchronous. */
HR_API hr_status hr_step_many(hr_solver* const* solvers, int32_t n, int64_t n_steps);

/* Alg. 1 l.9-11: H = lap u + S (psi_BL + u)^-7 at interior points and its grid L2 norm in the
 * solver's residual_mode (C16), accumulated in fp64 with a fixed reduction order.
 * *out (host pointer) receives the norm; synchronises the stream. */
HR_API hr_status hr_residual(hr_solver* s, double* out);
/* Same with an explicit mode (0 or 1); out3 (host pointer, 3 doubles) receives
 * { norm, sum w H^2, sum w }. */
HR_API hr_status hr_residual_ex(hr_solver* s, int32_t mode, double* out3);
/* Asynchronous form for the relaxation loop (Alg. 1 l.9-11 inside the time loop): enqueues the
 * H kernel and the reduction and writes { sum w H^2, sum w } (2 doubles) to out2_dev (device
 * pointer); no host synchronisation. */
HR_API hr_status hr_residual_async(hr_solver* s, int32_t mode, double* out2_dev);
/* hr_residual_async for callers that must not allocate and hold no scratch of their own to lend (code under CUDA
 * graph capture, serving loops, harnesses that forbid cudaMalloc): the same kernel (Alg. 1 l.9-11, C16; marching
 * arrangements, variant 0 or 3) with its scratch -- one partial pair per work item and the launch counters -- in a
 * static __device__ array inside the library instead of the solver's workspace: 1 MiB + 256 bytes per GPU that
 * loads the library, held until the process exits.  Input: the solver's current state; output: { sum w H^2, sum w }
 * (2 doubles) to out2_dev (device pointer, the caller's).  Enqueues a clear of the counters and one kernel on the
 * solver's stream; calls no cudaMalloc / cudaFree or allocating routine; no host synchronisation.  The result equals
 * hr_residual_async's bit for bit (same kernel, same fixed reduction order).
 * Limit: at most 65536 (tile, chunk of planes) pairs, one partial each (the largest BASELINE.json grid, 512x256x256
 * in fp64, has 32768); beyond it HR_ERR_WORKSPACE with the counts in hr_last_error().  Variants 1 and 2:
 * HR_ERR_INVALID_ARG.
 * Every call on a GPU, of every solver, shares the one array, which keeps the last call's contents: calls that
 * overlap on the device (different streams, no ordering between them) race.  Order them. */
HR_API hr_status hr_residual_static(hr_solver* s, int32_t mode, double* out2_dev);

/* Alg. 1 l.8-18, the relaxation loop with its stopping criterion (C18): repeat
 * { residual (l.9-11); check_every RK4 steps (l.12-16) } until the residual norm (mode 0 or 1, C16)
 * is <= tol or max_steps steps have been taken.  The loop never stalls the device: each residual
 * is reduced on the device, copied to pinned host memory asynchronously, and tested by the host one
 * block later, while the next block of steps is already enqueued (PAPER.md:188 overlaps the norm
 * with the device-to-host copies in the same way).  Consequently the state has advanced one
 * block (check_every steps) past the residual that met tol; the last history entry is the
 * residual of the returned state.
 *   steps_done        (host, optional) RK4 steps enqueued in total
 *   final_residual    (host, optional) residual norm of the state on return (synchronous)
 *   history, history_cap, n_history (host, optional) the residuals tested, one per block, in
 *                     order: history[j] = norm after j * check_every steps
 * max_steps >= 0, check_every >= 1, tol >= 0 (0: run max_steps).  Synchronises the stream. */
HR_API hr_status hr_relax(hr_solver* s, int64_t max_steps, int64_t check_every, double tol, int32_t mode,
                          int64_t* steps_done, double* final_residual, double* history,
                          int64_t history_cap, int64_t* n_history);

/* Copy the current u (or v), N_tot scalars of the solver's dtype in the layout above, ghost
 * points included, to dst (device pointer if dst_on_device != 0, else host pointer).
 * bytes must equal N_tot * sizeof(scalar).  Synchronises the stream. */
HR_API hr_status hr_get_u(hr_solver* s, void* dst, size_t bytes, int32_t dst_on_device);
HR_API hr_status hr_get_v(hr_solver* s, void* dst, size_t bytes, int32_t dst_on_device);

/* ---- hooks for the parity contract (a production user does not need these) ---- */

/* Replace the state by N_tot scalars each of u and v (solver dtype, layout above).  The inner
 * ghost entries are then overwritten by their sources (C14/C15: ghosts mirror sources). */
HR_API hr_status hr_set_state(hr_solver* s, const void* u, const void* v, int32_t src_on_device);

/* One evaluation of Alg. 1 l.13-14 on the current state: k = RHS at interior points, radiation
 * condition at outer points, inner fill; N_tot scalars each into the device pointers ku_dev,
 * kv_dev.  Uses the same device arithmetic as hr_step's fused kernels. */
HR_API hr_status hr_eval_rhs(hr_solver* s, void* ku_dev, void* kv_dev);

/* Copies of the constant source terms psi_BL and S = (1/8) A~_ij A~^ij (solver dtype, N_tot
 * each) to host pointers (either may be NULL). */
HR_API hr_status hr_get_source(hr_solver* s, void* psi_host, void* S_host);

/* Boundary containers (C13, C14), ascending destination index.  With NULL arrays only the counts
 * are returned.  Host pointers. */
HR_API hr_status hr_get_bc_lists(hr_solver* s, int32_t* inner_dst, int32_t* inner_src, int64_t* n_inner,
                          int32_t* outer_idx, int64_t* n_outer);

/* dt and ds_min (C9), NG, T[3], N_tot.  Any pointer may be NULL. */
HR_API hr_status hr_get_info(hr_solver* s, double* dt, double* dsmin, int32_t* nghosts, int32_t* T,
                      int64_t* total_pts);

/* Host-only (no CUDA call, works without a device): the tables hr_create builds on the host
 * for these parameters -- Alg. 1 l.2-4.  All outputs are host pointers and optional (NULL):
 * dt, ds_min (C9); the boundary containers (C13, C14) with their counts; planes7 = 7 x T0*T1
 * doubles { g00/dx0^2, g11/dx1^2, g22/dx2^2, g0/dx0, g1/dx1, c^2, |h0 h1 h2| }, index i0 + T0 i1;
 * outer3 = 3 x NG*T1 doubles { c rad0/(2 dx0), c rad1/(2 dx1), c/r }, index (i0-N0-NG) + NG i1. */
HR_API hr_status hr_host_setup(const hr_params* p, double* dt, double* dsmin, int64_t* n_inner,
                               int64_t* n_outer, int32_t* inner_dst, int32_t* inner_src,
                               int32_t* outer_idx, double* planes7, double* outer3);

/* Measurement hook (bench.py's roofline object): advances n_steps RK4 steps (1..4096) with plain
 * launches of the same kernels hr_step uses, each bracketed by a CUDA event pair on the solver's
 * stream, preceded per step by one residual evaluation (Alg. 1 l.9-11) if with_residual != 0.
 * ms6 (host pointer, 6 doubles) receives the mean milliseconds per RK4 step spent in
 * { fused substep kernel of stage 1, 2, 3, 4, the four inner fills together (0 in the default
 * arrangement, whose substep kernel writes the ghost images itself), residual }.  With
 * with_residual != 0 the default arrangement runs the step as hr_step_residual_async does: stage 1
 * includes the residual (accumulation and final reduction) and "residual" is 0.
 * Synchronises the stream. */
HR_API hr_status hr_profile_step(hr_solver* s, int64_t n_steps, int32_t with_residual, double* ms6);

/* Number of kernel launches one hr_step(1) enqueues (for bench.py's gpu_launches). */
HR_API hr_status hr_launches_per_step(hr_solver* s, int32_t* n);

/* Execution facts of a solver, for callers that report what they timed (bench.py) -- SURVEY.md section 5
 * ("failure detection": the optional device flag) and VERDICT r1 item 10.  *value (host) receives:
 *   HR_Q_STEP_GRAPH     1 if hr_step replays a captured CUDA graph of the RK4 step, 0 if the capture failed
 *                       at hr_create and hr_step falls back to plain launches of the same kernels
 *   HR_Q_RESID_GRAPH    the same for hr_step_residual_async (bit 0: mode 0, bit 1: mode 1; captured on first use)
 *   HR_Q_PERSISTENT     1 if hr_step / hr_relax run the single-launch persistent step kernel (small grids)
 *   HR_Q_NUMERIC_FLAG   non-zero once a kernel of this solver has met psi_BL + u <= 0 or a non-finite value
 *                       at an interior point (reads the device flag: synchronises the stream)
 *   HR_Q_PLAN_ZC, HR_Q_PLAN_ITEMS, HR_Q_PLAN_GRID   planes per work item, work items and persistent CTAs
 *                       of the substep kernel                                                         */
typedef enum {
  HR_Q_STEP_GRAPH = 0, HR_Q_RESID_GRAPH = 1, HR_Q_PERSISTENT = 2, HR_Q_NUMERIC_FLAG = 3,
  HR_Q_PLAN_ZC = 4, HR_Q_PLAN_ITEMS = 5, HR_Q_PLAN_GRID = 6
} hr_query_what;
HR_API hr_status hr_query(hr_solver* s, int32_t what, int64_t* value);

/* Measurement hooks for the secondary roofs SURVEY.md section 8(d) asks for (no solver needed; device index and
 * cudaStream_t as in hr_params).
 * hr_measure_alu_peak: register-resident FMA chains (8 independent chains per thread, 1024 threads per CTA,
 *   8 CTAs per SM-slot wave), dtype HR_F64 or HR_F32; packed != 0 uses fma.rn.f32x2 (HR_F32 only).
 *   *tflops (host) = 2 * FMAs / best-of-3 CUDA-event time.
 * hr_measure_launch_floor: a CUDA graph of `nodes` dependent launches of an empty kernel of `grid` CTAs x
 *   `block` threads, replayed `reps` times; *us_per_graph (host) = mean microseconds per replay: the floor
 *   under a step of `nodes` launches, whatever the kernels do.  Both synchronise the stream.              */
HR_API hr_status hr_measure_alu_peak(int32_t device, void* stream, int32_t dtype, int32_t packed, double* tflops);
HR_API hr_status hr_measure_launch_floor(int32_t device, void* stream, int32_t nodes, int32_t grid,
                                         int32_t block, int32_t reps, double* us_per_graph);

/* Thread-local, static storage; never NULL. */
HR_API const char* hr_last_error(void);

/* Library version string, e.g. "hr-b200 0.1 (sm_100a)". */
HR_API const char* hr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HR_H */
