/* agate.h — C-ABI boundary of the B200-native AGATE finite-volume MHD step.
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md, cited P:Lnnn; readings Rn are listed in
 * DESIGN.md): one explicit Godunov-type finite-volume time step dU/dt = Delta(U,t) for the ideal
 * and Hall MHD equations (Section 3.1, eqs.7-13) on a uniform periodic Cartesian grid:
 *
 *   A0 ghost fill (periodic, 2 layers)      A4 Riemann flux: HLL eq.5-6 or HLLD (R10)
 *   A1 primitive recovery (R2)                     A5 flux difference, eq.1
 *   A2 PLM reconstruction + eq.4 limiter       A6 Runge-Kutta stage combine (RK11 ... RK53, R11/R25/R27)
 *   A3 Davis signal speeds eq.6 + fast speed eq.12 (R3)    A7 global Courant reduction dt = C dx_min / v_max
 *   A8 Hall terms: face current J, v_H = -d_i J / rho, whistler speed eq.13
 *
 * Every step of that path runs in hand-written CUDA kernels for sm_100a (fp64).  There is no CPU fallback:
 * without a CUDA device every compute entry point returns AGATE_ERR_CUDA.
 *
 * Conventions
 *   - Variable order, conserved U = (rho, mx, my, mz, E, Bx, By, Bz); all values IEEE float64.
 *   - External state layout: interior-only SoA  U[8][nz][ny][nx] (U[9]... with AGATE_IDEAL_GLM), x fastest.  Ghost
 *     padding is internal.
 *   - Every function returns an int status (AGATE_OK = 0); nothing throws or aborts; out-parameters are written
 *     only on success.
 *   - Ownership: all device memory belongs to the caller.  The library carves its two ghost-padded state
 *     buffers, its scalars and its reduction scratch out of `workspace` and never allocates device memory.
 *     Host arrays are borrowed for the duration of the call.
 *   - All work is enqueued on the stream given to agate_init.  Calls that return a value to the host
 *     (agate_compute_dt, agate_get_state to a host buffer, agate_advance with t_out != NULL, agate_step with
 *     dt_used != NULL, agate_poll) synchronise that stream; the others do not.
 *   - One context per stream; no global state; a context is not thread-safe.
 */
#ifndef AGATE_H
#define AGATE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct agate_ctx agate_ctx;   /* opaque; created by agate_init, freed by agate_destroy */

typedef struct {
  int32_t ndim;         /* 1, 2, 3: active dimensions are x[, y[, z]]  */
  int32_t nx, ny, nz;   /* interior zones; inactive dimensions must be 1                             */
  double  dx, dy, dz;   /* uniform spacings; inactive ones are ignored  */
} agate_grid;

typedef struct {
  int32_t riemann;      /* 0 = HLL (eq.5), 1 = HLLD (R10; not in the paper)              */
  int32_t limiter;      /* 0 = none (dU = 0), 1 = central (unlimited), 2 = eq.4   */
  double  beta;         /* eq.4 beta in [1,2]: 1.0 = minmod, 1.3 = the paper's "MC" default */
  int32_t rk;           /* stages: 1 = RK11 (forward Euler), 2 = SSP-RK22 (R11), 3 = SSP-RK33 (R25),
                           4 = RK43, 5 = RK53 (P:L55 names them, ref.[25]; Shu-Osher forms of R27, third order);
                           rk >= 3 needs a third state copy in the workspace                             */
  double  cfl;          /* Courant number C; <= 0 selects the paper default 0.8/0.45/0.325   */
  double  d_i;          /* normalised ion inertial length (eqset AGATE_HALL only)            */
  double  relax;        /* eqsets AGATE_CGL, AGATE_CGL_GLM: dt/(dt+tau) of eqs.32-33 in [0,1]; the paper's default is
                           0.99; 0 = no relaxation                                            */
  int32_t bc[3];        /* ghost rule per dimension (x, y, z): 0 = periodic, 1 = zero-gradient /
                           open end (R26: ghost = nearest interior zone); bc[1] = 2: the sheared
                           zero-gradient ends of the 2-D whistler test (R28: ghost (i,j) = zone (i-1,j+2)
                           at the down side, (i+1,j-2) at the up side, x periodic: needs bc[0] = 0, ndim >= 2) */
  int32_t cgl_form;     /* eqsets AGATE_CGL, AGATE_CGL_GLM: 0 = the logarithmic variable A_log of eq.18 (eqs.26-27; the paper's
                           preferred form), 1 = A of eq.16 (eqs.24-25; "AGATE supports both"): U[8] is A      */
} agate_solver;

enum { AGATE_IDEAL = 0, AGATE_HALL = 1, AGATE_CGL = 2, AGATE_IDEAL_GLM = 3, AGATE_HALL_GLM = 4, AGATE_CGL_GLM = 5 };
/* AGATE_CGL_GLM (eqs.19-23; R30): CGL MHD with GLM divergence cleaning: TEN variables per
 * cell, U = (rho, m, E, B, A, psi); AGATE_CGL's rules (relax, cgl_form, HLL only) for the first nine and
 * AGATE_IDEAL_GLM's for B_n and psi -- face values (B_n*, psi*) from the 2x2 linear Riemann problem, CGL's flux of the
 * two face states with B_n* on both sides, F[B_n] = psi*, F[psi] = c_h^2 B_n*, psi *= exp(-dt c_h^2/c_p^2) after the
 * Runge-Kutta update; c_h = 0.95 v_max with eq.28's CGL speeds. */
/* AGATE_HALL_GLM (R29): Hall MHD with GLM divergence cleaning: the nine variables and every GLM rule of
 * AGATE_IDEAL_GLM with the Hall flux (face current, v_H, whistler speed) of AGATE_HALL; HLL only. */
/* AGATE_CGL (NEXT-2; eqs.14-33; R24): CGL MHD with the logarithmic state variable of
 * eq.18.  NINE variables per cell: U = (rho, m, E, B, A_log) with E = rho v^2/2 + B^2/2 + p_par/2 + p_perp.  HLL only,
 * speeds eq.29, dt eq.28, anisotropy relaxation eqs.31-33 (C1 = 0.3, C2 = 0.5) after the Runge-Kutta update.  1-D grids
 * run through the 2-D kernel as one row that is its own periodic neighbour (exact: both y faces carry the same flux). */
/* AGATE_IDEAL_GLM (NEXT-1; eqs.10-11, constants L142; R22): ideal MHD with GLM
 * divergence cleaning.  NINE variables per cell, the scalar psi last: every U below is U[9][nz][ny][nx].  Per step
 * c_h = 0.95 v_max(U^n), c_p^2 = 0.18 c_h; face (B_n, psi) from the 2x2 linear Riemann problem; psi is multiplied by
 * exp(-dt c_h^2/c_p^2) after the Runge-Kutta update.  1-D grids run through the 2-D kernel as one row (see AGATE_CGL). */

enum { AGATE_HLL = 0, AGATE_HLLD = 1 };
enum {
  AGATE_OK = 0,
  AGATE_ERR_ARG = 1,          /* null pointer, bad size, unsupported combination (Hall + HLLD)       */
  AGATE_ERR_STATE = 2,        /* call order: no state set yet                                        */
  AGATE_ERR_UNPHYSICAL = 3,   /* rho <= 0, p <= 0 or a non-finite speed seen by the dt reduction (R14) */
  AGATE_ERR_CUDA = 4,         /* CUDA runtime error, no CUDA device, or a hand-over wait inside a kernel ran out */
  AGATE_ERR_NOMEM = 5,        /* workspace too small or misaligned                                   */
  AGATE_ERR_LIMIT = 6         /* agate_cfl_static: the grid needs more scratch than the library's static array holds */
};

/* Bytes of device workspace agate_init needs for this problem (0 on invalid arguments): two ghost-padded copies of
 * the state (three with rk >= 3), 8 or 9 variables each, plus a few hundred bytes of device scalars. */
size_t agate_workspace_bytes(const agate_grid* grid, int eqset, const agate_solver* solver);

/* Create a context.  `workspace`: DEVICE pointer, caller-owned, >= agate_workspace_bytes(), 256-byte aligned,
 * must outlive the context.  `stream`: a cudaStream_t (as void*), NULL = the legacy default stream.
 * gamma > 1 is the adiabatic index.  Hall + HLLD is rejected with AGATE_ERR_ARG (the paper gives no
 * such solver). */
int agate_init(const agate_grid* grid, double gamma, int eqset, const agate_solver* solver,
               void* workspace, size_t workspace_bytes, void* stream, agate_ctx** out);

/* Copy an interior-only SoA state U[8][nz][ny][nx] (U[9]... for AGATE_IDEAL_GLM / AGATE_HALL_GLM / AGATE_CGL, U[10]... for AGATE_CGL_GLM) into the context and set
 * the time to t0.
 * `U` is a HOST pointer when src_is_device == 0 (borrowed for the call only: the call synchronises the stream), else
 * a DEVICE pointer, read in stream order without any synchronisation: whatever produced it must be ordered before
 * this call on the context's stream (an event wait if it ran on another stream), and it must stay untouched until the
 * copy has run.  The same holds for a DEVICE destination of agate_get_state.  Fills the ghost layers (A0; per
 * solver->bc).  Validates nothing physical (the dt reduction does). */
int agate_set_state(agate_ctx*, const double* U, int src_is_device, double t0);

/* A7: dt = C dx_min / max_cells(|v| + max(c_f, c_w)) of the current state -> *dt_out (HOST).
 * Synchronises.  AGATE_ERR_UNPHYSICAL if any cell has rho <= 0, p <= 0 or a non-finite speed. */
int agate_compute_dt(agate_ctx*, double* dt_out);

/* One full time step (all RK stages: A0-A6 per stage).  dt > 0: use it; dt <= 0: run the dt reduction first and
 * use its device-resident result (no host round trip).  dt_used (HOST, may be NULL): the step actually taken;
 * non-NULL synchronises. */
int agate_step(agate_ctx*, double dt, double* dt_used);

/* n_steps self-timed steps: per step  dt = reduction(U^n); stage 1; stage 2; t += dt  — all enqueued without a
 * host synchronisation (one CUDA graph launch per step).  t_out (HOST, may be NULL): time reached; non-NULL
 * synchronises and reports AGATE_ERR_UNPHYSICAL if the reduction flagged any step. */
int agate_advance(agate_ctx*, int32_t n_steps, double* t_out);

/* Copy the current state out as interior-only SoA.  U_out is HOST (dst_is_device == 0; synchronises) or DEVICE.
 * t_out (HOST, may be NULL) receives the current time (synchronises). */
int agate_get_state(agate_ctx*, double* U_out, int dst_is_device, double* t_out);

/* Synchronise the stream and report the sticky status (AGATE_ERR_UNPHYSICAL / AGATE_ERR_CUDA / AGATE_OK). */
int agate_poll(agate_ctx*);

/* The stage kernel's launch geometry for this context: out[0..2] = grid x,y,z, out[3] = threads per block,
 * out[4] = dynamic shared memory bytes, out[5] = registers per thread, out[6] = resident blocks per SM,
 * out[7] = kernels launched per step.  For bench.py's roofline bookkeeping; no device work. */
int agate_launch_info(agate_ctx*, int64_t out[8]);

/* Accumulated device time (ms, CUDA events on the context's stream) spent in stage-kernel launches since the
 * last call with reset != 0, and the number of launches.  Only counts launches made while timing is enabled
 * with agate_set_timing(ctx, 1) (timing forces per-launch events and bypasses the CUDA graph). */
int agate_set_timing(agate_ctx*, int enabled);
int agate_stage_time(agate_ctx*, double* ms_out, int64_t* launches_out, int reset);

/* Launch tuning of one context (optional; call before stepping).  No process-wide state, no environment variables. */
typedef struct {
  int32_t stage_grid;   /* CTAs of the 2-D / 3-D stage kernel's one-wave grid; 0 = automatic (every resident slot,
                           fewer on tiny grids).  The result does not depend on it bit for bit; the tests use it to
                           reach ragged work splits.  Ignored on 1-D grids.                                       */
  int32_t no_graph;     /* != 0: agate_advance enqueues the kernels directly instead of replaying its CUDA graph  */
} agate_tuning;
int agate_set_tuning(agate_ctx*, const agate_tuning*);

/* ---- NEXT-4: slab decomposition of the grid along its last active dimension ----------------------
 * A rank holds an ordinary context over its slab (grid.nz = planes of the slab on a 3-D grid, grid.ny = rows on a 2-D
 * one) and steps it stage by stage, exchanging the two ghost layers of each cut face with its neighbours in between:
 *
 *   v = agate_get_vmax;  v = max over ranks;  agate_set_vmax(v)          (A7: one allreduce(max) of one double per step)
 *   agate_step_begin(ctx, 0)                                             dt = C dx_min / v,  t += dt,  GLM: c_h = 0.95 v
 *   for stage = 0 .. rk-1:
 *     agate_stage_pre(ctx, stage, send_lo, send_hi)    A0 on the ends that are not cut, then the two interior layers
 *                                                       next to each cut face -> the caller's DEVICE buffers
 *     (send_hi -> the upper neighbour's recv_lo,  send_lo -> the lower neighbour's recv_hi: NCCL send/recv, peer
 *      copies, or plain device copies between two contexts of one GPU)
 *     agate_stage_post(ctx, stage, recv_lo, recv_hi)   the neighbours' layers -> this slab's ghost layers, then the
 *                                                       stage kernel (A1-A6); after the last stage the step is complete
 *
 * Every zone's new value depends on the ghost-padded stage input only, so the slabs reproduce the undivided run bit
 * for bit.  A halo buffer holds [nv][2][padded plane] doubles (agate_halo_bytes; whole padded planes, so edges and
 * corners travel with them: the Hall current needs them).  All calls enqueue on the context's stream and, except
 * agate_get_vmax, do not synchronise; the buffers must stay untouched until the enqueued copies have run.
 * agate_step / agate_advance return AGATE_ERR_STATE on a context with a cut face.  Call order errors (a stage out of
 * turn, a step begun twice) return AGATE_ERR_STATE. */
int agate_set_slab(agate_ctx*, int cut_lo, int cut_hi);        /* which ends of the last active dimension are cut faces */
size_t agate_halo_bytes(const agate_ctx*);                     /* bytes of ONE halo buffer (0: 1-D grid)               */
int agate_get_vmax(agate_ctx*, double* vmax_out);              /* max_cells(|v| + c) of this slab (HOST); synchronises */
int agate_set_vmax(agate_ctx*, double vmax);                   /* the maximum over all slabs, for the next step_begin  */
int agate_vmax_device(agate_ctx*, void** ptr_out);             /* DEVICE address of that maximum (8 bytes, a positive
                                                                  double): an in-place ncclAllReduce(max) on it replaces
                                                                  the get / set pair without a host round trip.  Only on
                                                                  2-D / 3-D grids with the fused reduction (not CGL).    */
int agate_step_begin(agate_ctx*, double dt);                   /* dt > 0: use it;  dt <= 0: from the device v_max       */
int agate_stage_pre(agate_ctx*, int stage, void* send_lo, void* send_hi);
int agate_stage_post(agate_ctx*, int stage, const void* recv_lo, const void* recv_hi);

int agate_destroy(agate_ctx*);
const char* agate_strerror(int status);

/* ---- allocation-free Courant reduction (A7; R3-R5, R14) ---------------------------
 * For callers that cannot allocate device memory or hand the library a workspace (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): v_max = max over zones of (|v| + c) and dt = C dx_min / v_max
 * of a caller-owned state, with no context, no workspace and no allocation of any kind.  The reduction's scratch (one
 * partial maximum per segment of <= 1024 consecutive zones of a grid row, a ticket counter, a flag) lives in a
 * file-scope __device__ array inside the library: 256 + 8 * AGATE_STATIC_MAX_SEGMENTS bytes (about 0.5 MiB), held by
 * every GPU that loads the library until the process exits.
 *
 *   grid, gamma, eqset  as for agate_init (any equation set).  Of `solver` only cfl (<= 0: the paper's default for
 *                       the grid's dimensionality), d_i (Hall sets: the whistler speed of eq.13) and cgl_form (CGL sets)
 *                       are read.
 *   U_dev     DEVICE, read only, the caller's: interior-only SoA state U[nv][nz][ny][nx] as agate_set_state takes it
 *             (nv = 8, 9 or 10 by equation set; only the variables the speed needs are read).
 *   out_dev   DEVICE, the caller's, 3 doubles:  [0] v_max,  [1] dt,  [2] 1.0 if a zone with rho <= 0, p <= 0 or a
 *             non-finite speed was seen (such zones are left out of the maximum, R14), else 0.0.
 *   stream    cudaStream_t; one memset of the scratch header and one kernel are enqueued on it; the call does not
 *             synchronise and may be captured into a CUDA graph.
 *
 * The speeds come from the same device functions as agate_compute_dt's, and max is exact under any association: v_max
 * and dt are bit for bit those of a context holding the same state.
 * Limit: ceil(nx / 1024) * ny * nz <= AGATE_STATIC_MAX_SEGMENTS (e.g. 256^3, 8192^2; not 512^3), else AGATE_ERR_LIMIT and
 * nothing is enqueued.  Other errors: AGATE_ERR_ARG (null pointer, bad grid / gamma / eqset), AGATE_ERR_CUDA.
 * Sharing: every call on a GPU uses the one array, which keeps the previous call's contents; the call clears what must
 * start at zero and overwrites the rest before reading it.  Calls that OVERLAP on one GPU (different streams with no
 * ordering between them, or a captured graph replayed concurrently with a direct call) race on it and return garbage:
 * order them.  Different GPUs have separate copies.
 * agate_cfl_static_setup resolves the array's device address for the CURRENT device (cudaGetSymbolAddress; once per
 * device).  agate_cfl_static does that itself on first use; call the setup explicitly, once per device, before
 * capturing a graph, since the lookup may load the module. */
#define AGATE_STATIC_MAX_SEGMENTS 65536
int agate_cfl_static_setup(void);
int64_t agate_cfl_static_max_segments(void);
int agate_cfl_static(const agate_grid* grid, double gamma, int eqset, const agate_solver* solver,
                     const double* U_dev, double* out_dev, void* stream);

/* ---- diagnostics (not on the hot path) -------------------------------------------------------------- */

/* Evaluate the device Riemann flux (A3+A4[+A8]) on n independent face pairs.  All pointers are DEVICE.
 * WL, WR: [8][n] primitive face states (rho,vx,vy,vz,p,Bx,By,Bz); J: [3][n] face current (Hall) or NULL;
 * F: [8][n] output flux along `dir` (0,1,2).  Used by the GPU unit tests of the HLL/HLLD device functions. */
int agate_test_face_flux(int eqset, int riemann, int dir, double gamma, double d_i, double dxmin,
                         const double* WL, const double* WR, const double* J, double* F, int64_t n, void* stream);

/* FP64 FMA throughput micro-benchmark (8 independent DFMA chains per thread on every SM): returns the sustained
 * TFLOP/s (FMA = 2 flop) over `iters` launches in *tflops_out.  Gives the ALU roofline denominator, which
 * MEASURED_PEAKS.json does not hold.  `scratch`: >= 8 bytes of the caller's DEVICE memory (the library allocates
 * none). */
int agate_measure_fp64_peak(int iters, double* tflops_out, void* scratch, void* stream);

#ifdef __cplusplus
}
#endif
#endif
