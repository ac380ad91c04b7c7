/* agate_ref.h — C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded restatement of the hot path of AGATE (Bard & Dorelli,
 * arXiv 2503.20899): one explicit Godunov-type finite-volume step for ideal / Hall MHD on a
 * uniform periodic Cartesian grid (§2.2, §3.1).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 * It shares no code, header or table with the CUDA path; these declarations are its own.
 *
 * All arrays are HOST memory, float64, interior-only SoA  U[8][nz][ny][nx]  (x fastest), variable
 * order U = (rho, mx, my, mz, E, Bx, By, Bz), W = (rho, vx, vy, vz, p, Bx, By, Bz).
 * Every function returns 0 on success or a positive status (1 bad argument, 2 call order,
 * 3 unphysical state, 5 out of memory).
 */
#ifndef AGATE_REF_H
#define AGATE_REF_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct agate_ref_ctx agate_ref_ctx;

typedef struct {
  int32_t ndim;          /* 1,2,3: active dimensions x[,y[,z]] */
  int32_t nx, ny, nz;    /* interior zones; inactive dims must be 1 */
  double  dx, dy, dz;    /* uniform spacings */
} agate_ref_grid;

typedef struct {
  int32_t riemann;       /* 0 HLL (eq.5), 1 HLLD */
  int32_t limiter;       /* 0 none (dW=0), 1 central (unlimited), 2 eq.4 */
  double  beta;          /* eq.4 beta: 1.0 = minmod, 1.3 = paper default "MC" */
  int32_t rk;            /* 1 = RK11 (forward Euler), 2 = SSP-RK2 (R11), 3 = SSP-RK33 (R25), 4 = RK43, 5 = RK53 (R27) */
  double  cfl;           /* Courant C; <=0 -> paper default 0.8/0.45/0.325 (L73) */
  double  d_i;           /* normalised ion inertial length (Hall) */
  double  relax;         /* CGL: dt/(dt+tau) of eqs.32-33 (paper default 0.99, L254); 0 = no relaxation */
  int32_t bc[3];         /* per dimension: 0 periodic, 1 zero-gradient (open end, L314: ghost = nearest interior zone);
                            bc[1] = 2: sheared zero-gradient ends in y (L314, R28), x periodic */
  int32_t cgl_form;      /* CGL: 0 = logarithmic A of eq.18 (eqs.26-27; the paper's preferred form), 1 = A of eq.16 (eqs.24-25) */
} agate_ref_solver;

enum { AGATE_REF_IDEAL = 0, AGATE_REF_HALL = 1, AGATE_REF_CGL = 2, AGATE_REF_IDEAL_GLM = 3, AGATE_REF_HALL_GLM = 4, AGATE_REF_CGL_GLM = 5 };
/* AGATE_REF_CGL_GLM (eqs.19-23; R30): CGL MHD with the GLM scalar: ten variables,
 * U = (rho, m, E, B, A, psi); CGL's rules for the first nine, IDEAL_GLM's (B_n*, psi*) face rule, fluxes and source
 * for B_n and psi (index 9), c_h = 0.95 v_max with eq.28's CGL speeds. */
/* AGATE_REF_HALL_GLM (R29): Hall MHD with the GLM scalar: the nine variables and every GLM rule of
 * AGATE_REF_IDEAL_GLM, the Hall flux (face current, v_H, whistler speed) of AGATE_REF_HALL; HLL only. */
/* AGATE_REF_CGL (R24): 9 variables, U = (rho, m, E, B, A_log) with eq.18's A_log,
 * W = (rho, v, p_par, B, p_perp); fluxes eqs.19-22 + eq.17, HLL only, speeds eq.29, dt eq.28, relaxation eqs.31-33
 * after the Runge-Kutta update. */
/* AGATE_REF_IDEAL_GLM (eqs.10-11; R22): 9 variables per cell, the GLM scalar psi
 * last: U[9][nz][ny][nx].  c_h = 0.95 v_max(U^n) per step, c_p^2 = 0.18 c_h; face (B_n, psi) from the 2x2
 * linear Riemann problem; psi <- psi exp(-dt c_h^2/c_p^2) after the Runge-Kutta update. */

/* ---- the stepping interface (mirrors the product's C-ABI on host memory) ---- */
int agate_ref_create(const agate_ref_grid*, double gamma, int eqset, const agate_ref_solver*, agate_ref_ctx** out);
int agate_ref_set_state(agate_ref_ctx*, const double* U, double t0);
int agate_ref_compute_dt(agate_ref_ctx*, double* dt_out);                 /* A7: C dx_min / v_max      */
int agate_ref_step(agate_ref_ctx*, double dt, double* dt_used);           /* dt<=0: compute_dt first   */
int agate_ref_advance(agate_ref_ctx*, int32_t n_steps, double* t_out);    /* n self-timed steps (R20)  */
int agate_ref_get_state(agate_ref_ctx*, double* U_out, double* t_out);
int agate_ref_rhs(agate_ref_ctx*, double* L_out);                         /* L(U) of eq.1, interior SoA */
int agate_ref_vmax(agate_ref_ctx*, double* vmax_out);                     /* max_i(|v_i|+c_i) (L156)    */
void   agate_ref_cgl_cons_to_prim(const double U[9], double W[9]);                      /* eqs.26-27 */
void   agate_ref_cgl_prim_to_cons(const double W[9], double U[9]);                      /* L166, eq.18 */
double agate_ref_cgl_cfast(int dir, const double W[9]);                                 /* eq.29 (+) */
void   agate_ref_cgl_face_flux(int dir, const double WL[9], const double WR[9], double F[9]);
void   agate_ref_cgl_relax(double f, double B2, double* p_par, double* p_perp);         /* eqs.31-33 */
void   agate_ref_cgl_cons_to_prim_form(int form, const double U[9], double W[9]);       /* form 1: eqs.24-25 */
void   agate_ref_cgl_prim_to_cons_form(int form, const double W[9], double U[9]);       /* form 1: eq.16 */
void   agate_ref_cgl_face_flux_form(int form, int dir, const double WL[9], const double WR[9], double F[9]);
int agate_ref_nvar(agate_ref_ctx*);                                       /* 8, or 9 with GLM          */
int agate_ref_glm_ch(agate_ref_ctx*, double* ch_out);                     /* c_h of the last step / rhs */
void agate_ref_glm_face(double ch, double bnL, double bnR, double psL, double psR, double* bn_star, double* psi_star);
int agate_ref_destroy(agate_ref_ctx*);
void agate_ref_set_threads(int n);      /* OpenMP build only: 0/1 = serial; results are bitwise identical */
int  agate_ref_get_threads(void);

/* ---- point functions, exported so that each formula can be pinned on its own ---- */
void   agate_ref_cons_to_prim(double gamma, const double U[8], double W[8]);           /* A1 */
void   agate_ref_prim_to_cons(double gamma, const double W[8], double U[8]);
double agate_ref_slope(int limiter, double beta, double dp, double dm);                /* eq.4 */
double agate_ref_cfast(int dir, double gamma, const double W[8]);                      /* eq.12 (R3) */
double agate_ref_cwhistler(double d_i, double dxmin, const double W[8]);               /* eq.13 */
void   agate_ref_phys_flux(int dir, double gamma, const double W[8], const double vH[3], double F[8]); /* eqs.7-10 */
/* Riemann flux at one face with normal `dir` (0,1,2). J may be NULL (ideal). */
void   agate_ref_face_flux(int eqset, int riemann, int dir, double gamma, double d_i, double dxmin,
                           const double WL[8], const double WR[8], const double J[3], double F[8]);
/* which HLLD branch was taken for this pair: 0 left-supersonic, 1 L*, 2 L**, 3 R**, 4 R*, 5 right-supersonic,
   +10 if a degenerate guard fired */
int    agate_ref_hlld_branch(int dir, double gamma, const double WL[8], const double WR[8]);

/* ---- algorithmic operation counts (Counted<double> instantiation of the same templates) ----
 * Runs ONE full step (dt reduction + all RK stages) on the given state and returns per-category
 * counts: out[0]=add/sub, out[1]=mul, out[2]=div, out[3]=sqrt, out[4]=compare/min/max. */
int agate_ref_count_ops(const agate_ref_grid*, double gamma, int eqset, const agate_ref_solver*,
                        const double* U, double out[5]);

#ifdef __cplusplus
}
#endif
#endif
