// agate.cu — C-ABI of the B200-native AGATE finite-volume MHD step (see include/agate.h).
// Host side only: argument checks, workspace carving, kernel selection, launches, the per-step CUDA graph.
// All arithmetic of the path is in agate_kernels.cuh / agate_physics.cuh.  No CPU fallback.
#include "agate.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "agate_kernels.cuh"
#include "agate_stage2d.cuh"
#include "agate_stage3d.cuh"

using namespace agate;

#ifndef AGATE_TY3
#define AGATE_TY3 11    // 3-D tile height: 11 owner warps + 1 helper = 12 warps (3 per scheduler, <= 168 registers), 162 KB.
                        // Measured at 512^3 (profiles/r2_stage3d.md): TY = 15 (16 warps, 128 registers, no spills) 32.9 ms
                        // per step, TY = 12 (13 warps, 128 registers) 35.2, TY = 11 31.5
#endif
#ifndef AGATE_TY3N
#define AGATE_TY3N 11   // ... with nine variables (GLM, CGL): 182 KB
#endif
#ifndef AGATE_TY3X
#define AGATE_TY3X 11   // ... with ten variables (CGL + GLM): 202 KB
#endif
#ifndef AGATE_MINB3
#define AGATE_MINB3 1
#endif

namespace {

constexpr int TY3 = AGATE_TY3;   // 3-D tile height (rows); CTA = 32 x (TY3+1) threads (agate_stage3d.cuh)
constexpr int TY3N = AGATE_TY3N;
constexpr int TY3X = AGATE_TY3X;
constexpr int TY2 = 6;    // 1-D / 2-D: 32x6 tile, 8 warps, 2 CTAs / SM
constexpr int kDtBlocksMax = 148 * 8;

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Layout {
  int ghy, ghz, nxp, nyp, nzp;
  long long sy, sz, sq;
  size_t state_bytes;      // one padded copy of U (8 variables)
  size_t off_A, off_B, off_C, off_scal, off_partial, total;   // off_C: third copy, SSP-RK33 only
};

Layout make_layout(const agate_grid& g, int nv, int rk = 2) {
  Layout L;
  L.ghy = (g.ndim >= 2) ? 2 : 0;
  L.ghz = (g.ndim >= 3) ? 2 : 0;
  L.nxp = g.nx + 4;
  L.nyp = g.ny + 2 * L.ghy;
  L.nzp = g.nz + 2 * L.ghz;
  L.sy = L.nxp;
  L.sz = (long long)L.nxp * L.nyp;
  L.sq = L.sz * L.nzp;
  L.sq = (long long)align_up((size_t)L.sq, 32);          // every variable starts 256-byte aligned
  L.state_bytes = sizeof(double) * (size_t)nv * (size_t)L.sq;
  L.off_A = 0;
  L.off_B = align_up(L.off_A + L.state_bytes, 256);
  L.off_C = align_up(L.off_B + L.state_bytes, 256);
  L.off_scal = (rk >= 3) ? align_up(L.off_C + L.state_bytes, 256) : L.off_C;
  L.off_partial = L.off_scal + 256;                       // scal: 3 doubles + flag + ticket
  L.total = L.off_partial + align_up(sizeof(double) * kDtBlocksMax, 256);
  return L;
}

inline bool is_hall(int eqset) { return eqset == AGATE_HALL || eqset == AGATE_HALL_GLM; }
inline bool is_glm(int eqset) { return eqset == AGATE_IDEAL_GLM || eqset == AGATE_HALL_GLM || eqset == AGATE_CGL_GLM; }
inline bool is_cgl(int eqset) { return eqset == AGATE_CGL || eqset == AGATE_CGL_GLM; }
inline int nvar_of(int eqset) { return 8 + (is_glm(eqset) ? 1 : 0) + (is_cgl(eqset) ? 1 : 0); }

int check_args(const agate_grid* g, double gamma, int eqset, const agate_solver* s) {
  if (!g || !s) return AGATE_ERR_ARG;
  if (g->ndim < 1 || g->ndim > 3) return AGATE_ERR_ARG;
  if (g->nx < 1 || g->ny < 1 || g->nz < 1) return AGATE_ERR_ARG;
  if (g->ndim < 3 && g->nz != 1) return AGATE_ERR_ARG;
  if (g->ndim < 2 && g->ny != 1) return AGATE_ERR_ARG;
  if (!(g->dx > 0.0) || (g->ndim >= 2 && !(g->dy > 0.0)) || (g->ndim >= 3 && !(g->dz > 0.0))) return AGATE_ERR_ARG;
  if (!(gamma > 1.0)) return AGATE_ERR_ARG;
  if (eqset != AGATE_IDEAL && eqset != AGATE_HALL && eqset != AGATE_IDEAL_GLM && eqset != AGATE_CGL && eqset != AGATE_HALL_GLM &&
      eqset != AGATE_CGL_GLM)
    return AGATE_ERR_ARG;
  if (is_cgl(eqset) && s->riemann != AGATE_HLL) return AGATE_ERR_ARG;    // CGL: HLL (the paper names no other solver)
  if (is_cgl(eqset) && !(s->relax >= 0.0 && s->relax <= 1.0)) return AGATE_ERR_ARG;
  if (s->cgl_form < 0 || s->cgl_form > 1) return AGATE_ERR_ARG;
  if (s->riemann < 0 || s->riemann > 1 || s->limiter < 0 || s->limiter > 2 || s->rk < 1 || s->rk > 5) return AGATE_ERR_ARG;
  if (s->limiter == 2 && !(s->beta >= 1.0 && s->beta <= 2.0)) return AGATE_ERR_ARG;
  for (int d = 0; d < 3; ++d) if (s->bc[d] < 0 || s->bc[d] > ((d == 1) ? 2 : 1)) return AGATE_ERR_ARG;
  if (s->bc[1] == 2 && (g->ndim < 2 || s->bc[0] != 0)) return AGATE_ERR_ARG;   // sheared ends in y need a periodic x (R28)
  if (is_hall(eqset) && s->riemann == AGATE_HLLD) return AGATE_ERR_ARG;   // no Hall-HLLD in the paper
  if (is_hall(eqset) && !(s->d_i >= 0.0)) return AGATE_ERR_ARG;
  return AGATE_OK;
}

// The equation sets with extra variables (GLM, CGL) have no 1-D kernel: a 1-D grid runs through the 2-D strip kernel as ONE row
// that is its own periodic neighbour in y.  Both y faces of a zone then see identical states, their fluxes are the same
// number and the y difference is an exact zero, so the result is that of the 1-D scheme (the oracle has no y sweep at
// all); Courant number and dx_min are still those of the 1-D grid.
agate_grid kernel_grid(const agate_grid& g, int eqset) {
  agate_grid k = g;
  if (g.ndim == 1 && nvar_of(eqset) > 8) { k.ndim = 2; k.dy = g.dx; }
  return k;
}

typedef void (*stage_fn_t)(const StageParams);

struct StageKernel {
  stage_fn_t fn;
  int ty, np, threads;
  size_t smem;
  bool even_split = false;   // stage3d_kernel: one-wave grid, work split evenly (see agate_stage3d.cuh)
  bool fused_dt = false;     // stage3d / stage2d kernels: A7 of the next step inside the last stage of this one
  bool strips2d = false;     // stage2d_kernel: one-wave grid of autonomous warps (see agate_stage2d.cuh)
  int warps2d = 0;           // ... warps per CTA
};

template <int TY, int NP, int R, bool H, int MINB>
StageKernel make_stage() {
  StageKernel k;
  k.fn = stage_kernel<TY, NP, R, H, MINB>;
  k.ty = TY; k.np = NP; k.threads = StageSmem<TY, NP>::NT; k.smem = StageSmem<TY, NP>::BYTES;
  return k;
}

template <int TY, int R, int LIM, int MINB, bool GLM = false, bool CGL = false, bool HALL = false>
StageKernel make_stage3d() {
  StageKernel k;
  k.fn = stage3d_kernel<TY, R, LIM, MINB, GLM, CGL, HALL>;
  using SM = Stage3dSmem<TY, 8 + (GLM ? 1 : 0) + (CGL ? 1 : 0), HALL ? 3 : 2>;
  static_assert(SM::BYTES <= 232448, "stage3d shared memory exceeds 227 KB");
  k.ty = TY; k.np = 3; k.threads = SM::NT;
  k.smem = SM::BYTES;
  k.even_split = true;
  k.fused_dt = !CGL;         // the fused reduction evaluates the ideal-MHD speed; CGL keeps the dt_kernel pass
  return k;
}

template <int R, int LIM, bool H, bool GLM = false, bool CGL = false>
StageKernel make_stage2d() {
  StageKernel k;
  k.fn = stage2d_kernel<R, LIM, H, GLM, CGL>;
  using SM = Stage2dSmem<8 + (GLM ? 1 : 0) + (CGL ? 1 : 0)>;
  k.ty = 1; k.np = 1; k.threads = 32 * SM::NW; k.smem = SM::BYTES;
  k.warps2d = SM::NW;
  k.strips2d = true;
  k.fused_dt = !CGL;         // the fused reduction evaluates the ideal / Hall speed; CGL keeps the dt_kernel pass
  return k;
}

StageKernel pick_stage(int ndim, int eqset, int riemann, int limiter) {
  if (ndim == 3) {
    if (eqset == AGATE_HALL_GLM)
      return (limiter == 2) ? make_stage3d<TY3N, 0, 2, AGATE_MINB3, true, false, true>()
                            : make_stage3d<TY3N, 0, -1, AGATE_MINB3, true, false, true>();
    if (eqset == AGATE_HALL)
      return (limiter == 2) ? make_stage3d<TY3, 0, 2, AGATE_MINB3, false, false, true>()
                            : make_stage3d<TY3, 0, -1, AGATE_MINB3, false, false, true>();
    if (eqset == AGATE_CGL_GLM)
      return (limiter == 2) ? make_stage3d<TY3X, 0, 2, AGATE_MINB3, true, true>() : make_stage3d<TY3X, 0, -1, AGATE_MINB3, true, true>();
    if (eqset == AGATE_CGL)
      return (limiter == 2) ? make_stage3d<TY3N, 0, 2, AGATE_MINB3, false, true>() : make_stage3d<TY3N, 0, -1, AGATE_MINB3, false, true>();
    if (eqset == AGATE_IDEAL_GLM) {
      if (riemann == AGATE_HLLD) return (limiter == 2) ? make_stage3d<TY3N, 1, 2, AGATE_MINB3, true>() : make_stage3d<TY3N, 1, -1, AGATE_MINB3, true>();
      return (limiter == 2) ? make_stage3d<TY3N, 0, 2, AGATE_MINB3, true>() : make_stage3d<TY3N, 0, -1, AGATE_MINB3, true>();
    }
    if (limiter == 2) {                  // eq.4 (every BASELINE config): limiter fixed at compile time
      if (riemann == AGATE_HLLD) return make_stage3d<TY3, 1, 2, AGATE_MINB3>();
      return make_stage3d<TY3, 0, 2, AGATE_MINB3>();
    }
    if (riemann == AGATE_HLLD) return make_stage3d<TY3, 1, -1, AGATE_MINB3>();
    return make_stage3d<TY3, 0, -1, AGATE_MINB3>();
  }
  if (ndim == 2) {   // warp-autonomous strips
    if (eqset == AGATE_HALL_GLM) return (limiter == 2) ? make_stage2d<0, 2, true, true>() : make_stage2d<0, -1, true, true>();
    if (eqset == AGATE_HALL)
      return (limiter == 3) ? make_stage2d<0, 3, true>() : ((limiter == 2) ? make_stage2d<0, 2, true>() : make_stage2d<0, -1, true>());
    if (eqset == AGATE_CGL_GLM) return (limiter == 2) ? make_stage2d<0, 2, false, true, true>() : make_stage2d<0, -1, false, true, true>();
    if (eqset == AGATE_CGL) return (limiter == 2) ? make_stage2d<0, 2, false, false, true>() : make_stage2d<0, -1, false, false, true>();
    if (eqset == AGATE_IDEAL_GLM) {
      if (riemann == AGATE_HLLD) return (limiter == 2) ? make_stage2d<1, 2, false, true>() : make_stage2d<1, -1, false, true>();
      return (limiter == 2) ? make_stage2d<0, 2, false, true>() : make_stage2d<0, -1, false, true>();
    }
    if (limiter == 3 && riemann == AGATE_HLL) return make_stage2d<0, 3, false>();     // eq.4 at beta = 1: minmod
    if (limiter >= 2) {
      if (riemann == AGATE_HLLD) return make_stage2d<1, 2, false>();
      return make_stage2d<0, 2, false>();
    }
    if (riemann == AGATE_HLLD) return make_stage2d<1, -1, false>();
    return make_stage2d<0, -1, false>();
  }
  if (eqset == AGATE_HALL) return make_stage<TY2, 1, 0, true, 2>();
  if (riemann == AGATE_HLLD) return make_stage<TY2, 1, 1, false, 2>();
  return make_stage<TY2, 1, 0, false, 2>();
}

}  // namespace

struct agate_ctx {
  agate_grid g;
  agate_solver s;
  double gamma;
  int eqset;
  int nv;                          // variables per cell: 8, +1 with CGL's A, +1 with the GLM scalar
  Layout L;
  Phys ph;
  double dxmin, cfl;
  cudaStream_t stream;
  char* ws;
  double *UA, *UB, *UC, *scal, *partial;
  int* flag;
  unsigned int* ticket;
  unsigned long long* vnext;       // fused A7: bit pattern of v_max of the current state (valid iff vmax_valid)
  bool vmax_valid = false;
  bool have_state = false;
  int sticky = AGATE_OK;
  StageKernel sk;
  dim3 sgrid;
  int lz;
  int dt_blocks, ghost_blocks;
  GhostParams gpA, gpB, gpC;
  cudaGraphExec_t graph = nullptr;
  bool timing = false;
  bool no_graph = false;           // agate_set_tuning: launch the kernels directly
  bool ext_lo = false, ext_hi = false;   // NEXT-4: cut faces of a slab decomposition (last active dimension)
  bool vmax_given = false;         // agate_set_vmax: the device v_max is the caller's global maximum
  int next_stage = -1;             // split-phase stepping: stage expected next (-1: no step open)
  bool pre_done = false;           // ... and whether its agate_stage_pre has run
  std::vector<cudaEvent_t> ev;     // pairs (start, stop) of timed stage launches
  size_t ev_used = 0;
  double stage_ms = 0.0;
  int64_t stage_launches = 0;
  int regs = 0, occ = 0;
};

namespace {

#define CU_TRY(expr)                                   \
  do {                                                 \
    cudaError_t e__ = (expr);                          \
    if (e__ != cudaSuccess) {                          \
      c->sticky = AGATE_ERR_CUDA;                      \
      return AGATE_ERR_CUDA;                           \
    }                                                  \
  } while (0)

GhostParams make_ghost(const agate_ctx* c, double* U) {
  GhostParams p;
  const Layout& L = c->L;
  p.U = U;
  p.nv = c->nv;
  p.bcx = c->s.bc[0]; p.bcy = c->s.bc[1]; p.bcz = c->s.bc[2];
  p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz;
  p.ghy = L.ghy; p.ghz = L.ghz; p.nxp = L.nxp; p.nyp = L.nyp; p.nzp = L.nzp;
  p.sy = L.sy; p.sz = L.sz; p.sq = L.sq;
  p.nzs = (long long)2 * L.ghz * L.nyp * L.nxp;
  p.nys = (long long)c->g.nz * 2 * L.ghy * L.nxp;
  p.nxs = (long long)c->g.nz * c->g.ny * 4;
  p.dcut = (c->g.ndim == 3) ? 2 : 1;
  p.skip_lo = c->ext_lo ? 1 : 0;
  p.skip_hi = c->ext_hi ? 1 : 0;
  return p;
}

StageParams make_stage_params(const agate_ctx* c, const double* Uin, const double* U0, double* Uout, double a0,
                              double a1, double cdt, bool last_stage) {
  StageParams p;
  const Layout& L = c->L;
  p.Uin = Uin; p.U0 = U0; p.Uout = Uout; p.dt_ptr = c->scal;
  p.a0 = a0; p.a1 = a1; p.r0 = (a0 != 0.0) ? a0 / a1 : 0.0; p.cdt = cdt;
  p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.ndim = c->g.ndim;
  p.ghy = L.ghy; p.ghz = L.ghz; p.nxp = L.nxp; p.nyp = L.nyp;
  p.sy = L.sy; p.sz = L.sz; p.sq = L.sq;
  p.idx = 1.0 / c->g.dx;
  p.idy = (c->g.ndim >= 2) ? 1.0 / c->g.dy : 0.0;
  p.idz = (c->g.ndim >= 3) ? 1.0 / c->g.dz : 0.0;
  p.limiter = c->s.limiter; p.beta = c->s.beta;
  p.vnext = (last_stage && c->sk.fused_dt) ? c->vnext : nullptr;
  p.flag = c->flag;
  p.ch_ptr = c->scal + 3;
  p.last_stage = last_stage ? 1 : 0;
  p.relax = is_cgl(c->eqset) ? c->s.relax : 0.0;
  p.lz = c->lz;
  p.ntx = (c->g.nx + TX - 1) / TX;
  p.nty = (c->g.ny + c->sk.ty - 1) / c->sk.ty;
  p.ph = c->ph;
  return p;
}

int launch_ghost(agate_ctx* c, const GhostParams& gp) {
  ghost_fill_kernel<<<c->ghost_blocks, 256, 0, c->stream>>>(gp);
  CU_TRY(cudaGetLastError());
  return AGATE_OK;
}

int launch_dt(agate_ctx* c, int add_t) {
  DtParams p;
  const Layout& L = c->L;
  p.U = c->UA;
  p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.ghy = L.ghy; p.ghz = L.ghz;
  p.sy = L.sy; p.sz = L.sz; p.sq = L.sq;
  p.cfl_dx = c->cfl * c->dxmin;
  p.ph = c->ph;
  p.scal = c->scal; p.flag = c->flag; p.ticket = c->ticket; p.partial = c->partial;
  p.add_t = add_t;
  p.cgl = is_cgl(c->eqset) ? 1 : 0;
  if (is_hall(c->eqset)) dt_kernel<true><<<c->dt_blocks, 256, 0, c->stream>>>(p);
  else dt_kernel<false><<<c->dt_blocks, 256, 0, c->stream>>>(p);
  CU_TRY(cudaGetLastError());
  return AGATE_OK;
}

int launch_stage(agate_ctx* c, const StageParams& sp) {
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (c->timing) {
    if (c->ev_used + 2 > c->ev.size()) {
      for (int i = 0; i < 2; ++i) {
        cudaEvent_t e;
        CU_TRY(cudaEventCreate(&e));
        c->ev.push_back(e);
      }
    }
    e0 = c->ev[c->ev_used]; e1 = c->ev[c->ev_used + 1];
    c->ev_used += 2;
    CU_TRY(cudaEventRecord(e0, c->stream));
  }
  c->sk.fn<<<c->sgrid, c->sk.threads, c->sk.smem, c->stream>>>(sp);
  CU_TRY(cudaGetLastError());
  if (c->timing) CU_TRY(cudaEventRecord(e1, c->stream));
  return AGATE_OK;
}

// One full time step enqueued on the stream; dt is already in scal[0].  Every stage is
//     Uout = a0 Uref + a1 (Uin + c dt L(Uin))                                   (Shu-Osher form, dt once per step: R11)
// with the ghost fill of Uin in front of it.  A, B, C are the state copies; the step starts and ends with U^n in A.
//   RK11:      B = A + dt L(A)                                                   (then A <-> B)
//   SSP-RK22:  B = A + dt L(A);  A = 1/2 A + 1/2 (B + dt L(B))                                              (R11)
//   SSP-RK33:  B = A + dt L(A);  C = 3/4 A + 1/4 (B + dt L(B));  A = 1/3 A + 2/3 (C + dt L(C))             (R25)
//   RK43:      c = 1/2:  B = A + c dt L(A);  C = B + c dt L(B);  B = 2/3 A + 1/3 (C + c dt L(C));  A = B + c dt L(B)   (R27)
//   RK53:      c = 0.377268915331368:  B = A + c dt L(A);  C = B + c dt L(B);  B = a30 A + a32 (C + c dt L(C));
//              A = a40 A + a43 (B + c dt L(B));  B = a52 C + a54 (A + c dt L(A))   (then A <-> B)             (R27)
// Uref may be the output buffer (the combine is pointwise); Uin never is (the stage reads its neighbours).
struct RkStage { int in, ref, out; double a0, a1, c; };
int rk_table(int rk, RkStage st[5], bool* swap_ab) {
  *swap_ab = false;
  switch (rk) {
    case 1: st[0] = {0, -1, 1, 0.0, 1.0, 1.0}; *swap_ab = true; return 1;
    case 2: st[0] = {0, -1, 1, 0.0, 1.0, 1.0}; st[1] = {1, 0, 0, 0.5, 0.5, 1.0}; return 2;
    case 3:
      st[0] = {0, -1, 1, 0.0, 1.0, 1.0}; st[1] = {1, 0, 2, 0.75, 0.25, 1.0}; st[2] = {2, 0, 0, 1.0 / 3.0, 2.0 / 3.0, 1.0};
      return 3;
    case 4:
      st[0] = {0, -1, 1, 0.0, 1.0, 0.5}; st[1] = {1, -1, 2, 0.0, 1.0, 0.5};
      st[2] = {2, 0, 1, 2.0 / 3.0, 1.0 / 3.0, 0.5}; st[3] = {1, -1, 0, 0.0, 1.0, 0.5};
      return 4;
    default: {
      const double c = 0.377268915331368;
      st[0] = {0, -1, 1, 0.0, 1.0, c}; st[1] = {1, -1, 2, 0.0, 1.0, c};
      st[2] = {2, 0, 1, 0.355909775063327, 0.644090224936674, c};
      st[3] = {1, 0, 0, 0.367933791638137, 0.632066208361863, c};
      st[4] = {0, 2, 1, 0.237593836598569, 0.762406163401431, c};
      *swap_ab = true;
      return 5;
    }
  }
}

// First half of stage i: ghost fill of the stage input (A0).  Second half: the stage kernel (A1-A6), and after the
// last stage the buffer rotation.  The slab decomposition (NEXT-4) puts its halo exchange between the two.
int stage_pre(agate_ctx* c, int i) {
  RkStage st[5];
  bool swap_ab;
  rk_table(c->s.rk, st, &swap_ab);
  const GhostParams* gp[3] = {&c->gpA, &c->gpB, &c->gpC};
  return launch_ghost(c, *gp[st[i].in]);
}
int stage_post(agate_ctx* c, int i) {
  RkStage st[5];
  bool swap_ab;
  const int ns = rk_table(c->s.rk, st, &swap_ab);
  double* U[3] = {c->UA, c->UB, c->UC};
  const double* ref = (st[i].ref >= 0) ? U[st[i].ref] : nullptr;
  int rc = launch_stage(c, make_stage_params(c, U[st[i].in], ref, U[st[i].out], st[i].a0, st[i].a1, st[i].c, i == ns - 1));
  if (rc) return rc;
  if (i == ns - 1 && swap_ab) {
    std::swap(c->UA, c->UB);
    std::swap(c->gpA, c->gpB);
  }
  return AGATE_OK;
}
double* stage_input(agate_ctx* c, int i) {
  RkStage st[5];
  bool swap_ab;
  rk_table(c->s.rk, st, &swap_ab);
  double* U[3] = {c->UA, c->UB, c->UC};
  return U[st[i].in];
}

int enqueue_stages(agate_ctx* c) {
  int rc;
  for (int i = 0; i < c->s.rk; ++i) {
    if ((rc = stage_pre(c, i))) return rc;
    if ((rc = stage_post(c, i))) return rc;
  }
  return AGATE_OK;
}

// Head of a self-timed step: dt = C dx_min / v_max(U^n), t += dt  (R11).  Separate reduction pass, or -- when the
// previous step's last stage already reduced v_max of what it stored -- one thread that turns it into dt.
int launch_step_head(agate_ctx* c) {
  if (!c->sk.fused_dt) return launch_dt(c, 1);
  begin_step_kernel<<<1, 1, 0, c->stream>>>(c->scal, c->vnext, c->cfl * c->dxmin);
  CU_TRY(cudaGetLastError());
  return AGATE_OK;
}

// the fused path needs v_max of the current state once after agate_set_state
int ensure_vmax(agate_ctx* c) {
  if (!c->sk.fused_dt || c->vmax_valid) return AGATE_OK;
  int rc = launch_dt(c, 0);
  if (rc) return rc;
  seed_vnext_kernel<<<1, 1, 0, c->stream>>>(c->scal, c->vnext);
  CU_TRY(cudaGetLastError());
  c->vmax_valid = true;
  return AGATE_OK;
}

// GLM with a host-chosen dt: c_h = 0.95 v_max(U^n) must still be on the device.  The fused path hands v_max to
// set_dt_kernel; a kernel without the fused reduction (CGL + GLM) runs the reduction pass, which writes c_h itself.
int ensure_ch(agate_ctx* c) {
  if (c->sk.fused_dt) return ensure_vmax(c);
  return launch_dt(c, 0);
}

int collect_status(agate_ctx* c) {
  CU_TRY(cudaStreamSynchronize(c->stream));
  int flag = 0;
  CU_TRY(cudaMemcpy(&flag, c->flag, sizeof(int), cudaMemcpyDeviceToHost));
  if ((flag & 2) && c->sticky == AGATE_OK) c->sticky = AGATE_ERR_CUDA;          // a hand-over wait ran out (stage3d)
  if ((flag & 1) && c->sticky == AGATE_OK) c->sticky = AGATE_ERR_UNPHYSICAL;
  return c->sticky;
}

int copy_state(agate_ctx* c, double* padded, double* ext, bool to_device, bool ext_is_device) {
  const Layout& L = c->L;
  for (int q = 0; q < c->nv; ++q) {
    cudaMemcpy3DParms m;
    memset(&m, 0, sizeof(m));
    cudaPitchedPtr pp = make_cudaPitchedPtr(padded + (size_t)q * L.sq, sizeof(double) * L.nxp, L.nxp, L.nyp);
    cudaPitchedPtr pe = make_cudaPitchedPtr(ext + (size_t)q * c->g.nx * c->g.ny * c->g.nz, sizeof(double) * c->g.nx,
                                            c->g.nx, c->g.ny);
    cudaPos ppos = make_cudaPos(sizeof(double) * 2, L.ghy, L.ghz);
    cudaPos epos = make_cudaPos(0, 0, 0);
    if (to_device) { m.srcPtr = pe; m.srcPos = epos; m.dstPtr = pp; m.dstPos = ppos; }
    else { m.srcPtr = pp; m.srcPos = ppos; m.dstPtr = pe; m.dstPos = epos; }
    m.extent = make_cudaExtent(sizeof(double) * c->g.nx, c->g.ny, c->g.nz);
    m.kind = ext_is_device ? cudaMemcpyDeviceToDevice : (to_device ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost);
    CU_TRY(cudaMemcpy3DAsync(&m, c->stream));
  }
  return AGATE_OK;
}

// Launch grid of the stage kernel.  The pooled kernel (1-D grids) takes one CTA per tile; the 2-D and 3-D kernels
// run as one resident wave whose CTAs (warps) split the work evenly: `forced` > 0 fixes the number of CTAs
// (agate_set_tuning; the tests use it to reach ragged splits), 0 = as many as are resident, fewer on tiny grids.
void set_stage_grid(agate_ctx* c, int forced) {
  const agate_grid& g = c->g;
  const int ntx = (g.nx + TX - 1) / TX, nty = (g.ny + c->sk.ty - 1) / c->sk.ty;
  c->sgrid = dim3(ntx, nty, 1);
  if (!c->sk.strips2d && !c->sk.even_split) return;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const long long slots = (long long)sms * (c->occ > 0 ? c->occ : 1);
  long long n;
  if (c->sk.strips2d) {
    // a warp gets at least ~4 rows of its 30-column strip
    const long long work = (long long)((g.nx + SW2 - 1) / SW2) * g.ny;
    n = (work + 4 * c->sk.warps2d - 1) / (4 * c->sk.warps2d);
  } else {
    // a CTA gets at least ~16 tile-planes so that a segment's start-up (three plane loads and the step that
    // closes its last plane) stays small on tiny grids
    const long long work = (long long)ntx * nty * g.nz;
    n = (work + 15) / 16;
  }
  if (n > slots) n = slots;
  if (n < 1) n = 1;
  if (forced > 0) n = forced;
  c->sgrid = dim3((unsigned)n, 1, 1);
}

}  // namespace

extern "C" {

size_t agate_workspace_bytes(const agate_grid* grid, int eqset, const agate_solver* solver) {
  if (check_args(grid, 5.0 / 3.0, eqset, solver) != AGATE_OK) return 0;
  return make_layout(kernel_grid(*grid, eqset), nvar_of(eqset), solver->rk).total;
}

int agate_init(const agate_grid* grid, double gamma, int eqset, const agate_solver* solver, void* workspace,
               size_t workspace_bytes, void* stream, agate_ctx** out) {
  if (!out) return AGATE_ERR_ARG;
  int rc = check_args(grid, gamma, eqset, solver);
  if (rc) return rc;
  if (!workspace) return AGATE_ERR_ARG;
  const int nv = nvar_of(eqset);
  const agate_grid user_grid = *grid;                 // Courant number and dx_min follow the caller's dimensionality
  const agate_grid kgrid = kernel_grid(*grid, eqset);
  grid = &kgrid;
  Layout L = make_layout(*grid, nv, solver->rk);
  if (workspace_bytes < L.total || ((uintptr_t)workspace & 255u)) return AGATE_ERR_NOMEM;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return AGATE_ERR_CUDA;   // no CPU fallback

  agate_ctx* c = new (std::nothrow) agate_ctx;
  if (!c) return AGATE_ERR_NOMEM;
  c->g = *grid; c->s = *solver; c->gamma = gamma; c->eqset = eqset; c->L = L; c->nv = nv;
  c->dxmin = user_grid.dx;
  if (user_grid.ndim >= 2) c->dxmin = fmin(c->dxmin, user_grid.dy);      // R5: min over ACTIVE dimensions
  if (user_grid.ndim >= 3) c->dxmin = fmin(c->dxmin, user_grid.dz);
  c->cfl = solver->cfl;
  if (!(c->cfl > 0.0)) c->cfl = (user_grid.ndim == 1) ? 0.8 : (user_grid.ndim == 2 ? 0.45 : 0.325);
  c->ph = make_phys(gamma, is_hall(eqset) ? solver->d_i : 0.0, c->dxmin);
  c->ph.cgl_form = is_cgl(eqset) ? solver->cgl_form : 0;
  c->stream = (cudaStream_t)stream;
  c->ws = (char*)workspace;
  c->UA = (double*)(c->ws + L.off_A);
  c->UB = (double*)(c->ws + L.off_B);
  c->UC = (double*)(c->ws + L.off_C);
  c->scal = (double*)(c->ws + L.off_scal);
  c->flag = (int*)(c->ws + L.off_scal + 64);
  c->ticket = (unsigned int*)(c->ws + L.off_scal + 128);
  c->vnext = (unsigned long long*)(c->ws + L.off_scal + 192);
  c->partial = (double*)(c->ws + L.off_partial);

  // eq.4 at beta = 1 is plain minmod: the 2-D HLL kernels (configs 1 and 4) have a variant without its third argument
  c->sk = pick_stage(grid->ndim, eqset, solver->riemann,
                     (solver->limiter == 2 && solver->beta == 1.0 && grid->ndim == 2 && solver->riemann == AGATE_HLL &&
                      (eqset == AGATE_IDEAL || eqset == AGATE_HALL)) ? 3 : solver->limiter);
  cudaError_t e = cudaFuncSetAttribute((const void*)c->sk.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->sk.smem);
  cudaFuncAttributes fa;
  if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, (const void*)c->sk.fn);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ, (const void*)c->sk.fn, c->sk.threads, c->sk.smem);
  if (e != cudaSuccess) { delete c; return AGATE_ERR_CUDA; }
  c->regs = fa.numRegs;

  c->lz = grid->nz;
  set_stage_grid(c, 0);
  long long nrows = (long long)grid->ny * grid->nz;
  c->dt_blocks = (int)(nrows < kDtBlocksMax ? nrows : kDtBlocksMax);
  c->gpA = make_ghost(c, c->UA);
  c->gpB = make_ghost(c, c->UB);
  c->gpC = make_ghost(c, c->UC);
  long long nghost = c->gpA.nzs + c->gpA.nys + c->gpA.nxs;
  long long gb = (nghost + 255) / 256;
  c->ghost_blocks = (int)(gb < 148 * 16 ? (gb < 1 ? 1 : gb) : 148 * 16);

  if (cudaMemsetAsync(c->ws + L.off_scal, 0, L.total - L.off_scal, c->stream) != cudaSuccess) { delete c; return AGATE_ERR_CUDA; }
  *out = c;
  return AGATE_OK;
}

int agate_set_state(agate_ctx* c, const double* U, int src_is_device, double t0) {
  if (!c || !U) return AGATE_ERR_ARG;
  int rc = copy_state(c, c->UA, const_cast<double*>(U), true, src_is_device != 0);
  if (rc) return rc;
  reset_scalars_kernel<<<1, 1, 0, c->stream>>>(c->scal, c->flag, t0);
  CU_TRY(cudaGetLastError());
  // a HOST array is borrowed only for this call; a DEVICE source is read in stream order, no synchronisation
  if (!src_is_device) CU_TRY(cudaStreamSynchronize(c->stream));
  if ((rc = launch_ghost(c, c->gpA))) return rc;
  c->have_state = true;
  c->vmax_valid = false;
  c->vmax_given = false;
  c->next_stage = -1;
  c->pre_done = false;
  if (c->sticky == AGATE_ERR_UNPHYSICAL) c->sticky = AGATE_OK;
  return AGATE_OK;
}

int agate_compute_dt(agate_ctx* c, double* dt_out) {
  if (!c || !dt_out) return AGATE_ERR_ARG;
  if (!c->have_state) return AGATE_ERR_STATE;
  int rc = launch_dt(c, 0);
  if (rc) return rc;
  rc = collect_status(c);
  if (rc) return rc;
  double dt;
  CU_TRY(cudaMemcpy(&dt, c->scal, sizeof(double), cudaMemcpyDeviceToHost));
  *dt_out = dt;
  return AGATE_OK;
}

int agate_step(agate_ctx* c, double dt, double* dt_used) {
  if (!c) return AGATE_ERR_ARG;
  if (!c->have_state || c->ext_lo || c->ext_hi) return AGATE_ERR_STATE;   // a slab steps through agate_stage_pre / _post
  int rc;
  if (dt > 0.0) {
    if (is_glm(c->eqset) && (rc = ensure_ch(c))) return rc;        // c_h = 0.95 v_max(U^n) whoever chose dt
    set_dt_kernel<<<1, 1, 0, c->stream>>>(c->scal, dt, c->sk.fused_dt ? c->vnext : nullptr);
    CU_TRY(cudaGetLastError());
  } else {
    if ((rc = ensure_vmax(c))) return rc;
    if ((rc = launch_step_head(c))) return rc;
  }
  if ((rc = enqueue_stages(c))) return rc;
  c->vmax_valid = c->sk.fused_dt;
  if (dt_used) {
    if ((rc = collect_status(c))) return rc;
    double v;
    CU_TRY(cudaMemcpy(&v, c->scal, sizeof(double), cudaMemcpyDeviceToHost));
    *dt_used = v;
  }
  return AGATE_OK;
}

int agate_advance(agate_ctx* c, int32_t n_steps, double* t_out) {
  if (!c || n_steps < 0) return AGATE_ERR_ARG;
  if (!c->have_state || c->ext_lo || c->ext_hi) return AGATE_ERR_STATE;
  int rc;
  // stream capture is not allowed on the legacy default stream
  const bool use_graph = (c->s.rk >= 2 && c->s.rk <= 4) && !c->timing && c->stream != nullptr && !c->no_graph;
  if (n_steps > 0 && (rc = ensure_vmax(c))) return rc;
  if (use_graph && !c->graph && n_steps > 0) {
    cudaGraph_t g = nullptr;
    CU_TRY(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed));
    rc = launch_step_head(c);
    if (!rc) rc = enqueue_stages(c);
    cudaError_t e = cudaStreamEndCapture(c->stream, &g);
    if (rc || e != cudaSuccess) { if (g) cudaGraphDestroy(g); c->sticky = AGATE_ERR_CUDA; return AGATE_ERR_CUDA; }
    e = cudaGraphInstantiate(&c->graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { c->graph = nullptr; c->sticky = AGATE_ERR_CUDA; return AGATE_ERR_CUDA; }
  }
  for (int i = 0; i < n_steps; ++i) {
    if (use_graph) {
      CU_TRY(cudaGraphLaunch(c->graph, c->stream));
    } else {
      if ((rc = launch_step_head(c))) return rc;
      if ((rc = enqueue_stages(c))) return rc;
    }
  }
  if (t_out) {
    if ((rc = collect_status(c))) return rc;
    double sc[3];
    CU_TRY(cudaMemcpy(sc, c->scal, sizeof(sc), cudaMemcpyDeviceToHost));
    *t_out = sc[2];
  }
  return AGATE_OK;
}

int agate_get_state(agate_ctx* c, double* U_out, int dst_is_device, double* t_out) {
  if (!c || !U_out) return AGATE_ERR_ARG;
  if (!c->have_state) return AGATE_ERR_STATE;
  int rc = copy_state(c, c->UA, U_out, false, dst_is_device != 0);
  if (rc) return rc;
  if (!dst_is_device || t_out) {
    CU_TRY(cudaStreamSynchronize(c->stream));
    if (t_out) {
      double sc[3];
      CU_TRY(cudaMemcpy(sc, c->scal, sizeof(sc), cudaMemcpyDeviceToHost));
      *t_out = sc[2];
    }
  }
  return AGATE_OK;
}

int agate_poll(agate_ctx* c) {
  if (!c) return AGATE_ERR_ARG;
  return collect_status(c);
}

int agate_launch_info(agate_ctx* c, int64_t out[8]) {
  if (!c || !out) return AGATE_ERR_ARG;
  out[0] = c->sgrid.x; out[1] = c->sgrid.y; out[2] = c->sgrid.z;
  out[3] = c->sk.threads; out[4] = (int64_t)c->sk.smem; out[5] = c->regs; out[6] = c->occ;
  out[7] = 1 + 2 * c->s.rk;          // dt + (ghost + stage) per RK stage (rk = number of stages)
  return AGATE_OK;
}

int agate_set_timing(agate_ctx* c, int enabled) {
  if (!c) return AGATE_ERR_ARG;
  c->timing = enabled != 0;
  return AGATE_OK;
}

int agate_set_tuning(agate_ctx* c, const agate_tuning* t) {
  if (!c || !t || t->stage_grid < 0) return AGATE_ERR_ARG;
  set_stage_grid(c, t->stage_grid);
  c->no_graph = t->no_graph != 0;
  if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }      // captured with the old grid
  return AGATE_OK;
}

int agate_stage_time(agate_ctx* c, double* ms_out, int64_t* launches_out, int reset) {
  if (!c) return AGATE_ERR_ARG;
  CU_TRY(cudaStreamSynchronize(c->stream));
  for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
    float ms = 0.f;
    CU_TRY(cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
    c->stage_ms += ms;
    c->stage_launches += 1;
  }
  c->ev_used = 0;
  if (ms_out) *ms_out = c->stage_ms;
  if (launches_out) *launches_out = c->stage_launches;
  if (reset) { c->stage_ms = 0.0; c->stage_launches = 0; }
  return AGATE_OK;
}

// ---- NEXT-4: slab decomposition along the last active dimension -------------------------------------
int agate_set_slab(agate_ctx* c, int ext_lo, int ext_hi) {
  if (!c) return AGATE_ERR_ARG;
  if (c->g.ndim < 2 || ((c->g.ndim == 3) ? c->g.nz : c->g.ny) < 2) return AGATE_ERR_ARG;   // two layers per cut face
  c->ext_lo = ext_lo != 0; c->ext_hi = ext_hi != 0;
  c->gpA = make_ghost(c, c->UA); c->gpB = make_ghost(c, c->UB); c->gpC = make_ghost(c, c->UC);
  if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
  return AGATE_OK;
}

size_t agate_halo_bytes(const agate_ctx* c) {
  if (!c || c->g.ndim < 2) return 0;
  const long long plane = (c->g.ndim == 3) ? c->L.sz : c->L.sy;      // one padded plane (row) incl. its own ghosts
  return sizeof(double) * (size_t)c->nv * 2 * (size_t)plane;
}

int agate_get_vmax(agate_ctx* c, double* vmax_out) {
  if (!c || !vmax_out) return AGATE_ERR_ARG;
  if (!c->have_state) return AGATE_ERR_STATE;
  int rc;
  double v;
  if (c->sk.fused_dt && c->vmax_valid) {
    if ((rc = collect_status(c))) return rc;
    CU_TRY(cudaMemcpy(&v, c->vnext, sizeof(double), cudaMemcpyDeviceToHost));     // bit pattern of a positive double
  } else {
    if ((rc = launch_dt(c, 0))) return rc;
    if ((rc = collect_status(c))) return rc;
    CU_TRY(cudaMemcpy(&v, c->scal + 1, sizeof(double), cudaMemcpyDeviceToHost));
  }
  *vmax_out = v;
  return AGATE_OK;
}

int agate_set_vmax(agate_ctx* c, double vmax) {
  if (!c || !(vmax > 0.0)) return AGATE_ERR_ARG;
  if (!c->have_state) return AGATE_ERR_STATE;
  set_vnext_kernel<<<1, 1, 0, c->stream>>>(c->scal, c->vnext, vmax);
  CU_TRY(cudaGetLastError());
  c->vmax_given = true;
  return AGATE_OK;
}

int agate_vmax_device(agate_ctx* c, void** ptr_out) {
  if (!c || !ptr_out) return AGATE_ERR_ARG;
  if (!c->sk.fused_dt) return AGATE_ERR_ARG;      // only the kernels with the fused reduction keep v_max there
  *ptr_out = c->vnext;
  return AGATE_OK;
}

int agate_step_begin(agate_ctx* c, double dt) {
  if (!c) return AGATE_ERR_ARG;
  if (!c->have_state || c->next_stage != -1) return AGATE_ERR_STATE;
  int rc;
  const bool have_v = c->vmax_given || (c->sk.fused_dt && c->vmax_valid);
  if (dt > 0.0) {
    if (is_glm(c->eqset) && !have_v && (rc = ensure_ch(c))) return rc;
    set_dt_kernel<<<1, 1, 0, c->stream>>>(c->scal, dt, (c->sk.fused_dt || c->vmax_given) ? c->vnext : nullptr);
    CU_TRY(cudaGetLastError());
  } else {
    if (!have_v) {                                   // local v_max: a slab wants agate_set_vmax with the global one
      if ((rc = launch_dt(c, 0))) return rc;
      seed_vnext_kernel<<<1, 1, 0, c->stream>>>(c->scal, c->vnext);
      CU_TRY(cudaGetLastError());
    }
    begin_step_kernel<<<1, 1, 0, c->stream>>>(c->scal, c->vnext, c->cfl * c->dxmin);
    CU_TRY(cudaGetLastError());
  }
  c->vmax_given = false;
  c->vmax_valid = false;
  c->next_stage = 0;
  c->pre_done = false;
  return AGATE_OK;
}

int agate_stage_pre(agate_ctx* c, int stage, void* send_lo, void* send_hi) {
  if (!c || stage < 0 || stage >= c->s.rk) return AGATE_ERR_ARG;
  if ((c->ext_lo && !send_lo) || (c->ext_hi && !send_hi)) return AGATE_ERR_ARG;
  if (!c->have_state || c->next_stage != stage || c->pre_done) return AGATE_ERR_STATE;
  int rc = stage_pre(c, stage);                      // A0 on the ends that are not cut faces
  if (rc) return rc;
  // the two interior layers next to each cut face, whole padded planes (their x / y ghosts were just filled), every
  // variable: [nv][2 planes] contiguous in the caller's buffer
  const double* U = stage_input(c, stage);
  const long long plane = (c->g.ndim == 3) ? c->L.sz : c->L.sy;
  const int gh = 2, n = (c->g.ndim == 3) ? c->g.nz : c->g.ny;
  const size_t w = sizeof(double) * 2 * (size_t)plane;
  if (c->ext_lo) CU_TRY(cudaMemcpy2DAsync(send_lo, w, U + (long long)gh * plane, sizeof(double) * (size_t)c->L.sq, w, c->nv,
                                          cudaMemcpyDeviceToDevice, c->stream));
  if (c->ext_hi) CU_TRY(cudaMemcpy2DAsync(send_hi, w, U + (long long)n * plane, sizeof(double) * (size_t)c->L.sq, w, c->nv,
                                          cudaMemcpyDeviceToDevice, c->stream));
  c->pre_done = true;
  return AGATE_OK;
}

int agate_stage_post(agate_ctx* c, int stage, const void* recv_lo, const void* recv_hi) {
  if (!c || stage < 0 || stage >= c->s.rk) return AGATE_ERR_ARG;
  if ((c->ext_lo && !recv_lo) || (c->ext_hi && !recv_hi)) return AGATE_ERR_ARG;
  if (!c->have_state || c->next_stage != stage || !c->pre_done) return AGATE_ERR_STATE;
  double* U = stage_input(c, stage);
  const long long plane = (c->g.ndim == 3) ? c->L.sz : c->L.sy;
  const int gh = 2, n = (c->g.ndim == 3) ? c->g.nz : c->g.ny;
  const size_t w = sizeof(double) * 2 * (size_t)plane;
  // the neighbour's layers become this slab's ghost layers: below the low cut face, above the high one
  if (c->ext_lo) CU_TRY(cudaMemcpy2DAsync(U, sizeof(double) * (size_t)c->L.sq, recv_lo, w, w, c->nv, cudaMemcpyDeviceToDevice,
                                          c->stream));
  if (c->ext_hi) CU_TRY(cudaMemcpy2DAsync(U + (long long)(n + gh) * plane, sizeof(double) * (size_t)c->L.sq, recv_hi, w, w, c->nv,
                                          cudaMemcpyDeviceToDevice, c->stream));
  int rc = stage_post(c, stage);
  if (rc) return rc;
  c->pre_done = false;
  c->next_stage = (stage == c->s.rk - 1) ? -1 : stage + 1;
  if (c->next_stage == -1) c->vmax_valid = c->sk.fused_dt;
  return AGATE_OK;
}

int agate_destroy(agate_ctx* c) {
  if (!c) return AGATE_ERR_ARG;
  cudaStreamSynchronize(c->stream);
  if (c->graph) cudaGraphExecDestroy(c->graph);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  delete c;
  return AGATE_OK;
}

const char* agate_strerror(int status) {
  switch (status) {
    case AGATE_OK: return "ok";
    case AGATE_ERR_ARG: return "invalid argument or unsupported combination";
    case AGATE_ERR_STATE: return "call order: no state set";
    case AGATE_ERR_UNPHYSICAL: return "unphysical state (rho <= 0, p <= 0 or non-finite speed)";
    case AGATE_ERR_CUDA: return "CUDA error or no CUDA device";
    case AGATE_ERR_NOMEM: return "workspace too small or misaligned";
    case AGATE_ERR_LIMIT: return "grid needs more scratch than the library's static array holds (AGATE_STATIC_MAX_SEGMENTS)";
    default: return "unknown status";
  }
}

int agate_test_face_flux(int eqset, int riemann, int dir, double gamma, double d_i, double dxmin, const double* WL,
                         const double* WR, const double* J, double* F, int64_t n, void* stream) {
  if (!WL || !WR || !F || n < 0 || dir < 0 || dir > 2 || !(gamma > 1.0)) return AGATE_ERR_ARG;
  if (eqset == AGATE_HALL && riemann == AGATE_HLLD) return AGATE_ERR_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return AGATE_ERR_CUDA;
  if (n == 0) return AGATE_OK;
  Phys ph = make_phys(gamma, (eqset == AGATE_HALL) ? d_i : 0.0, dxmin);
  const int nb = (int)((n + 127) / 128);
  cudaStream_t st = (cudaStream_t)stream;
  if (eqset == AGATE_HALL) face_flux_kernel<0, true><<<nb, 128, 0, st>>>(ph, dir, WL, WR, J, F, n);
  else if (riemann == AGATE_HLLD) face_flux_kernel<1, false><<<nb, 128, 0, st>>>(ph, dir, WL, WR, J, F, n);
  else face_flux_kernel<0, false><<<nb, 128, 0, st>>>(ph, dir, WL, WR, J, F, n);
  if (cudaGetLastError() != cudaSuccess) return AGATE_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return AGATE_ERR_CUDA;
  return AGATE_OK;
}

int agate_measure_fp64_peak(int iters, double* tflops_out, void* scratch, void* stream) {
  if (!tflops_out || !scratch || iters < 1) return AGATE_ERR_ARG;
  int ndev = 0, dev = 0, sms = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return AGATE_ERR_CUDA;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaStream_t st = (cudaStream_t)stream;
  double* d = (double*)scratch;     // 8 bytes of the caller's device memory (never written in practice)
  const int blocks = sms * 8, trips = 4096;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  fp64_peak_kernel<<<blocks, 256, 0, st>>>(d, trips, 1.0000001, 1e-9);   // warm-up
  cudaEventRecord(e0, st);
  for (int i = 0; i < iters; ++i) fp64_peak_kernel<<<blocks, 256, 0, st>>>(d, trips, 1.0000001, 1e-9);
  cudaEventRecord(e1, st);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e != cudaSuccess || !(ms > 0.f)) return AGATE_ERR_CUDA;
  const double flops = 2.0 * 8 * 16 * (double)trips * 256.0 * blocks * iters;
  *tflops_out = flops / (ms * 1e-3) / 1e12;
  return AGATE_OK;
}

}  // extern "C"
