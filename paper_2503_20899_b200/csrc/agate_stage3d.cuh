// agate_stage3d.cuh — row-owner fused stage kernel for 3-D grids, sm_100a.
//
// Same arithmetic as stage_kernel (agate_kernels.cuh); what differs is how the CTA is organised:
//   * CTA = TY "owner" warps + 1 helper warp H.  Owner warp j owns row j of a 32 x TY x-y tile and marches along z;
//     lane i owns cell (i, j).  The owner of a cell computes its limited slopes and the Riemann flux through its
//     HIGH face in x and y and its LOW face in z, so every slope and every flux is computed once.
//   * x: neighbours are lanes of the same warp -> the right state and the low-face flux travel by warp shuffles.
//     The cells outside the row (x = -1, 32) belong to H, which hands  R(32)  and  F(-1/2)  over in XR / XF.
//   * y: neighbours are adjacent warps -> one hand-over row per tile row, Y[r]: first the right state of row r, then,
//     written over it by its only reader (the owner of row r-1), the flux through face r-1/2.  Row -1 (its flux
//     through face -1/2) and row TY (its right state) belong to H.
//   * z: private column, one plane behind: step k computes F(k-1/2) from planes k-1, k, k+1 and completes plane
//     k-1.  The left state W(k-1)+dW(k-1)/2 is carried in a per-thread shared slot.
//   * no register state across the Riemann calls: the flux differences of the plane being assembled live in a
//     per-thread shared slot (ACC), seeded with +dt/dz F(k-1/2) when that flux is formed and closed with the same
//     rounded product of F(k+1/2) one step later, so a uniform state stays bitwise fixed; Uin (+U0) of the own cell
//     is read when the plane is completed (A6).
//   * NO CTA-wide barrier in the steady state: three sub-phases per plane, and at each boundary a warp publishes a
//     counter (st.release) and waits (ld.acquire) only for the warps whose data it reads or overwrites -- its
//     two neighbours and H; H waits for all owners once per plane.  Phase A: z slope + flux, completion and store of
//     plane k-1, y slope -> Y.  Phase B1: y flux -> Y.  Phase B2: x slope + flux, x and y differences -> ACC.  H mirrors
//     the owners with the tile-edge tasks (one Riemann call in A and in B1, the halo cells in B2).
//   * no global-load latency on the critical path: conserved cells are brought in by cp.async (LDGSTS) one phase
//     ahead, straight into their final shared-memory slot, and turned into primitives IN PLACE (A1) by the thread
//     that issued the copy: owners their own cell of plane k+2, H the x-halo columns and the y-halo rows.
//   * the three tasks of a warp per plane run through one loop that is unrolled: three inlined copies of the solver,
//     each with its direction's variable permutation resolved at compile time.
//
// Shared memory per CTA (NV = 8 variables; 9 with GLM or CGL, 10 with both): ring 3 planes x NV x TY x 36, y-halo rows
// 2 x NV x 4 x 36, Y NV x (TY+1) x 32, z carry and accumulator NV x TY x 32 each, XR / XF NV x TY each, 16 counters:
// TY = 11 -> 162 KB (182 KB with 9 variables), one CTA of 12 warps per SM, <= 168 registers.  (TY = 15, 16 warps at
// 128 registers without spills, fits in 213 KB and was measured slower: profiles/r2_stage3d.md.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "agate_kernels.cuh"

namespace agate {

__device__ __forceinline__ void cp_async8(double* sdst, const double* gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(sdst)), "l"(gsrc)
               : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// Pairwise hand-over between the warps of a CTA: prog[w] = number of phases warp w has completed and published.
__device__ __forceinline__ void publish(int* prog_w, int value, int lane) {
  __syncwarp();                                   // every lane's shared-memory writes are ordered before lane 0's release
  if (lane == 0) asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(prog_w)), "r"(value) : "memory");
}
__device__ __forceinline__ int peek(const int* prog_w) {
  int v;
  asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(prog_w)) : "memory");
  return v;
}
// spin until prog[w] >= value; a bounded spin (a lost hand-over would otherwise hang the GPU): on overflow the
// caller's sticky flag gets bit 1 and the kernel runs on
__device__ __forceinline__ void await(const int* prog_w, int value, int* flag) {
  int spins = 0;
  while (peek(prog_w) < value) {
    __nanosleep(40);                              // the wait is for ~a phase of another warp; keep the issue slots free
    if (++spins > (1 << 22)) { atomicOr(flag, 2); break; }
  }
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// Bulk asynchronous copies (the TMA engine's 1-D form, cp.async.bulk) for the y-halo rows: a halo row of a tile, its x
// halo and corners included, is 36 contiguous doubles of the padded array, so one 288-byte copy per (row, variable)
// replaces 36 eight-byte cp.async.  Completion is counted in bytes on an mbarrier in shared memory.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(double* sdst, const double* gsrc, uint32_t bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(sdst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ bool mbar_test_wait(unsigned long long* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// generic-proxy accesses to a shared buffer are ordered before the async proxy (the bulk copy) overwrites it
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// rotated slot -> fixed variable; the scalars behind the MHD variables (CGL's A, the GLM psi) are not rotated
__host__ __device__ __forceinline__ int rv(int r, int n) { return (r < 8) ? rot_var(r, n) : r; }

template <int TY, int NV = 8, int NHB = 2>
struct Stage3dSmem {
  static_assert(TY >= 2 && TY <= 16, "the x-edge task packs two cells per row into one warp");
  static constexpr int NW = TY + 1;                 // warps: TY owners + H
  static constexpr int NT = 32 * NW;
  static constexpr int PL = TY * RS;                // one ring plane of one variable
  static constexpr int SB = 4 * RS;                 // one y-halo buffer of one variable (rows -2,-1,TY,TY+1)
  static constexpr int QS = 3 * PL + NHB * SB;      // per-variable stride of W (NHB y-halo buffers: 3 with Hall)
  static constexpr int YS = (TY + 1) * 32;          // y hand-over rows 0..TY (right state of row r, then flux of face r-1/2)
  static constexpr int ZS = TY * 32;                // per-thread slots: z carry, accumulator
  static constexpr int XS = TY;                     // x hand-over, one entry per row
  static constexpr int OFF_Y = NV * QS;
  static constexpr int OFF_WLZ = OFF_Y + NV * YS;
  static constexpr int OFF_ACC = OFF_WLZ + NV * ZS;
  static constexpr int OFF_XR = OFF_ACC + NV * ZS;
  static constexpr int OFF_XF = OFF_XR + NV * XS;
  static constexpr int OFF_PROG = OFF_XF + NV * XS;  // 16 ints: per-warp phase counters
  static constexpr int OFF_MBAR = OFF_PROG + 8;      // one mbarrier: H's bulk copies of the y-halo rows
  static constexpr int TOTAL = OFF_MBAR + 2;
  static constexpr size_t BYTES = sizeof(double) * (size_t)TOTAL;
};

// A8 (R15): rotated face current (J_n, J_t1, J_t2), J = curl B, at the face between cells C and D = C + e_n from
// the cell-centred B of the stage input: central difference across the face along n; along a transverse direction
// the mean of the two cells' central differences.  o* are offsets into one variable's shared array (stride QS per
// variable): C, D, and their neighbours at +-1 along t1 = n+1 and t2 = n+2 (cyclic).  q1 = 1/(4 h_t1), q2 = 1/(4 h_t2).
template <int N>
__device__ __forceinline__ void hall_current(const double* W, int QS, int oC, int oD, int oCp1, int oCm1, int oDp1,
                                             int oDm1, int oCp2, int oCm2, int oDp2, int oDm2, double idn, double q1,
                                             double q2, double Jr[3]) {
  constexpr int a1 = (N + 1) % 3, a2 = (N + 2) % 3;
  const double* Bn = W + (5 + N) * QS;
  const double* B1 = W + (5 + a1) * QS;
  const double* B2 = W + (5 + a2) * QS;
  const double dnB1 = (B1[oD] - B1[oC]) * idn, dnB2 = (B2[oD] - B2[oC]) * idn;
  const double d1Bn = ((Bn[oCp1] - Bn[oCm1]) + (Bn[oDp1] - Bn[oDm1])) * q1;
  const double d1B2 = ((B2[oCp1] - B2[oCm1]) + (B2[oDp1] - B2[oDm1])) * q1;
  const double d2Bn = ((Bn[oCp2] - Bn[oCm2]) + (Bn[oDp2] - Bn[oDm2])) * q2;
  const double d2B1 = ((B1[oCp2] - B1[oCm2]) + (B1[oDp2] - B1[oDm2])) * q2;
  Jr[0] = d1B2 - d2B1;
  Jr[1] = d2Bn - dnB2;
  Jr[2] = dnB1 - d1Bn;
}

// LIM >= 0 fixes the limiter at compile time (no branch per slope, one basic block for all eight variables);
// LIM < 0 reads it from the parameters.
// GLM = true: nine variables per cell, the scalar psi (index 8) behind the MHD ones (NEXT-1; eqs.10-11; R22).
// CGL = true: CGL MHD (NEXT-2; R24): nine variables, W = (rho, v, p_par, B, p_perp), HLL only.
// GLM and CGL (eqs.19-23; R30): ten variables, A at index 8, psi at index 9.
// HALL = true: Hall MHD (A8; R15): HLL with the Hall velocity in the induction and energy fluxes and
// max(c_f, c_w) in the Davis speeds; the face current needs B one zone around every face, so the y-halo rows keep
// three planes, carry their x-halo corners, and a few more hand-overs guard the planes k-1 and k+1.
template <int TY, int RIEMANN, int LIM, int MINB, bool GLM = false, bool CGL = false, bool HALL = false>
__global__ void __launch_bounds__(32 * (TY + 1), MINB) stage3d_kernel(const __grid_constant__ StageParams P) {
  static_assert(!(CGL && RIEMANN != 0) && !(HALL && (CGL || RIEMANN != 0)), "combination not built");
  constexpr int NV = 8 + (GLM ? 1 : 0) + (CGL ? 1 : 0);      // CGL's A is index 8; psi is always the last variable
  constexpr int NHB = HALL ? 3 : 2;
  using SM = Stage3dSmem<TY, NV, NHB>;
  constexpr int NT = SM::NT, PL = SM::PL, SB = SM::SB, QS = SM::QS, YS = SM::YS, ZS = SM::ZS, XS = SM::XS;
  extern __shared__ __align__(16) double smem[];
  double* const W = smem;                    // [8][QS]  primitives: ring planes + two y-halo buffers
  // Y row r holds, in turn, the right state  W(r) - dW_y(r)/2  of row r (fixed variable order; written in phase A by
  // the owner of row r, H for r = TY) and the y flux through face r-1/2 (rotated order, n = 1; written over it in phase
  // B1 by the only reader of that state, the owner of row r-1, H for r = 0)
  double* const Y = smem + SM::OFF_Y;        // [8][YS]
  double* const WLz = smem + SM::OFF_WLZ;    // [8][ZS]  z: left state of the next face                (fixed order)
  double* const ACC = smem + SM::OFF_ACC;    // [8][ZS]  -dt (flux differences) of the plane being assembled (fixed order)
  double* const XR = smem + SM::OFF_XR;      // [8][XS]  right state of cell x = 32, per row
  double* const XF = smem + SM::OFF_XF;      // [8][XS]  x flux through face -1/2, per row
  int* const prog = reinterpret_cast<int*>(smem + SM::OFF_PROG);   // [TY+1] phases completed, per warp
  unsigned long long* const hbar = reinterpret_cast<unsigned long long*>(smem + SM::OFF_MBAR);

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const bool owner = wid < TY;
  const double dtf = *P.dt_ptr, dt = dtf * P.cdt;      // full step, and the stage's share of it (R27)
  const double cx = dt * P.idx, cy = dt * P.idy, cz = dt * P.idz;
  const bool two = (P.a0 != 0.0);                       // second SSP stage: Uout = a1 (U0 + Uin + dt L)
  const double c0 = two ? P.a1 : 1.0;
  const int limiter = (LIM >= 0) ? LIM : P.limiter;
  const double beta2 = 2.0 * P.beta;
  // GLM (R22): c_h of this step from the device scalar; the source term multiplies psi by exp(-dt c_h / 0.18)
  // (c_h^2 / c_p^2 with c_p^2 = 0.18 c_h) in the stage that completes the step
  const double ch = GLM ? *P.ch_ptr : 0.0;
  const double ich = GLM ? 1.0 / ch : 0.0;
  const double decay = (GLM && P.last_stage) ? exp(-dtf * ch / 0.18) : 1.0;

  // Work = (x-y tile, plane) pairs, split EVENLY over the CTAs of a one-wave grid (no tail wave, whatever the grid
  // size).  First the rounds: in round r CTA b takes the whole column of tile r * grid + b, so the CTAs resident at
  // one time march side by side through neighbouring tiles and the halo cells they share are served by L2, not by
  // DRAM.  Then the tiles that do not fill a round: their planes, in tile-major order, are cut into equal ranges,
  // and a CTA walks its range as segments [k0, k1) of consecutive planes of one tile.
  double vmx = 0.0;
  int bad = 0;
  int ph = 0;                                     // phases this warp has completed (the same count in every warp)
  if (tid < 16) prog[tid] = 0;
  if (tid == 0) mbar_init(hbar, 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();
  // bulk copies need 16-byte aligned rows: an even padded row length (the arrays start 256-byte aligned and every
  // variable, plane and tile starts at an even element); odd nx falls back to the eight-byte copies
  // Used by the Hall variant only (its halo rows need their corners and are copied on H's critical path: 5.16 -> 5.04 ms
  // per step at 256^3); the ideal-MHD kernel measured slower with them (31.3 -> 33.6 ms at 512^3, profiles/r2_stage3d.md).
  constexpr bool BULK = HALL;
  const bool bulk_ok = BULK && ((P.nxp & 1) == 0) && ((P.sq & 1) == 0);
  uint32_t hpar = 0;                              // parity of the mbarrier phase H waits for next
  bool hpend = false;                             // a bulk transfer is in flight
  const int ntile = P.ntx * P.nty;
  const int nround = ntile / (int)gridDim.x;
  const long long wtot = (long long)(ntile - nround * (int)gridDim.x) * P.nz;
  long long wpos = wtot * blockIdx.x / gridDim.x;
  const long long wend = wtot * (blockIdx.x + 1) / gridDim.x;
  for (int round = 0; round < nround || wpos < wend; ++round) {
  int tile, k0, k1;
  if (round < nround) {
    tile = round * (int)gridDim.x + (int)blockIdx.x;
    k0 = 0;
    k1 = P.nz;
  } else {
    const int rt = (int)(wpos / P.nz);
    tile = nround * (int)gridDim.x + rt;
    k0 = (int)(wpos - (long long)rt * P.nz);
    k1 = (int)min((long long)P.nz, k0 + (wend - wpos));
    wpos += k1 - k0;
  }
  const int x0 = (tile % P.ntx) * TX, y0 = (tile / P.ntx) * TY;
  const int tw = min(TX, P.nx - x0), th = min(TY, P.ny - y0);
  const bool cell_ok = owner && lane < tw && wid < th;
  // padded-array bounds of what this thread copies (ragged tiles only)
  const bool own_in = owner && (x0 + lane + 2 < P.nxp) && (y0 + wid + 2 < P.nyp);
  const int own_off = wid * RS + lane + 2;              // own cell inside a ring plane (owners)
  const long long own_g = (long long)(y0 + wid + 2) * P.sy + (x0 + lane + 2);   // + (p+2) * sz

  auto slot_of = [](int p) { return ((p + 3) % 3) * PL; };     // p >= -2
  auto conv_in_place = [&](int off) {
    if (CGL) {
      double u[9], w[9];
#pragma unroll
      for (int q = 0; q < 9; ++q) u[q] = W[q * QS + off];
      cgl_cons_to_prim(u, w, P.ph.cgl_form);
#pragma unroll
      for (int q = 0; q < 9; ++q)
        if (q < 5 || q > 7) W[q * QS + off] = w[q];       // B is its own primitive: the copied value stays
    } else {
      double u[8], w[8];                     // the GLM scalar (index 8) is its own primitive
#pragma unroll
      for (int q = 0; q < 8; ++q) u[q] = W[q * QS + off];
      cons_to_prim(P.ph, u, w);
#pragma unroll
      for (int q = 0; q < 5; ++q) W[q * QS + off] = w[q];       // B is its own primitive: the copied value stays
    }
  };
  auto copy_cell = [&](int off, long long g) {
    const double* src = P.Uin + g;           // running pointer: one 64-bit add per variable
#pragma unroll
    for (int q = 0; q < NV; ++q, src += P.sq) cp_async8(W + q * QS + off, src);
  };
  // H's halo cells of plane p.  The four y-halo rows: one pass per row, lane = column of the tile (the row's own
  // x-halo corners are never read).  The x-halo columns of the ring rows: four cells per row, ceil(4 TY / 32) passes.
  // Fully unrolled with closed-form offsets: this work sits on H's critical path in phase B.
  // Hall: also the x-halo corners (columns -1 and 32) of the four y-halo rows, for the transverse differences of J
  constexpr int NHC = (4 * TY + (HALL ? 8 : 0) + 31) / 32;
  auto hbuf_of = [](int p) { return 3 * PL + ((p + NHB) % NHB) * SB; };       // y-halo rows of plane p >= -2
  auto h_cells = [&](int p, int slot, bool rows, auto&& fn) {
    const long long gp = (long long)(p + 2) * P.sz + x0;
    const bool xin = x0 + lane + 2 < P.nxp;
    if (rows) {
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int j = (r < 2) ? r - 2 : TY + r - 2;
        if (xin && y0 + j + 2 < P.nyp)
          fn(hbuf_of(p) + r * RS + lane + 2, gp + (long long)(y0 + j + 2) * P.sy + lane + 2);
      }
    }
#pragma unroll
    for (int i = 0; i < NHC; ++i) {
      const int t = lane + 32 * i;
      if (t < 4 * TY) {
        const int j = t >> 2, cc = t & 3, c = (cc < 2) ? cc : 32 + cc;
        if (x0 + c < P.nxp && y0 + j + 2 < P.nyp) fn(slot + j * RS + c, gp + (long long)(y0 + j + 2) * P.sy + c);
      } else if (HALL && rows && t < 4 * TY + 8) {
        const int u = t - 4 * TY, r = u >> 1, c = (u & 1) ? 34 : 1, j = (r < 2) ? r - 2 : TY + r - 2;
        if (x0 + c < P.nxp && y0 + j + 2 < P.nyp) fn(hbuf_of(p) + r * RS + c, gp + (long long)(y0 + j + 2) * P.sy + c);
      }
    }
  };
  // the four y-halo rows of plane p as bulk copies: lane = (row r, variable q), 4 x 8 = 32 (a ninth variable: second
  // pass); each moves the row's 36 cells (fewer at the right end of the grid), x halo and corners included
  auto h_rows_bulk = [&](int p) {
    const long long gp = (long long)(p + 2) * P.sz + x0;
    const int ncell = min(RS, P.nxp - x0) & ~1;
    uint32_t total = 0;
#pragma unroll
    for (int pass = 0; pass < (NV + 7) / 8; ++pass) {
      const int r = lane & 3, q = (lane >> 2) + 8 * pass, j = (r < 2) ? r - 2 : TY + r - 2;
      const bool ok = q < NV && y0 + j + 2 < P.nyp && ncell > 0;
      total += __reduce_add_sync(0xffffffffu, ok ? (uint32_t)ncell * 8u : 0u);
    }
    if (total == 0) return;
    fence_proxy_async();
    if (lane == 0) mbar_arrive_expect_tx(hbar, total);
    __syncwarp();
#pragma unroll
    for (int pass = 0; pass < (NV + 7) / 8; ++pass) {
      const int r = lane & 3, q = (lane >> 2) + 8 * pass, j = (r < 2) ? r - 2 : TY + r - 2;
      if (q < NV && y0 + j + 2 < P.nyp && ncell > 0)
        bulk_g2s(W + q * QS + hbuf_of(p) + r * RS, P.Uin + q * P.sq + gp + (long long)(y0 + j + 2) * P.sy, (uint32_t)ncell * 8u, hbar);
    }
    hpend = true;
  };
  // H: every copy it has issued has landed (eight-byte copies of this thread; the bulk transfer of the warp)
  auto h_wait = [&]() {
    cp_async_wait_all();
    if (hpend) {
      int spins = 0;
      while (!mbar_test_wait(hbar, hpar)) {      // bounded like the hand-over waits: a lost transfer must not hang the GPU
        __nanosleep(20);
        if (++spins > (1 << 22)) { atomicOr(P.flag, 2); break; }
      }
      hpar ^= 1u;
      hpend = false;
    }
  };
  auto h_copy = [&](int p, int slot) {
    if (bulk_ok) h_rows_bulk(p);
    h_cells(p, slot, !bulk_ok, [&](int off, long long g) { copy_cell(off, g); });
  };
  auto h_conv = [&](int p, int slot) { h_cells(p, slot, true, [&](int off, long long) { conv_in_place(off); }); };

  // ---- prologue: everything step k0 needs that the steady state would have produced earlier ----
  for (int i = tid; i < NV * QS; i += NT) W[i] = 1.0;           // cells outside the padded array (ragged tiles)
  __syncthreads();
  if (owner) {
    if (own_in) {
      copy_cell(slot_of(k0 - 2) + own_off, own_g + (long long)k0 * P.sz);
      copy_cell(slot_of(k0 - 1) + own_off, own_g + (long long)(k0 + 1) * P.sz);
      copy_cell(slot_of(k0) + own_off, own_g + (long long)(k0 + 2) * P.sz);
    }
    cp_async_wait_all();
    if (own_in) {
      conv_in_place(slot_of(k0 - 2) + own_off);
      conv_in_place(slot_of(k0 - 1) + own_off);
      conv_in_place(slot_of(k0) + own_off);
    }
    const int ca = slot_of(k0 - 2) + own_off, cb = slot_of(k0 - 1) + own_off, cc = slot_of(k0) + own_off;
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      const double a = W[q * QS + ca], b = W[q * QS + cb], c = W[q * QS + cc];
      double lo, hi;
      plm_faces(limiter, beta2, a, b, c, lo, hi);
      WLz[q * ZS + tid] = hi;
    }
    // plane k0+1 goes into the slot plane k0-2 just left (own cell only: no other thread touches it)
    if (own_in) copy_cell(slot_of(k0 + 1) + own_off, own_g + (long long)(k0 + 3) * P.sz);
  } else {
    if (HALL) { h_copy(k0 - 1, slot_of(k0 - 1)); h_wait(); }   // only its B is read (current at face k0 - 1/2): no conversion
    h_copy(k0, slot_of(k0));
    h_wait();
    h_conv(k0, slot_of(k0));
    if (!HALL && k0 + 1 < k1) h_copy(k0 + 1, slot_of(k0 + 1));
  }
  __syncthreads();

  // ring slots of planes k-1, k, k+1 (rotated at the end of a step) and the own cell's offset in plane k-1
  int sm = slot_of(k0 - 1), sc = slot_of(k0), sp = slot_of(k0 + 1);
  long long gm = own_g + (long long)(k0 + 1) * P.sz;
  for (int k = k0; k <= k1; ++k, gm += P.sz) {
    const bool full = k < k1;       // plane k gets its x and y sweeps (step k1 only closes plane k1-1)
    const bool emit = k > k0;       // plane k-1 is completed in this step
    const int hb = hbuf_of(k);                            // y-halo rows of plane k
    const int ph0 = ph;                                   // sub-phases completed when this plane starts
    double ua[NV], ub[NV];
    // face states and flux of the task in hand.  L outlives a sub-phase once: the y slope formed in phase A leaves the
    // left state of face j+1/2 in it for phase B1 (no copy at the hand-over between the two)
    double L[NV], R[NV], F[NV], Jr[3];

#pragma unroll
    for (int s = 0; s < 3; ++s) {
      bool flux = false;
      // ---- hand-over: what this sub-phase reads must be published, what it overwrites must have been read.  Every
      //      wait is on a sub-phase EARLIER than the one about to start, so the waits cannot form a cycle.
      if (s == 0) {
        // phase A.  owner j: the row below is done with plane k-1 (it has read Y[j], the state this phase replaces,
        // and converted its ring row); the row above has converted its ring row of plane k (its phase A of plane
        // k-1), H its y-halo rows (all of plane k-1).  H: every owner is done with XR / XF / Y[TY] / the halo columns.
        if (owner) {
          await(prog + (wid == 0 ? TY : wid - 1), ph0, P.flag);
          await(prog + (wid == TY - 1 ? TY : wid + 1), wid == TY - 1 ? ph0 : ph0 - 2, P.flag);
        } else {
          await(prog + min(lane, TY - 1), ph0, P.flag);
          __syncwarp();
          // Hall: the owners read the B of plane k-1's halo cells until the end of their phase B2 (currents at the x
          // faces), so the halo cells of plane k+1 cannot take that slot before now; they are read (raw B) from phase
          // B1 on, so the copies are awaited before this phase is published
          if (HALL && k + 1 <= k1) h_copy(k + 1, sp);
        }
      } else if (s == 1) {
        // phase B1.  owner j: the right state in Y[j+1] (phase A of the row above, H for the top row).
        // H: Y[0] (owner 0).
        if (owner) await(prog + (wid == TY - 1 ? TY : wid + 1), ph0 + 1, P.flag);
        else await(prog + 0, ph0 + 1, P.flag);
      } else {
        // phase B2.  owner j: XR / XF and the halo columns (phase A of H).
        // H: both edge owners are done with the y-halo rows H is about to refill (their phase A).
        if (owner) {
          await(prog + TY, ph0 + 1, P.flag);
        } else if (!HALL) {
          await(prog + 0, ph0 + 1, P.flag);
          await(prog + TY - 1, ph0 + 1, P.flag);
        }
      }
      // ------------------------------------------------------------------ prepare the face states of task s
      if (owner) {
        if (s == 0) {
          cp_async_wait_all();
          if (own_in) conv_in_place(sp + own_off);          // A1 of the own cell of plane k+1
          // A2 (z): slope of plane k;  face k-1/2:  L carried,  R = W(k) - dW/2
#pragma unroll
          for (int r = 0; r < NV; ++r) {
            const int v = rv(r, 2);
            const double a = W[v * QS + sm + own_off], b = W[v * QS + sc + own_off], c = W[v * QS + sp + own_off];
            double lo, hi;
            plm_faces(limiter, beta2, a, b, c, lo, hi);
            L[r] = WLz[v * ZS + tid];
            R[r] = lo;
            WLz[v * ZS + tid] = hi;
          }
          if (HALL) {
            // face k-1/2 of the own column: C = plane k-1, D = plane k; transverse x (lanes), y (rows; halo rows at
            // the tile's edges)
            const int oC = sm + own_off, oD = sc + own_off;
            const int hm = hbuf_of(k - 1) + lane + 2;
            const int oCym = (wid == 0) ? hm + RS : oC - RS, oCyp = (wid == TY - 1) ? hm + 2 * RS : oC + RS;
            const int oDym = (wid == 0) ? hb + RS + lane + 2 : oD - RS, oDyp = (wid == TY - 1) ? hb + 2 * RS + lane + 2 : oD + RS;
            hall_current<2>(W, QS, oC, oD, oC + 1, oC - 1, oD + 1, oD - 1, oCyp, oCym, oDyp, oDym, P.idz, 0.25 * P.idx,
                            0.25 * P.idy, Jr);
          }
          flux = true;
        } else if (full) {
          if (s == 1) {
#pragma unroll
            for (int r = 0; r < NV; ++r) {
              R[r] = Y[rv(r, 1) * YS + (wid + 1) * 32 + lane];      // L: left there by phase A
            }
            if (HALL) {
              // face j+1/2: C = own cell, D = the row above (halo row TY for the top row); transverse z (planes
              // k-1, k+1), x (lanes; the halo rows carry their x corners)
              const bool top = (wid == TY - 1);
              const int oC = sc + own_off, oD = top ? hb + 2 * RS + lane + 2 : oC + RS;
              const int oCzp = sp + own_off, oCzm = sm + own_off;
              const int oDzp = top ? hbuf_of(k + 1) + 2 * RS + lane + 2 : oCzp + RS;
              const int oDzm = top ? hbuf_of(k - 1) + 2 * RS + lane + 2 : oCzm + RS;
              hall_current<1>(W, QS, oC, oD, oCzp, oCzm, oDzp, oDzm, oC + 1, oC - 1, oD + 1, oD - 1, P.idy, 0.25 * P.idz,
                              0.25 * P.idx, Jr);
            }
          } else {
            // A2 (x): own slope; the right state of face i+1/2 comes from lane i+1 (lane 31: from H)
            const int c = sc + own_off;
#pragma unroll
            for (int r = 0; r < NV; ++r) {
              const double a = W[r * QS + c - 1], b = W[r * QS + c], cc = W[r * QS + c + 1];
              double lo, hi;
              plm_faces(limiter, beta2, a, b, cc, lo, hi);
              L[r] = hi;
              const double rn = __shfl_down_sync(0xffffffffu, lo, 1);
              R[r] = (lane == 31) ? XR[r * XS + wid] : rn;
            }
            if (HALL) {
              // face i+1/2: C = own cell, D = the next column (x-halo column for lane 31); transverse y (rows), z
              const int oC = c, oD = c + 1;
              const int oCym = (wid == 0) ? hb + RS + lane + 2 : oC - RS, oCyp = (wid == TY - 1) ? hb + 2 * RS + lane + 2 : oC + RS;
              hall_current<0>(W, QS, oC, oD, oCyp, oCym, oCyp + 1, oCym + 1, sp + own_off, sm + own_off, sp + own_off + 1,
                              sm + own_off + 1, P.idx, 0.25 * P.idy, 0.25 * P.idz, Jr);
            }
          }
          flux = true;
        }
      } else if (full) {
        if (s == 0) {
          // row TY: right state for the owners of row TY-1
          {
            const int cm = sc + (TY - 1) * RS + lane + 2, c0r = hb + 2 * RS + lane + 2, cp = hb + 3 * RS + lane + 2;
#pragma unroll
            for (int q = 0; q < NV; ++q) {
              const double a = W[q * QS + cm], b = W[q * QS + c0r], c = W[q * QS + cp];
              double lo, hi;
              plm_faces(limiter, beta2, a, b, c, lo, hi);
              Y[q * YS + TY * 32 + lane] = lo;
            }
          }
          // column x = 32: right state for lane 31 of every row
          if (lane < TY) {
            const int c = sc + lane * RS + 34;
#pragma unroll
            for (int q = 0; q < NV; ++q) {
              const double a = W[q * QS + c - 1], b = W[q * QS + c], cc = W[q * QS + c + 1];
              double lo, hi;
              plm_faces(limiter, beta2, a, b, cc, lo, hi);
              XR[q * XS + lane] = lo;
            }
          }
          // face x = -1/2 of every row: lanes 0..15 hold cell -1 (left state), lanes 16..31 cell 0 (right state)
          {
            const int row = min(lane & 15, TY - 1), half = lane >> 4;
            const int c = sc + row * RS + 1 + half;
#pragma unroll
            for (int r = 0; r < NV; ++r) {
              const double a = W[r * QS + c - 1], b = W[r * QS + c], cc = W[r * QS + c + 1];
              double lo, hi;
              plm_faces(limiter, beta2, a, b, cc, lo, hi);
              L[r] = hi;
              R[r] = __shfl_down_sync(0xffffffffu, lo, 16);
            }
            if (HALL) {
              // face x = -1/2 of row `row`: C = column -1, D = column 0.  D's cell of plane k+1 belongs to an owner
              // that may still be converting it: its B comes straight from the stage input (the copy that brought
              // it into shared memory has already pulled the line into L2)
              const int oC = sc + row * RS + 1, oD = oC + 1;
              const int oCym = (row == 0) ? hb + RS + 1 : oC - RS, oCyp = (row == TY - 1) ? hb + 2 * RS + 1 : oC + RS;
              const int oCzm = sm + row * RS + 1;
              // B_x, B_y of columns -1 and 0 in plane k+1 straight from the stage input (the halo copies of that plane
              // were issued a moment ago; column 0 belongs to an owner that may still be converting it)
              double bc[2] = {0.0, 0.0}, bd[2] = {0.0, 0.0};
              if (y0 + row + 2 < P.nyp) {
                const double* g = P.Uin + 5 * P.sq + (long long)(k + 3) * P.sz + (long long)(y0 + row + 2) * P.sy + (x0 + 1);
                bc[0] = __ldg(g); bc[1] = __ldg(g + P.sq);
                bd[0] = __ldg(g + 1); bd[1] = __ldg(g + P.sq + 1);
              }
              const double* Bx = W + 5 * QS; const double* By = W + 6 * QS; const double* Bz = W + 7 * QS;
              const double q1 = 0.25 * P.idy, q2 = 0.25 * P.idz;
              const double dnB1 = (By[oD] - By[oC]) * P.idx, dnB2 = (Bz[oD] - Bz[oC]) * P.idx;
              const double d1Bn = ((Bx[oCyp] - Bx[oCym]) + (Bx[oCyp + 1] - Bx[oCym + 1])) * q1;
              const double d1B2 = ((Bz[oCyp] - Bz[oCym]) + (Bz[oCyp + 1] - Bz[oCym + 1])) * q1;
              const double d2Bn = ((bc[0] - Bx[oCzm]) + (bd[0] - Bx[oCzm + 1])) * q2;
              const double d2B1 = ((bc[1] - By[oCzm]) + (bd[1] - By[oCzm + 1])) * q2;
              Jr[0] = d1B2 - d2B1; Jr[1] = d2Bn - dnB2; Jr[2] = dnB1 - d1Bn;
            }
          }
          flux = true;
        } else if (s == 1) {
          // row -1: flux through face y = -1/2
          const int cm = hb + lane + 2, c0r = hb + RS + lane + 2, cp = sc + lane + 2;
#pragma unroll
          for (int r = 0; r < NV; ++r) {
            const int v = rv(r, 1);
            const double a = W[v * QS + cm], b = W[v * QS + c0r], c = W[v * QS + cp];
            double lo, hi;
            plm_faces(limiter, beta2, a, b, c, lo, hi);
            L[r] = hi;
            R[r] = Y[v * YS + lane];
          }
          if (HALL) {
            // face y = -1/2: C = halo row -1, D = row 0; transverse z (the halo rows of planes k-1, k+1; owner 0's
            // cells), x (the halo row carries its x corners)
            const int oC = c0r, oD = cp;
            const int oCzp = hbuf_of(k + 1) + RS + lane + 2, oCzm = hbuf_of(k - 1) + RS + lane + 2;
            hall_current<1>(W, QS, oC, oD, oCzp, oCzm, sp + lane + 2, sm + lane + 2, oC + 1, oC - 1, oD + 1, oD - 1, P.idy,
                            0.25 * P.idz, 0.25 * P.idx, Jr);
          }
          flux = true;
        }
      }

      // ------------------------------------------------------------------ A3 + A4: the one Riemann call site
      if (GLM && flux) {
        // (B_n, psi) at the face from the 2x2 linear Riemann problem (speeds -+c_h); the MHD solver sees B_n* on
        // both sides, and  F[B_n] = psi*,  F[psi] = c_h^2 B_n*   (rotated slot 5 = B_n in every task)
        const double bns = 0.5 * (L[5] + R[5]) - 0.5 * (R[NV - 1] - L[NV - 1]) * ich;
        const double pss = 0.5 * (L[NV - 1] + R[NV - 1]) - 0.5 * ch * (R[5] - L[5]);
        L[5] = bns; R[5] = bns;
        if (CGL) flux_hll_cgl(L, R, F, P.ph.cgl_form);                         // CGL + GLM (R30): CGL's flux with B_n*
        else riemann_flux<RIEMANN, HALL>(P.ph, L, R, HALL ? Jr : nullptr, F);  // Hall + GLM (R29): Hall flux with B_n*
        F[5] = pss;
        F[NV - 1] = ch * ch * bns;
      } else if (flux) {
        if (CGL) flux_hll_cgl(L, R, F, P.ph.cgl_form);
        else riemann_flux<RIEMANN, HALL>(P.ph, L, R, HALL ? Jr : nullptr, F);
      }

      // ------------------------------------------------------------------ consume the flux of task s
      if (owner) {
        if (s == 0) {
          // Uin (+U0) of the own cell of plane k-1, needed when the plane is completed below: the loads are in
          // flight while the y slopes are formed.  Uniform branches on the stage kind: the first stage issues no U0
          // loads and no selects.
#pragma unroll
          for (int q = 0; q < NV; ++q) { ua[q] = 0.0; ub[q] = 0.0; }
          if (emit && cell_ok) {
            const double* pa = P.Uin + gm;
            const double* pb = P.U0 + gm;
            if (two) {
#pragma unroll
              for (int q = 0; q < NV; ++q, pa += P.sq, pb += P.sq) { ua[q] = __ldg(pa); ub[q] = *pb; }
            } else {
#pragma unroll
              for (int q = 0; q < NV; ++q, pa += P.sq) ua[q] = __ldg(pa);
            }
          }
          if (full) {
            // A2 (y): own slope -> right state for the row below, left state kept for phase B1
            const int c = sc + own_off;
            const int cm = (wid == 0) ? hb + RS + lane + 2 : c - RS;
            const int cp = (wid == TY - 1) ? hb + 2 * RS + lane + 2 : c + RS;
#pragma unroll
            for (int r = 0; r < NV; ++r) {
              const int v = rv(r, 1);
              const double a = W[v * QS + cm], b = W[v * QS + c], cc = W[v * QS + cp];
              double lo, hi;
              plm_faces(limiter, beta2, a, b, cc, lo, hi);
              Y[v * YS + wid * 32 + lane] = lo;
              L[r] = hi;
            }
          }
          // A5 (z) + A6: plane k-1 is complete:  Uout = a1 ((a0/a1) U0 + Uin + [-dt (flux differences)]);  the
          // accumulator of plane k starts with its low z face.  The flux terms are summed on their own and the two
          // z terms are the same rounded product, so a uniform state stays bitwise fixed (pin P1).
          double* po = P.Uout + gm;                                       // own cell of plane k-1
          double o[NV];
#pragma unroll
          for (int v = 0; v < NV; ++v, po += P.sq) {
            constexpr int inv2[10] = {0, 2, 3, 1, 4, 6, 7, 5, 8, 9};         // rv(inv2[v], 2) == v
            const double t = cz * F[inv2[v]];
            const double d = ACC[v * ZS + tid] - t;
            o[v] = c0 * ((two ? fma(P.r0, ub[v], ua[v]) : ua[v]) + d);
            if (GLM && v == NV - 1) o[v] *= decay;                        // eq.11's source, integrated exactly
            if (CGL && v == 8 && P.last_stage && P.relax > 0.0 && emit && cell_ok)
              o[v] = cgl_relaxed_alog(P.relax, o, P.ph.cgl_form);                        // eqs.31-33: E stays, A_log moves
            if (emit && cell_ok) *po = o[v];
            ACC[v * ZS + tid] = t;
          }
          if (P.vnext != nullptr && emit && cell_ok) {                    // A7 on the values just stored
            const double sp = cell_speed_inline<HALL>(P.ph, o);
            if (sp < 0.0) bad = 1; else vmx = dmax(vmx, sp);
          }
        } else if (full) {
          if (s == 1) {
#pragma unroll
            for (int r = 0; r < NV; ++r) Y[r * YS + (wid + 1) * 32 + lane] = F[r];
          } else {
            // A5 (x): low-face flux from lane i-1 (lane 0: from H)
            double dFx[NV];
#pragma unroll
            for (int r = 0; r < NV; ++r) {
              const double fl = __shfl_up_sync(0xffffffffu, F[r], 1);
              dFx[r] = F[r] - ((lane == 0) ? XF[r * XS + wid] : fl);
            }
            // Hall: the row below reads this row's cell of plane k-1 until the end of its phase B1 (current at its y face)
            if (HALL) await(prog + (wid == 0 ? TY : wid - 1), ph0 + 2, P.flag);
            // own cell of plane k+2 -> the slot plane k-1 left in phase A
            if (own_in && k + 2 <= k1 + 1) copy_cell(sm + own_off, gm + 3 * P.sz);
            // second SSP stage: U0 of plane k+1 is first touched two steps from now; pull its lines into L2 (one
            // lane per 64 bytes)
            if (two && cell_ok && (lane & 7) == 0 && k + 1 < k1) {
#pragma unroll
              for (int q = 0; q < NV; ++q) prefetch_l2(P.U0 + q * P.sq + gm + 2 * P.sz);
            }
            // A5 (y): Y[j+1] holds this row's own flux (phase B1), Y[j] the flux of the row below (its phase B1)
            if (!HALL) await(prog + (wid == 0 ? TY : wid - 1), ph0 + 2, P.flag);
#pragma unroll
            for (int v = 0; v < NV; ++v) {
              constexpr int inv1[10] = {0, 3, 1, 2, 4, 7, 5, 6, 8, 9};       // rv(inv1[v], 1) == v
              const int r = inv1[v];
              const double dFy = Y[r * YS + (wid + 1) * 32 + lane] - Y[r * YS + wid * 32 + lane];
              ACC[v * ZS + tid] = fma(-cx, dFx[v], fma(-cy, dFy, ACC[v * ZS + tid]));
            }
          }
        }
      } else {
        if (s == 0) {
          if (full && lane < 16 && lane < TY) {
#pragma unroll
            for (int r = 0; r < NV; ++r) XF[r * XS + lane] = F[r];
          }
          if (HALL) h_wait();                  // plane k+1's halo cells have landed when this phase is published
        } else if (s == 1) {
          if (full) {
#pragma unroll
            for (int r = 0; r < NV; ++r) Y[r * YS + lane] = F[r];
          }
        } else {
          // A1 for the halo cells of plane k+1 (copies issued one phase B2 ago), then the copies for plane k+2
          if (!HALL) h_wait();
          if (k + 1 < k1) h_conv(k + 1, sp);
          if (!HALL && k + 2 < k1) h_copy(k + 2, sm);
        }
      }
      publish(prog + wid, ++ph, lane);   // end of phase A, B1, B2
    }
    { const int t = sm; sm = sc; sc = sp; sp = t; }
  }
  if (owner) cp_async_wait_all(); else h_wait();
  __syncthreads();                 // the next segment reuses the shared buffers
  }
  if (P.vnext != nullptr) {
    vmx = warp_max(vmx);
    bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
      if (vmx > 0.0) atomicMax(P.vnext, (unsigned long long)__double_as_longlong(vmx));
      if (bad) atomicOr(P.flag, 1);
    }
  }
}

}  // namespace agate
