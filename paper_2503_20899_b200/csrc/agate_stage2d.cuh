// agate_stage2d.cuh — warp-autonomous fused stage kernel for 2-D grids, ideal and Hall MHD,
// sm_100a.
//
// Same arithmetic as the other two stage kernels; what differs is that a WARP, not a CTA, is the unit of work:
//   * a warp owns a strip of 30 columns and marches along y.  Lanes 1..30 own the strip's cells of the current row,
//     lanes 0 and 31 hold the strip's x-halo cells (x = -1, 30): they compute slopes and face states like the others
//     but store nothing.  30 of 32 lanes do useful updates; in exchange there is NO synchronisation between warps at
//     all (no barrier, no flag) and no helper warp.
//   * x: the right state of face i+1/2 and the flux of face i-1/2 travel by warp shuffles.
//   * y: private column, one row behind (like z in stage3d_kernel): step j computes F(j-1/2) from rows j-1, j, j+1 and
//     completes row j-1.  The left state W(j-1)+dW/2 and the low-face flux are carried in per-lane shared slots,
//     the accumulator in registers.
//   * conserved rows arrive by cp.async one step ahead in a private ring of 4 rows x 34 cells and are turned into
//     primitives in place (A1); the raw Uin (+U0, copied straight into the same slot) of the own cell is kept for A6.
//   * work = (strip, row) pairs over the warps of a one-wave grid: every strip cut into the same row ranges,
//     consecutive warps on consecutive strips (L2 serves the shared halo columns).
//   * A7 of the next step rides in the last stage, as in stage3d_kernel (ideal, Hall, GLM; CGL keeps the dt_kernel pass).
//   * Hall (A8): the face current comes from the cell-centred B of the three ring rows around the face.
//
// Shared memory per warp: ring 4 x 8 x 34, two y carries 8 x 32, raw U 2 x 8 x 32  =  16.5 KB;  6 warps per CTA,
// 2 CTAs per SM (12 warps, <= 168 registers).  Nine / ten variables: one CTA of 12 / 11 warps per SM.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "agate_stage3d.cuh"

namespace agate {

constexpr int SW2 = 30;        // cells a warp updates per row
constexpr int RW2 = 34;        // cells per ring row: x = xs-2 .. xs+31
constexpr int NW2 = 6;         // warps per CTA of the 8-variable kernels

// GLM = true: nine variables per cell, the scalar psi (index 8) behind the MHD ones (NEXT-1; eqs.10-11; R22)
template <int NVAR>
struct Stage2dSmem {
  static constexpr int NV = NVAR;                   // 8; 9 with GLM or CGL; 10 with both (A at 8, psi at 9)
  // warps per CTA.  The warps are autonomous, so only their number per SM matters: 8 variables 2 CTAs x 6 warps; with
  // 9 (10) variables a warp's buffers take 18.6 (20.6) KB and two CTAs would hold 2 x 5 warps, so ONE CTA of 12 (11) warps
  // fills the 227 KB instead
  static constexpr int NW = (NVAR == 8) ? 6 : ((NVAR == 9) ? 12 : 11);
  static constexpr int MINB = (NVAR == 8) ? 2 : 1;  // CTAs per SM
  static constexpr int RING = 4 * NV * RW2;         // [slot][q][c]
  static constexpr int OFF_WLY = RING;              // [q][lane]
  static constexpr int OFF_FYL = OFF_WLY + NV * 32;
  static constexpr int OFF_URAW = OFF_FYL + NV * 32; // [2][q][lane]
  static constexpr int PER_WARP = OFF_URAW + 2 * NV * 32;
  static constexpr size_t BYTES = sizeof(double) * (size_t)PER_WARP * NW;
};

// CGL = true: CGL MHD (NEXT-2; R24): nine variables, W = (rho, v, p_par, B, p_perp), HLL only
template <int RIEMANN, int LIM, bool HALL, bool GLM, bool CGL = false>
__global__ void __launch_bounds__(32 * Stage2dSmem<8 + (GLM ? 1 : 0) + (CGL ? 1 : 0)>::NW,
                                  Stage2dSmem<8 + (GLM ? 1 : 0) + (CGL ? 1 : 0)>::MINB) stage2d_kernel(const __grid_constant__ StageParams P) {
  static_assert(!(HALL && RIEMANN != 0) && !(CGL && (HALL || RIEMANN != 0)), "combination not built");
  using SM = Stage2dSmem<8 + (GLM ? 1 : 0) + (CGL ? 1 : 0)>;
  static_assert(SM::MINB * (SM::BYTES + 1024) <= 233472 && SM::BYTES <= 232448, "shared memory per SM / per CTA");
  constexpr int NV = SM::NV, NW2 = SM::NW;
  extern __shared__ __align__(16) double smem[];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  double* const ring = smem + (size_t)wid * SM::PER_WARP;      // this warp's private buffers
  double* const WLy = ring + SM::OFF_WLY;
  double* const FyL = ring + SM::OFF_FYL;
  double* const Uraw = ring + SM::OFF_URAW;

  const double dtf = *P.dt_ptr, dt = dtf * P.cdt;      // full step, and the stage's share of it (R27)
  const double cx = dt * P.idx, cy = dt * P.idy;
  const bool two = (P.a0 != 0.0);
  const double c0 = two ? P.a1 : 1.0;
  const int limiter = (LIM >= 0) ? LIM : P.limiter;
  const double beta2 = 2.0 * P.beta;
  double vmx = 0.0;
  int bad = 0;
  // GLM (R22): c_h of this step from the device scalar; the source term multiplies psi by exp(-dt c_h / 0.18)
  // (c_h^2 / c_p^2 with c_p^2 = 0.18 c_h) in the stage that completes the step
  const double ch = GLM ? *P.ch_ptr : 0.0;
  const double ich = GLM ? 1.0 / ch : 0.0;
  const double decay = (GLM && P.last_stage) ? exp(-dtf * ch / 0.18) : 1.0;

  const int nstrip = (P.nx + SW2 - 1) / SW2;
  const long long wtot = (long long)nstrip * P.ny;
  const long long nwarp = (long long)gridDim.x * NW2, gw = (long long)blockIdx.x * NW2 + wid;
  // Work = (strip, row) pairs, strip-major.  With at least one warp per strip, every strip is cut into the SAME
  // nchunk row ranges and consecutive warps take consecutive strips of one range: neighbouring strips advance side
  // by side and the halo columns they share are served by L2 (a few warps of the wave stay idle: nwarp mod nstrip).
  // Otherwise (more strips than warps) the pairs are cut into equal ranges and a warp walks its range as segments.
  long long wpos, wend;
  if (nwarp >= nstrip) {
    const int nchunk = (int)min(nwarp / nstrip, (long long)P.ny);
    const int chunk = (int)(gw / nstrip), strip = (int)(gw - (long long)chunk * nstrip);
    if (chunk < nchunk) {
      wpos = (long long)strip * P.ny + (long long)P.ny * chunk / nchunk;
      wend = (long long)strip * P.ny + (long long)P.ny * (chunk + 1) / nchunk;
    } else {
      wpos = wend = 0;
    }
  } else {
    wpos = wtot * gw / nwarp;
    wend = wtot * (gw + 1) / nwarp;
  }

  auto slot_of = [](int r) { return ((r + 4) & 3) * (NV * RW2); };     // r >= -4
  auto conv = [&](int off) {                                            // A1 in place; returns nothing
    if (CGL) {
      double u[9], w[9];
#pragma unroll
      for (int q = 0; q < 9; ++q) u[q] = ring[off + q * RW2];
      cgl_cons_to_prim(u, w, P.ph.cgl_form);
#pragma unroll
      for (int q = 0; q < 9; ++q) ring[off + q * RW2] = w[q];
    } else {
      double u[8], w[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) u[q] = ring[off + q * RW2];
      cons_to_prim(P.ph, u, w);
#pragma unroll
      for (int q = 0; q < 8; ++q) ring[off + q * RW2] = w[q];
    }
  };

  while (wpos < wend) {
    const int strip = (int)(wpos / P.ny);
    const int j0 = (int)(wpos - (long long)strip * P.ny);
    const int j1 = (int)min((long long)P.ny, j0 + (wend - wpos));
    wpos += j1 - j0;
    const int xs = strip * SW2;
    const int x = xs - 1 + lane;                                 // the lane's own column
    const bool cell_ok = lane >= 1 && lane <= SW2 && x < P.nx;
    const bool own_in = xs + lane + 1 < P.nxp;                   // own cell c = lane + 1 inside the padded row
    // extra halo cell of lanes 0 (c = 0) and 1 (c = 33)
    const int cex = (lane == 0) ? 0 : RW2 - 1;
    const bool ex_in = lane < 2 && xs + cex < P.nxp;
    const long long g_own = (long long)xs + lane + 1, g_ex = (long long)xs + cex;     // + (row + 2) * sy

    // copies of row r: the own cell (and U0 of it straight into the raw-U slot), the extra cell
    auto copy_row = [&](int r, bool with_u0) {
      const long long gr = (long long)(r + 2) * P.sy;
      const int so = slot_of(r);
      if (own_in) {
        const double* src = P.Uin + gr + g_own;
#pragma unroll
        for (int q = 0; q < NV; ++q, src += P.sq) cp_async8(ring + so + q * RW2 + lane + 1, src);
        if (two && with_u0) {
          const double* s0 = P.U0 + gr + g_own;
#pragma unroll
          for (int q = 0; q < NV; ++q, s0 += P.sq) cp_async8(Uraw + ((r & 1) * NV + q) * 32 + lane, s0);
        }
      }
      if (ex_in) {
        const double* src = P.Uin + gr + g_ex;
#pragma unroll
        for (int q = 0; q < NV; ++q, src += P.sq) cp_async8(ring + so + q * RW2 + cex, src);
      }
    };
    // A1 for row r, and the raw Uin (+U0) of the own cell for A6
    auto conv_row = [&](int r, bool keep_raw) {
      const int so = slot_of(r);
      if (own_in) {
        if (keep_raw) {
#pragma unroll
          for (int q = 0; q < NV; ++q) {
            const int a = ((r & 1) * NV + q) * 32 + lane;
            const double u = ring[so + q * RW2 + lane + 1];
            Uraw[a] = two ? fma(P.r0, Uraw[a], u) : u;          // Uin + (a0/a1) U0
          }
        }
        conv(so + lane + 1);
      }
      if (ex_in) conv(so + cex);
    };

    // ---- prologue: rows j0-2, j0-1, j0 and the carried left state of face j0-1/2 ----
#pragma unroll
    for (int i = 0; i < 4 * NV * RW2 / 32; ++i) ring[i * 32 + lane] = 1.0;     // cells outside the padded array
    __syncwarp();
    copy_row(j0 - 2, false); copy_row(j0 - 1, false); copy_row(j0, true);
    cp_async_wait_all();
    __syncwarp();
    conv_row(j0 - 2, false); conv_row(j0 - 1, false); conv_row(j0, true);
    __syncwarp();
    {
      const int c = lane + 1;
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        const double a = ring[slot_of(j0 - 2) + q * RW2 + c], b = ring[slot_of(j0 - 1) + q * RW2 + c];
        const double cc = ring[slot_of(j0) + q * RW2 + c];
        double lo, hi;
        plm_faces(limiter, beta2, a, b, cc, lo, hi);
        WLy[q * 32 + lane] = hi;
      }
    }
    copy_row(j0 + 1, true);

    double acc[NV];
#pragma unroll
    for (int q = 0; q < NV; ++q) acc[q] = 0.0;

    for (int j = j0; j <= j1; ++j) {
      const bool full = j < j1;       // row j gets its x sweep (step j1 only closes row j1-1)
      const bool emit = j > j0;       // row j-1 is completed in this step
      const int sm = slot_of(j - 1), sc = slot_of(j), sp = slot_of(j + 1);
      const int c = lane + 1;
      double L[NV], R[NV], F[NV];

      // row j+1 has had a whole step to arrive
      cp_async_wait_all();
      __syncwarp();
      conv_row(j + 1, true);
      __syncwarp();

      // ---- y task: A2 slope of row j, face j-1/2 (L carried, R = W(j) - dW/2), A3 + A4 ----
#pragma unroll
      for (int r = 0; r < NV; ++r) {
        const int v = (r < 8) ? rot_var(r, 1) : r;
        const double a = ring[sm + v * RW2 + c], b = ring[sc + v * RW2 + c], cc = ring[sp + v * RW2 + c];
        double lo, hi;
        plm_faces(limiter, beta2, a, b, cc, lo, hi);
        L[r] = WLy[v * 32 + lane];
        R[r] = lo;
        WLy[v * 32 + lane] = hi;
      }
      double Jr[3];
      if (HALL) {
        // A8 (R15): J = curl B at the y-face j-1/2 of column c from the cell-centred B of rows j-1 (sm) and j (sc)
        const double* Bx = ring + 5 * RW2; const double* By = ring + 6 * RW2; const double* Bz = ring + 7 * RW2;
        const int cL = sm + c, cR = sc + c;
        const double dyBx = (Bx[cR] - Bx[cL]) * P.idy, dyBz = (Bz[cR] - Bz[cL]) * P.idy;
        const double h = 0.25 * P.idx;
        const double dxBy = ((By[cL + 1] - By[cL - 1]) + (By[cR + 1] - By[cR - 1])) * h;
        const double dxBz = ((Bz[cL + 1] - Bz[cL - 1]) + (Bz[cR + 1] - Bz[cR - 1])) * h;
        Jr[0] = -dxBz; Jr[1] = dxBy - dyBx; Jr[2] = dyBz;              // rotated for n = 1: (Jy, Jz, Jx)
      }
      double bns = 0.0, pss = 0.0;
      if (GLM) {
        // (B_n, psi) at the face from the 2x2 linear Riemann problem (speeds -+c_h); the MHD solver sees B_n* on
        // both sides, and  F[B_n] = psi*,  F[psi] = c_h^2 B_n*
        bns = 0.5 * (L[5] + R[5]) - 0.5 * (R[NV - 1] - L[NV - 1]) * ich;
        pss = 0.5 * (L[NV - 1] + R[NV - 1]) - 0.5 * ch * (R[5] - L[5]);
        L[5] = bns; R[5] = bns;
      }
      if (CGL) flux_hll_cgl(L, R, F, P.ph.cgl_form);
      else riemann_flux<RIEMANN, HALL>(P.ph, L, R, HALL ? Jr : nullptr, F);
      if (GLM) { F[5] = pss; F[NV - 1] = ch * ch * bns; }
      {
        // A5 (y) + A6: row j-1 is complete; the accumulator of row j starts from the raw Uin (+U0)
        double* po = P.Uout + (long long)(j + 1) * P.sy + g_own;          // own cell of row j-1
        double o[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v, po += P.sq) {
          constexpr int inv1[10] = {0, 3, 1, 2, 4, 7, 5, 6, 8, 9};          // rot_var(inv1[v], 1) == v
          const int r = inv1[v];
          // the difference is formed before it meets U, so that a uniform state stays bitwise fixed (pin P1)
          o[v] = c0 * (acc[v] - cy * (F[r] - FyL[v * 32 + lane]));
          if (GLM && v == NV - 1) o[v] *= decay;                          // eq.11's source, integrated exactly
          if (CGL && v == 8 && P.last_stage && P.relax > 0.0 && emit && cell_ok)
            o[v] = cgl_relaxed_alog(P.relax, o, P.ph.cgl_form);                          // eqs.31-33: E stays, A_log moves
          if (emit && cell_ok) *po = o[v];
          FyL[v * 32 + lane] = F[r];
          acc[v] = Uraw[((j & 1) * NV + v) * 32 + lane];
        }
        if (P.vnext != nullptr && emit && cell_ok) {                      // A7 on the values just stored
          const double sp2 = cell_speed_inline<HALL>(P.ph, o);
          if (sp2 < 0.0) bad = 1; else vmx = dmax(vmx, sp2);
        }
      }
      __syncwarp();
      // row j+2 into the slot row j-2 left; its U0 into the raw slot row j just left
      if (j + 2 <= j1 + 1) copy_row(j + 2, true);

      // ---- x task: A2 own slope, right state from lane i+1, A3 + A4, low-face flux from lane i-1 ----
      if (full) {
#pragma unroll
        for (int r = 0; r < NV; ++r) {
          const double a = ring[sc + r * RW2 + c - 1], b = ring[sc + r * RW2 + c], cc = ring[sc + r * RW2 + c + 1];
          double lo, hi;
          plm_faces(limiter, beta2, a, b, cc, lo, hi);
          L[r] = hi;
          R[r] = __shfl_down_sync(0xffffffffu, lo, 1);
        }
        if (HALL) {
          // A8: J at the x-face between columns c and c+1 of row j; transverse differences from rows j-1, j+1
          const double* Bx = ring + 5 * RW2; const double* By = ring + 6 * RW2; const double* Bz = ring + 7 * RW2;
          const int cc1 = min(c + 1, RW2 - 1);                           // lane 31 has no right neighbour (its face is unused)
          const double dxBy = (By[sc + cc1] - By[sc + c]) * P.idx, dxBz = (Bz[sc + cc1] - Bz[sc + c]) * P.idx;
          const double h = 0.25 * P.idy;
          const double dyBx = ((Bx[sp + c] - Bx[sm + c]) + (Bx[sp + cc1] - Bx[sm + cc1])) * h;
          const double dyBz = ((Bz[sp + c] - Bz[sm + c]) + (Bz[sp + cc1] - Bz[sm + cc1])) * h;
          Jr[0] = dyBz; Jr[1] = -dxBz; Jr[2] = dxBy - dyBx;              // rotated for n = 0: (Jx, Jy, Jz)
        }
        if (GLM) {
          bns = 0.5 * (L[5] + R[5]) - 0.5 * (R[NV - 1] - L[NV - 1]) * ich;
          pss = 0.5 * (L[NV - 1] + R[NV - 1]) - 0.5 * ch * (R[5] - L[5]);
          L[5] = bns; R[5] = bns;
        }
        if (CGL) flux_hll_cgl(L, R, F, P.ph.cgl_form);
        else riemann_flux<RIEMANN, HALL>(P.ph, L, R, HALL ? Jr : nullptr, F);
        if (GLM) { F[5] = pss; F[NV - 1] = ch * ch * bns; }
#pragma unroll
        for (int r = 0; r < NV; ++r) {
          const double fl = __shfl_up_sync(0xffffffffu, F[r], 1);
          acc[r] -= cx * (F[r] - fl);
        }
      }
    }
    cp_async_wait_all();
    __syncwarp();
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
