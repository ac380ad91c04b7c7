// agate_stage3d.cuh — warp-specialised fused stage kernel for 3-D grids, sm_100a.
//
// Same arithmetic as stage_kernel (agate_kernels.cuh); what differs is how the CTA is organised:
//   * CTA = TY "owner" warps + 2 helper warps.  Owner warp j owns row j of a 32 x TY x-y tile and marches along z;
//     lane i owns cell (i, j).  The owner of a cell computes its limited slopes, both face states, the Riemann flux
//     through its HIGH face in x, y and z, and the flux difference (A2-A5), so slopes and fluxes are computed once.
//   * x: neighbours are lanes of the same warp -> right state and low-face flux travel by warp shuffles.  The two
//     cells outside the row (x = -1 and x = 32) belong to helper warp H0, which hands  R(32)  and  F(-1/2)  over
//     through tiny shared buffers.
//   * y: neighbours are adjacent warps -> right state and flux travel through the shared buffers YR / YF, guarded
//     by per-row mbarriers (producer = one warp, consumer = the neighbouring warp).  Row -1 belongs to H0, row TY
//     (slopes only) to helper warp H1.  There is no CTA-wide barrier in the steady state.
//   * z: private column; the left state W(k)+dW(k)/2 and the flux F(k-1/2) are carried in per-thread shared slots.
//   * H1 is also the PRODUCER: when every warp is done with plane k-1 it issues TMA bulk copies
//     (cp.async.bulk ... mbarrier::complete_tx) of the conserved rows of plane k+2 straight into the freed ring
//     slot and of the y-halo rows ("strips") of plane k+1 into the idle strip buffer.  Owners turn their own cell of
//     the raw plane into primitives in place (A1) when the z sweep first needs it; H1 converts the strips and the
//     x-halo columns.  Global-load latency is therefore never on the owners' critical path.
//   * A6: the accumulator starts as Uin (+U0 in the second SSP stage), loaded at the top of the plane.
//
// Shared memory per CTA (TY = 6): ring 3 planes x 8 x 6 x 36, strips 2 x 8 x 4 x 36, YR 8 x 8 x 32, YF 8 x 6 x 32,
// z carries 2 x 8 x 192, x hand-over buffers, 25 mbarriers  =  115 KB  ->  2 CTAs per SM.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "agate_kernels.cuh"

namespace agate {

// ---- mbarrier / TMA bulk-copy wrappers (PTX ISA: mbarrier, cp.async.bulk) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// one warp announces "my writes are published": all lanes' writes ordered before lane 0's release-arrive
__device__ __forceinline__ void warp_arrive(uint32_t bar, int lane) {
  __syncwarp();
  if (lane == 0) mbar_arrive(bar);
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}

template <int TY>
struct Stage3dSmem {
  static constexpr int NW = TY + 2;                 // warps: TY owners + H0 + H1
  static constexpr int NT = 32 * NW;
  static constexpr int PL = TY * RS;                // one ring plane of one variable
  static constexpr int NRING = 3 * PL;
  static constexpr int SB = 4 * RS;                 // one strip buffer of one variable (rows -2,-1,TY,TY+1)
  static constexpr int QS = NRING + 2 * SB;         // per-variable stride of W
  static constexpr int YQS = (TY + 2) * 32;         // YR: rows 0..TY-1 owners, rows TY, TY+1 = H1's two buffers
  static constexpr int FQS = TY * 32;               // YF: row j = flux through face j+1/2 (written by owner j)
  static constexpr int ZQ = TY * 32;                // z carries
  static constexpr int XQ = TY;                     // x hand-over: [buf][q][row]
  static constexpr int OFF_W = 0;
  static constexpr int OFF_YR = OFF_W + 8 * QS;
  static constexpr int OFF_YF = OFF_YR + 8 * YQS;
  static constexpr int OFF_WLZ = OFF_YF + 8 * FQS;
  static constexpr int OFF_FZP = OFF_WLZ + 8 * ZQ;
  static constexpr int OFF_XR = OFF_FZP + 8 * ZQ;   // [2][8][TY]
  static constexpr int OFF_XF = OFF_XR + 2 * 8 * XQ;
  static constexpr int OFF_XO = OFF_XF + 2 * 8 * XQ;   // [8][TY] lane 0's own x flux
  static constexpr int OFF_BAR = OFF_XO + 8 * XQ;      // mbarriers (8 bytes each)
  static constexpr int NBAR = 13 + 2 * TY;
  static constexpr size_t BYTES = sizeof(double) * (size_t)(OFF_BAR + NBAR);
};

