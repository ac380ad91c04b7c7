// agate_noalloc.cu — the allocation-free entry point of the library (include/agate.h "allocation-free Courant reduction").
//
// agate_cfl_static is the Courant reduction A7 (R3-R5, R14: v_max = max over zones of |v| + c, dt = C dx_min /
// v_max) on a caller-owned interior-only device state, for callers that cannot hand the library a workspace or call
// cudaMalloc themselves (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).  It is a
// variant of dt_kernel (agate_kernels.cuh): the same point functions give the speed of a zone, so both paths return the
// same bits; what differs is where the reduction's scratch lives -- the per-block partial maxima, the ticket counter and
// the unphysical-state flag sit in ONE file-scope __device__ array of fixed size instead of the context's workspace.
//
// Consequences of that array, all stated in the header too:
//   * every GPU that loads libagate.so holds kScratchBytes (about 0.5 MiB) of device memory until the process exits;
//   * a grid that needs more partial slots than the array has is rejected with AGATE_ERR_LIMIT, nothing is launched;
//   * every call on a device shares the array and finds the last call's contents in it: the header is cleared on the
//     stream before each launch, the partial slots are all written before they are read;
//   * two calls that overlap on one GPU (different streams, no ordering between them) race on it.
// In host code the array's name is a host-side stand-in, not a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, once per device with that device current (scratch_address below).
#include "agate.h"

#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "agate_physics.cuh"

namespace {

using namespace agate;

constexpr int kSegZones = 1024;                                  // zones of one row that one block reduces
constexpr int kThreads = 256;
constexpr int kMaxSegments = AGATE_STATIC_MAX_SEGMENTS;          // partial slots in the static array
constexpr size_t kHeaderBytes = 256;                             // [0] ticket (u32), [64] flag (i32)
constexpr size_t kScratchBytes = kHeaderBytes + sizeof(double) * (size_t)kMaxSegments;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_cfl_scratch[kScratchBytes];

struct CflStaticParams {
  const double* U;       // interior-only SoA [nv][nz][ny][nx]
  long long sq;          // zones per variable
  int nx, segs_per_row;
  long long nseg;
  double cfl_dx;         // C * dx_min
  Phys ph;
  int hall, cgl;
  unsigned char* scratch;
  double* out;           // [0] v_max, [1] dt, [2] 1.0 if an unphysical zone was seen, else 0.0
};

__device__ __forceinline__ double warp_max_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// One block per segment (<= 1024 consecutive zones of one grid row); the last block to take a ticket reduces the
// partial maxima.  max is exact under any association, so the result does not depend on the block order.
__global__ void __launch_bounds__(kThreads) cfl_static_kernel(const __grid_constant__ CflStaticParams P) {
  __shared__ double wmax[kThreads / 32];
  __shared__ int wbad[kThreads / 32];
  __shared__ bool last;
  unsigned int* const ticket = reinterpret_cast<unsigned int*>(P.scratch);
  int* const flag = reinterpret_cast<int*>(P.scratch + 64);
  double* const partial = reinterpret_cast<double*>(P.scratch + kHeaderBytes);
  const long long seg = blockIdx.x;
  const long long row = seg / P.segs_per_row;
  const int i0 = (int)(seg - row * P.segs_per_row) * kSegZones;
  const int i1 = min(P.nx, i0 + kSegZones);
  const double* base = P.U + row * P.nx;
  double vm = 0.0;
  int bad = 0;
  for (int i = i0 + threadIdx.x; i < i1; i += kThreads) {
    double u[9];
#pragma unroll
    for (int q = 0; q < 8; ++q) u[q] = __ldg(base + q * P.sq + i);
    u[8] = P.cgl ? __ldg(base + 8 * P.sq + i) : 0.0;
    const double sp = P.cgl ? cell_speed_cgl(u, P.ph.cgl_form)
                            : (P.hall ? cell_speed_inline<true>(P.ph, u) : cell_speed_inline<false>(P.ph, u));
    if (sp < 0.0) bad = 1; else vm = fmax(vm, sp);
  }
  vm = warp_max_d(vm);
  bad = __any_sync(0xffffffffu, bad);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) { wmax[wid] = vm; wbad[wid] = bad; }
  __syncthreads();
  if (wid == 0) {
    vm = (lane < kThreads / 32) ? wmax[lane] : 0.0;
    bad = (lane < kThreads / 32) ? wbad[lane] : 0;
    vm = warp_max_d(vm);
    bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
      partial[seg] = vm;
      if (bad) atomicOr(flag, 1);
      __threadfence();
      last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double v = 0.0;
  for (long long b = threadIdx.x; b < P.nseg; b += kThreads) v = fmax(v, __ldcg(partial + b));
  v = warp_max_d(v);
  if (lane == 0) wmax[wid] = v;
  __syncthreads();
  if (wid == 0) {
    v = (lane < kThreads / 32) ? wmax[lane] : 0.0;
    v = warp_max_d(v);
    if (lane == 0) {
      P.out[0] = v;
      P.out[1] = P.cfl_dx / v;
      P.out[2] = (__ldcg(flag) & 1) ? 1.0 : 0.0;
      *ticket = 0u;                        // the next call clears the header anyway; leave it clean
    }
  }
}

// Device address of the static array on the CURRENT device, resolved once per device.
std::mutex g_mu;
void* g_ptr[kMaxDevices] = {};

int scratch_address(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return AGATE_ERR_CUDA;
  if (dev < 0 || dev >= kMaxDevices) return AGATE_ERR_ARG;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_cfl_scratch) != cudaSuccess || !p) return AGATE_ERR_CUDA;
    g_ptr[dev] = p;
  }
  *out = static_cast<unsigned char*>(g_ptr[dev]);
  return AGATE_OK;
}

}  // namespace

extern "C" {

int64_t agate_cfl_static_max_segments(void) { return kMaxSegments; }

int agate_cfl_static_setup(void) {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return AGATE_ERR_CUDA;   // no CPU fallback
  unsigned char* p = nullptr;
  return scratch_address(&p);
}

int agate_cfl_static(const agate_grid* g, double gamma, int eqset, const agate_solver* s, const double* U_dev,
                     double* out_dev, void* stream) {
  if (!g || !s || !U_dev || !out_dev) return AGATE_ERR_ARG;
  if (g->ndim < 1 || g->ndim > 3 || g->nx < 1 || g->ny < 1 || g->nz < 1) return AGATE_ERR_ARG;
  if ((g->ndim < 3 && g->nz != 1) || (g->ndim < 2 && g->ny != 1)) return AGATE_ERR_ARG;
  if (!(g->dx > 0.0) || (g->ndim >= 2 && !(g->dy > 0.0)) || (g->ndim >= 3 && !(g->dz > 0.0))) return AGATE_ERR_ARG;
  if (!(gamma > 1.0) || eqset < AGATE_IDEAL || eqset > AGATE_CGL_GLM) return AGATE_ERR_ARG;
  const bool hall = (eqset == AGATE_HALL || eqset == AGATE_HALL_GLM);
  const bool cgl = (eqset == AGATE_CGL || eqset == AGATE_CGL_GLM);
  if (hall && !(s->d_i >= 0.0)) return AGATE_ERR_ARG;
  if (s->cgl_form < 0 || s->cgl_form > 1) return AGATE_ERR_ARG;
  // the limit of the static array: one partial slot per segment of <= 1024 zones of a row
  const long long segs_per_row = (g->nx + kSegZones - 1) / kSegZones;
  const long long nseg = segs_per_row * (long long)g->ny * (long long)g->nz;
  if (nseg > kMaxSegments) return AGATE_ERR_LIMIT;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return AGATE_ERR_CUDA;   // no CPU fallback
  unsigned char* scratch = nullptr;
  int rc = scratch_address(&scratch);
  if (rc) return rc;

  CflStaticParams p;
  p.U = U_dev;
  p.sq = (long long)g->nx * g->ny * g->nz;
  p.nx = g->nx;
  p.segs_per_row = (int)segs_per_row;
  p.nseg = nseg;
  double dxmin = g->dx;                                            // R5: min over ACTIVE dimensions
  if (g->ndim >= 2) dxmin = fmin(dxmin, g->dy);
  if (g->ndim >= 3) dxmin = fmin(dxmin, g->dz);
  double cfl = s->cfl;
  if (!(cfl > 0.0)) cfl = (g->ndim == 1) ? 0.8 : (g->ndim == 2 ? 0.45 : 0.325);
  p.cfl_dx = cfl * dxmin;
  p.ph = make_phys(gamma, hall ? s->d_i : 0.0, dxmin);
  p.ph.cgl_form = cgl ? s->cgl_form : 0;
  p.hall = hall ? 1 : 0;
  p.cgl = cgl ? 1 : 0;
  p.scratch = scratch;
  p.out = out_dev;
  cudaStream_t st = (cudaStream_t)stream;
  // the array keeps the last call's contents: ticket and flag must start at zero (an earlier launch that failed half
  // way would otherwise leave them set); the partial slots 0 .. nseg-1 are all written before the last block reads them
  if (cudaMemsetAsync(scratch, 0, kHeaderBytes, st) != cudaSuccess) return AGATE_ERR_CUDA;
  cfl_static_kernel<<<(unsigned)nseg, kThreads, 0, st>>>(p);
  if (cudaGetLastError() != cudaSuccess) return AGATE_ERR_CUDA;
  return AGATE_OK;
}

}  // extern "C"
