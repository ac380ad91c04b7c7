"""paper_2503_20899_b200 — B200-native AGATE finite-volume MHD step (arXiv 2503.20899, Sections 2.2 / 3.1).

Thin Python binding over the C-ABI library `libagate.so` (include/agate.h): argument marshalling only.  Every step
of the path (ghost fill, primitive recovery, PLM reconstruction, HLL/HLLD flux, flux difference, Runge-Kutta
combine, Courant reduction) runs in the hand-written sm_100a kernels of `csrc/`.  PyTorch supplies device memory
and the CUDA stream, nothing else.  There is no CPU fallback: without the built library or without a CUDA device
the binding raises.

    from paper_2503_20899_b200 import Agate
    sim = Agate(shape=(512, 512, 512), dx=(1/512,)*3, ndim=3, riemann=HLLD, beta=1.3)
    sim.set_state(U)            # numpy / torch, interior-only SoA [8, nz, ny, nx]
    t = sim.advance(20)
    U1 = sim.get_state()
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

IDEAL, HALL = 0, 1
CGL = 2              # CGL MHD: 9 variables per cell, U = (rho, m, E, B, A_log); see include/agate.h
IDEAL_GLM = 3        # 9 variables per cell (psi last); see include/agate.h
HALL_GLM = 4         # Hall MHD + GLM: 9 variables per cell
CGL_GLM = 5          # CGL MHD + GLM (eqs.19-23): 10 variables per cell, U = (rho, m, E, B, A, psi)
HLL, HLLD = 0, 1
OK, ERR_ARG, ERR_STATE, ERR_UNPHYSICAL, ERR_CUDA, ERR_NOMEM = range(6)

# every symbol include/agate.h declares (tests check that the library exports each of them)
SYMBOLS = ("agate_workspace_bytes", "agate_init", "agate_set_state", "agate_compute_dt", "agate_step",
           "agate_advance", "agate_get_state", "agate_poll", "agate_launch_info", "agate_set_timing",
           "agate_stage_time", "agate_set_tuning", "agate_set_slab", "agate_halo_bytes", "agate_get_vmax",
           "agate_set_vmax", "agate_vmax_device", "agate_step_begin", "agate_stage_pre", "agate_stage_post",
           "agate_destroy", "agate_strerror", "agate_test_face_flux",
           "agate_measure_fp64_peak", "agate_cfl_static", "agate_cfl_static_setup", "agate_cfl_static_max_segments")


class Grid(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double)]


class SolverCfg(C.Structure):
    _fields_ = [("riemann", C.c_int32), ("limiter", C.c_int32), ("beta", C.c_double),
                ("rk", C.c_int32), ("cfl", C.c_double), ("d_i", C.c_double), ("relax", C.c_double),
                ("bc", C.c_int32 * 3), ("cgl_form", C.c_int32)]


class Tuning(C.Structure):
    _fields_ = [("stage_grid", C.c_int32), ("no_graph", C.c_int32)]


class AgateError(RuntimeError):
    def __init__(self, code, where):
        msg = lib().agate_strerror(code).decode() if _lib is not None else "?"
        super().__init__(f"{where}: status {code} ({msg})")
        self.code = code


_lib = None
_vp, _dp = C.c_void_p, C.POINTER(C.c_double)


def lib():
    """Load (building if stale) libagate.so.  Raises if it cannot be built or loaded — never falls back."""
    global _lib
    if _lib is None:
        path = os.environ.get("AGATE_LIB")          # explicit override (kernel-variant experiments)
        if not path:
            path = _build.LIB
            if _build.is_stale():
                path = _build.build()
        L = C.CDLL(path)
        L.agate_workspace_bytes.argtypes = [C.POINTER(Grid), C.c_int, C.POINTER(SolverCfg)]
        L.agate_workspace_bytes.restype = C.c_size_t
        L.agate_init.argtypes = [C.POINTER(Grid), C.c_double, C.c_int, C.POINTER(SolverCfg), _vp, C.c_size_t, _vp,
                                 C.POINTER(_vp)]
        L.agate_set_state.argtypes = [_vp, _vp, C.c_int, C.c_double]
        L.agate_compute_dt.argtypes = [_vp, _dp]
        L.agate_step.argtypes = [_vp, C.c_double, _dp]
        L.agate_advance.argtypes = [_vp, C.c_int32, _dp]
        L.agate_get_state.argtypes = [_vp, _vp, C.c_int, _dp]
        L.agate_poll.argtypes = [_vp]
        L.agate_launch_info.argtypes = [_vp, C.POINTER(C.c_int64)]
        L.agate_set_timing.argtypes = [_vp, C.c_int]
        L.agate_stage_time.argtypes = [_vp, _dp, C.POINTER(C.c_int64), C.c_int]
        L.agate_set_tuning.argtypes = [_vp, C.POINTER(Tuning)]
        L.agate_set_slab.argtypes = [_vp, C.c_int, C.c_int]
        L.agate_halo_bytes.argtypes = [_vp]
        L.agate_halo_bytes.restype = C.c_size_t
        L.agate_get_vmax.argtypes = [_vp, _dp]
        L.agate_set_vmax.argtypes = [_vp, C.c_double]
        L.agate_vmax_device.argtypes = [_vp, C.POINTER(_vp)]
        L.agate_step_begin.argtypes = [_vp, C.c_double]
        L.agate_stage_pre.argtypes = [_vp, C.c_int, _vp, _vp]
        L.agate_stage_post.argtypes = [_vp, C.c_int, _vp, _vp]
        L.agate_destroy.argtypes = [_vp]
        L.agate_strerror.argtypes = [C.c_int]
        L.agate_strerror.restype = C.c_char_p
        L.agate_test_face_flux.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                           _vp, _vp, _vp, _vp, C.c_int64, _vp]
        L.agate_measure_fp64_peak.argtypes = [C.c_int, _dp, _vp, _vp]
        L.agate_cfl_static.argtypes = [C.POINTER(Grid), C.c_double, C.c_int, C.POINTER(SolverCfg), _vp, _vp, _vp]
        L.agate_cfl_static_setup.argtypes = []
        L.agate_cfl_static_max_segments.argtypes = []
        L.agate_cfl_static_max_segments.restype = C.c_int64
        _lib = L
    return _lib


def _torch_cuda():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2503_20899_b200 needs a CUDA device (no CPU fallback)")
    return torch


class Agate:
    """One simulation context (agate_ctx) on a dedicated CUDA stream.  Names follow include/agate.h."""

    def __init__(self, shape, dx, ndim, gamma=5.0 / 3.0, eqset=IDEAL, riemann=HLL, limiter=2, beta=1.3, rk=2,
                 cfl=0.0, d_i=0.0, relax=0.0, bc=(0, 0, 0), device="cuda:0", stream=None, stage_grid=0, no_graph=False,
                 cgl_form=0):
        torch = _torch_cuda()
        nx, ny, nz = (int(s) for s in shape)
        self.shape = (nx, ny, nz)
        self.zones = nx * ny * nz
        self.nvar = {IDEAL_GLM: 9, CGL: 9, HALL_GLM: 9, CGL_GLM: 10}.get(int(eqset), 8)
        self.grid = Grid(ndim, nx, ny, nz, dx[0], dx[1], dx[2])
        self.cfg = SolverCfg(riemann, limiter, beta, rk, cfl, d_i, relax, (C.c_int32 * 3)(*[int(b) for b in bc]),
                             int(cgl_form))
        self.device = torch.device(device)
        L = lib()
        nbytes = L.agate_workspace_bytes(C.byref(self.grid), eqset, C.byref(self.cfg))
        if nbytes == 0:
            raise AgateError(ERR_ARG, "agate_workspace_bytes")
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            # torch's allocator returns >= 512-byte aligned blocks
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._h = _vp()
            rc = L.agate_init(C.byref(self.grid), float(gamma), int(eqset), C.byref(self.cfg),
                              _vp(self.workspace.data_ptr()), nbytes, _vp(self.stream.cuda_stream), C.byref(self._h))
        if rc:
            raise AgateError(rc, "agate_init")
        if stage_grid or no_graph:
            tun = Tuning(int(stage_grid), 1 if no_graph else 0)
            self._chk(L.agate_set_tuning(self._h, C.byref(tun)), "agate_set_tuning")

    @classmethod
    def from_workload(cls, wl, **over):
        kw = dict(shape=wl.shape, dx=wl.dx, ndim=wl.ndim, gamma=wl.gamma, eqset=wl.eqset, riemann=wl.riemann,
                  limiter=wl.limiter, beta=wl.beta, rk=wl.rk, cfl=wl.cfl, d_i=wl.d_i,
                  relax=getattr(wl, "relax", 0.0))
        set_state = over.pop("set_state", True)
        kw.update(over)
        s = cls(**kw)
        if set_state:
            s.set_state(wl.U)
        return s

    def _chk(self, rc, where):
        if rc:
            raise AgateError(rc, where)

    # -- state in / out ------------------------------------------------------------------------------------
    def set_state(self, U, t0=0.0):
        """U: numpy array / CPU torch tensor (host path) or CUDA torch tensor (device path), [8,nz,ny,nx] f64."""
        torch = _torch_cuda()
        n = self.nvar * self.zones
        if isinstance(U, torch.Tensor):
            assert U.dtype == torch.float64 and U.numel() == n and U.is_contiguous()
            self._keep = U
            ptr, on_dev = U.data_ptr(), U.is_cuda
        else:
            U = np.ascontiguousarray(U, dtype=np.float64)
            assert U.size == n
            self._keep = U
            ptr, on_dev = U.ctypes.data, False
        with torch.cuda.device(self.device):
            if on_dev:      # the copy runs on the context's stream: order it after whatever produced U (include/agate.h)
                self.stream.wait_stream(torch.cuda.current_stream())
            self._chk(lib().agate_set_state(self._h, _vp(ptr), int(on_dev), float(t0)), "agate_set_state")

    def get_state(self, out=None):
        """Returns (or fills `out`: numpy, CPU or CUDA torch tensor) the interior-only SoA state [8,nz,ny,nx]."""
        torch = _torch_cuda()
        nx, ny, nz = self.shape
        if out is None:
            out = np.empty((self.nvar, nz, ny, nx))
        t = C.c_double()
        if isinstance(out, torch.Tensor):
            assert out.dtype == torch.float64 and out.numel() == self.nvar * self.zones and out.is_contiguous()
            ptr, on_dev = out.data_ptr(), out.is_cuda
        else:
            assert out.dtype == np.float64 and out.size == self.nvar * self.zones and out.flags.c_contiguous
            ptr, on_dev = out.ctypes.data, False
        with torch.cuda.device(self.device):
            self._chk(lib().agate_get_state(self._h, _vp(ptr), int(on_dev), C.byref(t)), "agate_get_state")
            if on_dev:      # later work on torch's current stream sees the copied state
                torch.cuda.current_stream().wait_stream(self.stream)
        self.t = t.value
        return out

    # -- stepping ------------------------------------------------------------------------------------------
    def compute_dt(self):
        dt = C.c_double()
        self._chk(lib().agate_compute_dt(self._h, C.byref(dt)), "agate_compute_dt")
        return dt.value

    def step(self, dt=0.0, sync=True):
        used = C.c_double()
        self._chk(lib().agate_step(self._h, float(dt), C.byref(used) if sync else None), "agate_step")
        return used.value if sync else None

    def advance(self, n, sync=True):
        t = C.c_double()
        self._chk(lib().agate_advance(self._h, int(n), C.byref(t) if sync else None), "agate_advance")
        return t.value if sync else None

    def poll(self):
        self._chk(lib().agate_poll(self._h), "agate_poll")

    # -- NEXT-4: slab decomposition (include/agate.h) ---------------------------------------------------------
    def set_slab(self, cut_lo, cut_hi):
        self._chk(lib().agate_set_slab(self._h, int(bool(cut_lo)), int(bool(cut_hi))), "agate_set_slab")
        self.rk = int(self.cfg.rk)

    def halo_bytes(self):
        return int(lib().agate_halo_bytes(self._h))

    def halo_buffers(self):
        """Four device buffers (send_lo, send_hi, recv_lo, recv_hi) of halo_bytes() each, as float64 tensors."""
        torch = _torch_cuda()
        n = self.halo_bytes() // 8
        return tuple(torch.zeros(n, dtype=torch.float64, device=self.device) for _ in range(4))

    def get_vmax(self):
        v = C.c_double()
        self._chk(lib().agate_get_vmax(self._h, C.byref(v)), "agate_get_vmax")
        return v.value

    def set_vmax(self, v):
        self._chk(lib().agate_set_vmax(self._h, float(v)), "agate_set_vmax")

    def vmax_tensor(self):
        """The device-resident v_max as a one-element float64 view of the workspace (for an in-place all-reduce)."""
        torch = _torch_cuda()
        p = _vp()
        self._chk(lib().agate_vmax_device(self._h, C.byref(p)), "agate_vmax_device")
        off = p.value - self.workspace.data_ptr()
        return self.workspace[off:off + 8].view(torch.float64)

    def step_begin(self, dt=0.0):
        self._chk(lib().agate_step_begin(self._h, float(dt)), "agate_step_begin")

    def stage_pre(self, stage, send_lo=None, send_hi=None):
        p = lambda t: _vp(t.data_ptr()) if t is not None else None
        self._chk(lib().agate_stage_pre(self._h, int(stage), p(send_lo), p(send_hi)), "agate_stage_pre")

    def stage_post(self, stage, recv_lo=None, recv_hi=None):
        p = lambda t: _vp(t.data_ptr()) if t is not None else None
        self._chk(lib().agate_stage_post(self._h, int(stage), p(recv_lo), p(recv_hi)), "agate_stage_post")

    # -- bookkeeping ---------------------------------------------------------------------------------------
    def launch_info(self):
        out = (C.c_int64 * 8)()
        self._chk(lib().agate_launch_info(self._h, out), "agate_launch_info")
        return dict(grid=(out[0], out[1], out[2]), threads=out[3], smem=out[4], regs=out[5], blocks_per_sm=out[6],
                    launches_per_step=out[7])

    def set_timing(self, on):
        self._chk(lib().agate_set_timing(self._h, int(bool(on))), "agate_set_timing")

    def stage_time(self, reset=True):
        ms, n = C.c_double(), C.c_int64()
        self._chk(lib().agate_stage_time(self._h, C.byref(ms), C.byref(n), int(reset)), "agate_stage_time")
        return ms.value, n.value

    def close(self):
        if getattr(self, "_h", None):
            lib().agate_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def test_face_flux(eqset, riemann, d, gamma, WL, WR, J=None, d_i=0.0, dxmin=1.0):
    """Device Riemann flux on n face pairs (diagnostic entry agate_test_face_flux).  WL, WR: [8,n]; J: [3,n]."""
    torch = _torch_cuda()
    WLd = torch.as_tensor(np.ascontiguousarray(WL), dtype=torch.float64, device="cuda")
    WRd = torch.as_tensor(np.ascontiguousarray(WR), dtype=torch.float64, device="cuda")
    n = WLd.shape[1]
    Jd = None if J is None else torch.as_tensor(np.ascontiguousarray(J), dtype=torch.float64, device="cuda")
    F = torch.empty((8, n), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    rc = lib().agate_test_face_flux(int(eqset), int(riemann), int(d), float(gamma), float(d_i), float(dxmin),
                                    _vp(WLd.data_ptr()), _vp(WRd.data_ptr()),
                                    _vp(Jd.data_ptr()) if Jd is not None else None, _vp(F.data_ptr()), n, None)
    if rc:
        raise AgateError(rc, "agate_test_face_flux")
    return F.cpu().numpy()


def measure_fp64_peak(iters=20):
    torch = _torch_cuda()
    v = C.c_double()
    scratch = torch.zeros(8, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    rc = lib().agate_measure_fp64_peak(int(iters), C.byref(v), _vp(scratch.data_ptr()), None)
    if rc:
        raise AgateError(rc, "agate_measure_fp64_peak")
    return v.value


def cfl_static(U, out, shape, dx, ndim, gamma=5.0 / 3.0, eqset=IDEAL, cfl=0.0, d_i=0.0, cgl_form=0, stream=None):
    """Allocation-free Courant reduction (agate_cfl_static; see include/agate.h): v_max, dt and the unphysical flag of
    the interior-only device state `U` ([nv,nz,ny,nx] f64 CUDA tensor) into the caller's `out` (3 f64 on the same
    device).  Argument marshalling only: no tensor is created here and nothing synchronises; the work is enqueued on
    `stream` (default: torch's current stream).  Raises AgateError (status 6) beyond the static scratch's limit."""
    torch = _torch_cuda()
    nx, ny, nz = (int(v) for v in shape)
    if not (U.is_cuda and out.is_cuda and U.dtype == torch.float64 and out.dtype == torch.float64):
        raise TypeError("cfl_static: U and out must be float64 CUDA tensors")
    if not (U.is_contiguous() and out.is_contiguous()) or out.numel() < 3 or U.device != out.device:
        raise ValueError("cfl_static: contiguous tensors on one device, out with >= 3 elements")
    nvar = {IDEAL_GLM: 9, CGL: 9, HALL_GLM: 9, CGL_GLM: 10}.get(int(eqset), 8)
    if U.numel() != nvar * nx * ny * nz:
        raise ValueError(f"cfl_static: U has {U.numel()} elements, the grid needs {nvar * nx * ny * nz}")
    grid = Grid(int(ndim), nx, ny, nz, float(dx[0]), float(dx[1]), float(dx[2]))
    cfg = SolverCfg(HLL, 2, 1.3, 2, float(cfl), float(d_i), 0.0, (C.c_int32 * 3)(0, 0, 0), int(cgl_form))
    with torch.cuda.device(U.device):
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = lib().agate_cfl_static(C.byref(grid), float(gamma), int(eqset), C.byref(cfg), _vp(U.data_ptr()),
                                    _vp(out.data_ptr()), _vp(st.cuda_stream))
    if rc:
        raise AgateError(rc, "agate_cfl_static")
    return out


def cfl_static_setup(device=None):
    """Resolve the static scratch's device address on `device` (default: the current one); once per device, before
    capturing a graph that contains cfl_static."""
    torch = _torch_cuda()
    with torch.cuda.device(device if device is not None else torch.cuda.current_device()):
        rc = lib().agate_cfl_static_setup()
    if rc:
        raise AgateError(rc, "agate_cfl_static_setup")
