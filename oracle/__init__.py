"""CPU ORACLE of the AGATE finite-volume MHD step — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes loader around `oracle/agate_ref.cpp` (plain single-threaded C++, written from PAPER.md
§2.2 / §3.1 and the readings in DESIGN.md).  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import this package.  It shares no code with, and never
imports, `paper_2503_20899_b200` (the CUDA path); the CUDA path never imports this.

Pins: tests/test_oracle_pins.py (closed forms, invariants, the paper's printed values).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "agate_ref.cpp")
_HDR = os.path.join(_HERE, "agate_ref.h")
_LIB = os.path.join(_HERE, "libagate_ref.so")

IDEAL, HALL = 0, 1
CGL = 2              # CGL MHD: 9 variables per cell, U = (rho, m, E, B, A_log), W = (rho, v, p_par, B, p_perp) (R24)
IDEAL_GLM = 3        # ideal MHD + GLM divergence cleaning: 9 variables per cell, psi last (eqs.10-11; R22)
HALL_GLM = 4         # Hall MHD + GLM (R29): 9 variables per cell
CGL_GLM = 5          # CGL MHD + GLM (eqs.19-23; R30): 10 variables per cell, U = (rho, m, E, B, A, psi)
HLL, HLLD = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (IEEE fp64, no contraction, no fast-math).  Returns the .so path."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(p) > os.path.getmtime(_LIB) for p in (_SRC, _HDR))
    if force or stale:
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
               "-shared", "-Wall", "-o", tmp, _SRC]
        subprocess.run(cmd, check=True, cwd=_HERE)
        os.replace(tmp, _LIB)
    return _LIB


class Grid(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double)]


class SolverCfg(C.Structure):
    _fields_ = [("riemann", C.c_int32), ("limiter", C.c_int32), ("beta", C.c_double),
                ("rk", C.c_int32), ("cfl", C.c_double), ("d_i", C.c_double), ("relax", C.c_double),
                ("bc", C.c_int32 * 3), ("cgl_form", C.c_int32)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp = C.c_void_p
        L.agate_ref_create.argtypes = [C.POINTER(Grid), C.c_double, C.c_int, C.POINTER(SolverCfg), C.POINTER(vp)]
        L.agate_ref_set_state.argtypes = [vp, _dp, C.c_double]
        L.agate_ref_compute_dt.argtypes = [vp, _dp]
        L.agate_ref_vmax.argtypes = [vp, _dp]
        L.agate_ref_step.argtypes = [vp, C.c_double, _dp]
        L.agate_ref_advance.argtypes = [vp, C.c_int32, _dp]
        L.agate_ref_get_state.argtypes = [vp, _dp, _dp]
        L.agate_ref_rhs.argtypes = [vp, _dp]
        L.agate_ref_destroy.argtypes = [vp]
        L.agate_ref_cgl_cons_to_prim.argtypes = [_dp, _dp]
        L.agate_ref_cgl_cons_to_prim.restype = None
        L.agate_ref_cgl_prim_to_cons.argtypes = [_dp, _dp]
        L.agate_ref_cgl_prim_to_cons.restype = None
        L.agate_ref_cgl_cfast.argtypes = [C.c_int, _dp]
        L.agate_ref_cgl_cfast.restype = C.c_double
        L.agate_ref_cgl_face_flux.argtypes = [C.c_int, _dp, _dp, _dp]
        L.agate_ref_cgl_face_flux.restype = None
        L.agate_ref_cgl_cons_to_prim_form.argtypes = [C.c_int, _dp, _dp]
        L.agate_ref_cgl_cons_to_prim_form.restype = None
        L.agate_ref_cgl_prim_to_cons_form.argtypes = [C.c_int, _dp, _dp]
        L.agate_ref_cgl_prim_to_cons_form.restype = None
        L.agate_ref_cgl_face_flux_form.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp]
        L.agate_ref_cgl_face_flux_form.restype = None
        L.agate_ref_cgl_relax.argtypes = [C.c_double, C.c_double, _dp, _dp]
        L.agate_ref_cgl_relax.restype = None
        L.agate_ref_nvar.argtypes = [vp]
        L.agate_ref_nvar.restype = C.c_int
        L.agate_ref_glm_ch.argtypes = [vp, _dp]
        L.agate_ref_glm_face.argtypes = [C.c_double] * 5 + [_dp, _dp]
        L.agate_ref_glm_face.restype = None
        L.agate_ref_set_threads.argtypes = [C.c_int]
        L.agate_ref_get_threads.restype = C.c_int
        L.agate_ref_cons_to_prim.argtypes = [C.c_double, _dp, _dp]
        L.agate_ref_cons_to_prim.restype = None
        L.agate_ref_prim_to_cons.argtypes = [C.c_double, _dp, _dp]
        L.agate_ref_prim_to_cons.restype = None
        L.agate_ref_slope.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
        L.agate_ref_slope.restype = C.c_double
        L.agate_ref_cfast.argtypes = [C.c_int, C.c_double, _dp]
        L.agate_ref_cfast.restype = C.c_double
        L.agate_ref_cwhistler.argtypes = [C.c_double, C.c_double, _dp]
        L.agate_ref_cwhistler.restype = C.c_double
        L.agate_ref_phys_flux.argtypes = [C.c_int, C.c_double, _dp, _dp, _dp]
        L.agate_ref_phys_flux.restype = None
        L.agate_ref_face_flux.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                          _dp, _dp, _dp, _dp]
        L.agate_ref_face_flux.restype = None
        L.agate_ref_hlld_branch.argtypes = [C.c_int, C.c_double, _dp, _dp]
        L.agate_ref_hlld_branch.restype = C.c_int
        L.agate_ref_count_ops.argtypes = [C.POINTER(Grid), C.c_double, C.c_int, C.POINTER(SolverCfg), _dp, _dp]
        _lib = L
    return _lib


def _vec(a, n=8):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(n))
    return a, a.ctypes.data_as(_dp)


def set_threads(n: int) -> None:
    """OpenMP threads for the grid loops (bitwise identical results); 1 = the single-threaded oracle."""
    lib().agate_ref_set_threads(int(n))


def get_threads() -> int:
    return int(lib().agate_ref_get_threads())


# ---- point functions -------------------------------------------------------------------------
def cons_to_prim(U, gamma):
    u, pu = _vec(U); w = np.empty(8); lib().agate_ref_cons_to_prim(gamma, pu, w.ctypes.data_as(_dp)); return w


def prim_to_cons(W, gamma):
    w, pw = _vec(W); u = np.empty(8); lib().agate_ref_prim_to_cons(gamma, pw, u.ctypes.data_as(_dp)); return u


def slope(limiter, beta, dp, dm):
    return float(lib().agate_ref_slope(int(limiter), float(beta), float(dp), float(dm)))


def cfast(d, gamma, W):
    w, pw = _vec(W); return float(lib().agate_ref_cfast(int(d), float(gamma), pw))


def cwhistler(d_i, dxmin, W):
    w, pw = _vec(W); return float(lib().agate_ref_cwhistler(float(d_i), float(dxmin), pw))


def phys_flux(d, gamma, W, vH=None):
    w, pw = _vec(W); F = np.empty(8)
    if vH is None:
        lib().agate_ref_phys_flux(int(d), float(gamma), pw, None, F.ctypes.data_as(_dp))
    else:
        h, ph = _vec(vH, 3)
        lib().agate_ref_phys_flux(int(d), float(gamma), pw, ph, F.ctypes.data_as(_dp))
    return F


def face_flux(riemann, d, gamma, WL, WR, eqset=IDEAL, d_i=0.0, dxmin=1.0, J=None):
    wl, pl = _vec(WL); wr, pr = _vec(WR); F = np.empty(8)
    if J is None:
        pj = None
    else:
        jj, pj = _vec(J, 3)
    lib().agate_ref_face_flux(int(eqset), int(riemann), int(d), float(gamma), float(d_i), float(dxmin),
                              pl, pr, pj, F.ctypes.data_as(_dp))
    return F


def cgl_cons_to_prim(U, form=0):
    u, pu = _vec(U, 9); W = np.empty(9)
    lib().agate_ref_cgl_cons_to_prim_form(int(form), pu, W.ctypes.data_as(_dp)); return W


def cgl_prim_to_cons(W, form=0):
    w, pw = _vec(W, 9); U = np.empty(9)
    lib().agate_ref_cgl_prim_to_cons_form(int(form), pw, U.ctypes.data_as(_dp)); return U


def cgl_cfast(d, W):
    w, pw = _vec(W, 9); return float(lib().agate_ref_cgl_cfast(int(d), pw))


def cgl_face_flux(d, WL, WR, form=0):
    wl, pl = _vec(WL, 9); wr, pr = _vec(WR, 9); F = np.empty(9)
    lib().agate_ref_cgl_face_flux_form(int(form), int(d), pl, pr, F.ctypes.data_as(_dp)); return F


def cgl_relax(f, B2, ppar, pperp):
    a, b = C.c_double(ppar), C.c_double(pperp)
    lib().agate_ref_cgl_relax(float(f), float(B2), C.byref(a), C.byref(b))
    return a.value, b.value


def glm_face(ch, bnL, bnR, psL, psR):
    """(B_n*, psi*) of the 2x2 linear GLM Riemann problem at one face."""
    a, b = C.c_double(), C.c_double()
    lib().agate_ref_glm_face(float(ch), float(bnL), float(bnR), float(psL), float(psR), C.byref(a), C.byref(b))
    return a.value, b.value


def hlld_branch(d, gamma, WL, WR):
    wl, pl = _vec(WL); wr, pr = _vec(WR)
    return int(lib().agate_ref_hlld_branch(int(d), float(gamma), pl, pr))


# ---- the stepping interface ------------------------------------------------------------------
class RefError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"oracle {where} failed with status {code}")
        self.code = code


class RefSolver:
    """Host-memory solver with the same call shape as the product's C-ABI (agate_ref_* functions)."""

    def __init__(self, shape, dx, ndim, gamma=5.0 / 3.0, eqset=IDEAL, riemann=HLL, limiter=2, beta=1.3,
                 rk=2, cfl=0.0, d_i=0.0, relax=0.0, bc=(0, 0, 0), cgl_form=0):
        nx, ny, nz = (int(s) for s in shape)
        self.shape = (nx, ny, nz)
        self.grid = Grid(ndim, nx, ny, nz, dx[0], dx[1], dx[2])
        self.cfg = SolverCfg(riemann, limiter, beta, rk, cfl, d_i, relax, (C.c_int32 * 3)(*[int(b) for b in bc]),
                             int(cgl_form))
        self.gamma, self.eqset = float(gamma), int(eqset)
        self._h = C.c_void_p()
        rc = lib().agate_ref_create(C.byref(self.grid), self.gamma, self.eqset, C.byref(self.cfg), C.byref(self._h))
        if rc:
            raise RefError(rc, "create")
        self.nvar = int(lib().agate_ref_nvar(self._h))

    @classmethod
    def from_workload(cls, wl, **over):
        kw = dict(shape=wl.shape, dx=wl.dx, ndim=wl.ndim, gamma=wl.gamma, eqset=wl.eqset, riemann=wl.riemann,
                  limiter=wl.limiter, beta=wl.beta, rk=wl.rk, cfl=wl.cfl, d_i=wl.d_i,
                  relax=getattr(wl, "relax", 0.0))
        kw.update(over)
        s = cls(**kw)
        s.set_state(wl.U)
        return s

    def _chk(self, rc, where):
        if rc:
            raise RefError(rc, where)

    def set_state(self, U, t0=0.0):
        nx, ny, nz = self.shape
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.size == self.nvar * nx * ny * nz
        self._chk(lib().agate_ref_set_state(self._h, U.ctypes.data_as(_dp), float(t0)), "set_state")

    def compute_dt(self):
        dt = C.c_double()
        self._chk(lib().agate_ref_compute_dt(self._h, C.byref(dt)), "compute_dt")
        return dt.value

    def glm_ch(self):
        v = C.c_double()
        self._chk(lib().agate_ref_glm_ch(self._h, C.byref(v)), "glm_ch")
        return v.value

    def vmax(self):
        v = C.c_double()
        self._chk(lib().agate_ref_vmax(self._h, C.byref(v)), "vmax")
        return v.value

    def step(self, dt=0.0):
        used = C.c_double()
        self._chk(lib().agate_ref_step(self._h, float(dt), C.byref(used)), "step")
        return used.value

    def advance(self, n):
        t = C.c_double()
        self._chk(lib().agate_ref_advance(self._h, int(n), C.byref(t)), "advance")
        return t.value

    def get_state(self):
        nx, ny, nz = self.shape
        U = np.empty((self.nvar, nz, ny, nx))
        t = C.c_double()
        self._chk(lib().agate_ref_get_state(self._h, U.ctypes.data_as(_dp), C.byref(t)), "get_state")
        self.t = t.value
        return U

    def rhs(self):
        nx, ny, nz = self.shape
        Lo = np.empty((self.nvar, nz, ny, nx))
        self._chk(lib().agate_ref_rhs(self._h, Lo.ctypes.data_as(_dp)), "rhs")
        return Lo

    def close(self):
        if self._h:
            lib().agate_ref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def count_ops(wl):
    """Algorithmic operation counts of ONE full step on workload `wl` (Counted<double> instantiation).
    Returns dict(add, mul, div, sqrt, cmp, flops) per zone-update."""
    nx, ny, nz = wl.shape
    grid = Grid(wl.ndim, nx, ny, nz, wl.dx[0], wl.dx[1], wl.dx[2])
    cfg = SolverCfg(wl.riemann, wl.limiter, wl.beta, wl.rk, wl.cfl, wl.d_i, getattr(wl, "relax", 0.0))
    U = np.ascontiguousarray(wl.U, dtype=np.float64)
    out = np.zeros(5)
    rc = lib().agate_ref_count_ops(C.byref(grid), wl.gamma, wl.eqset, C.byref(cfg), U.ctypes.data_as(_dp),
                                   out.ctypes.data_as(_dp))
    if rc:
        raise RefError(rc, "count_ops")
    per = out / (nx * ny * nz)
    return dict(add=per[0], mul=per[1], div=per[2], sqrt=per[3], cmp=per[4], flops=float(per.sum()))
