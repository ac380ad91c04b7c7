"""Host-side check of the CUDA path's point functions (agate_physics.cuh) against the oracle — no GPU needed.

The header is __host__ __device__; tests/host_shim/physics_shim.cpp compiles it with g++ and this file compares
each function with the oracle's (oracle/agate_ref.cpp) on random and degenerate inputs.  The two sides share no
code: the CUDA path restructures HLLD (mirrored fan, shared reciprocals), so agreement to a few ulp on every
branch is a real test of that restructuring before any GPU time is spent.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

import oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SHIM_SRC = os.path.join(ROOT, "tests", "host_shim", "physics_shim.cpp")
CSRC = os.path.join(ROOT, "paper_2503_20899_b200", "csrc")
SHIM_LIB = os.path.join(ROOT, "tests", "host_shim", "libphysics_shim.so")
_dp = C.POINTER(C.c_double)
G = 5.0 / 3.0


@pytest.fixture(scope="module")
def shim():
    deps = [SHIM_SRC, os.path.join(CSRC, "agate_physics.cuh")]
    if not os.path.exists(SHIM_LIB) or any(os.path.getmtime(p) > os.path.getmtime(SHIM_LIB) for p in deps):
        tmp = SHIM_LIB + f".tmp{os.getpid()}"
        subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-I", CSRC,
                        "-o", tmp, SHIM_SRC], check=True)
        os.replace(tmp, SHIM_LIB)
    L = C.CDLL(SHIM_LIB)
    L.shim_face_flux.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp, _dp, _dp]
    L.shim_face_flux.restype = None
    L.shim_cons_to_prim.argtypes = [C.c_double, _dp, _dp]
    L.shim_cons_to_prim.restype = None
    L.shim_slope.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
    L.shim_slope.restype = C.c_double
    L.shim_cell_speed.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, _dp]
    L.shim_cell_speed.restype = C.c_double
    L.shim_half_slope.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
    L.shim_half_slope.restype = C.c_double
    L.shim_cell_speed_inline.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, _dp]
    L.shim_cell_speed_inline.restype = C.c_double
    L.shim_plm_faces.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, _dp, _dp]
    L.shim_plm_faces.restype = None
    L.shim_hlld_fast.argtypes = [C.c_int, C.c_double, _dp, _dp, _dp]
    L.shim_hlld_fast.restype = C.c_int
    L.shim_hlld_general.argtypes = [C.c_int, C.c_double, _dp, _dp, _dp]
    L.shim_hlld_general.restype = None
    L.shim_cgl_cons_to_prim.argtypes = [_dp, _dp]
    L.shim_cgl_cons_to_prim.restype = None
    L.shim_cgl_face_flux.argtypes = [C.c_int, _dp, _dp, _dp]
    L.shim_cgl_face_flux.restype = None
    L.shim_cgl_cons_to_prim_form.argtypes = [C.c_int, _dp, _dp]
    L.shim_cgl_cons_to_prim_form.restype = None
    L.shim_cgl_face_flux_form.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp]
    L.shim_cgl_face_flux_form.restype = None
    L.shim_cgl_relaxed_form.argtypes = [C.c_int, C.c_double, _dp]
    L.shim_cgl_relaxed_form.restype = C.c_double
    L.shim_cell_speed_cgl_form.argtypes = [C.c_int, _dp]
    L.shim_cell_speed_cgl_form.restype = C.c_double
    L.shim_cgl_relaxed_alog.argtypes = [C.c_double, _dp]
    L.shim_cgl_relaxed_alog.restype = C.c_double
    L.shim_cell_speed_cgl.argtypes = [_dp]
    L.shim_cell_speed_cgl.restype = C.c_double
    return L


def _p(a):
    return a.ctypes.data_as(_dp)


def shim_flux(L, eqset, riemann, d, gamma, WL, WR, d_i=0.0, dxmin=1.0, J=None):
    WL = np.ascontiguousarray(WL, dtype=np.float64); WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.empty(8)
    if J is None:
        L.shim_face_flux(eqset, riemann, d, gamma, d_i, dxmin, _p(WL), _p(WR), None, _p(F))
    else:
        J = np.ascontiguousarray(J, dtype=np.float64)
        L.shim_face_flux(eqset, riemann, d, gamma, d_i, dxmin, _p(WL), _p(WR), _p(J), _p(F))
    return F


def rand_state(rng, amp=0.5):
    W = np.empty(8)
    W[0] = 0.2 + 2.0 * rng.random()
    W[4] = 0.1 + 2.0 * rng.random()
    W[1:4] = amp * (2 * rng.random(3) - 1)
    W[5:8] = amp * (2 * rng.random(3) - 1)
    return W


def relerr(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


@pytest.mark.parametrize("riemann", [0, 1])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_flux_random_pairs(shim, riemann, d):
    rng = np.random.default_rng(100 + 10 * riemann + d)
    worst = 0.0
    branches = set()
    for n in range(4000):
        amp = [0.1, 0.5, 2.0, 6.0][n % 4]       # the large amplitudes reach the supersonic branches
        WL, WR = rand_state(rng, amp), rand_state(rng, amp)
        if n % 7 == 0:
            WR = WL + 1e-3 * (rand_state(rng) - 1.0)      # near-smooth pair
            WR[0] = abs(WR[0]) + 0.1; WR[4] = abs(WR[4]) + 0.1
        Fo = oracle.face_flux(riemann, d, G, WL, WR)
        Fs = shim_flux(shim, 0, riemann, d, G, WL, WR)
        worst = max(worst, relerr(Fs, Fo))
        if riemann == 1:
            branches.add(oracle.hlld_branch(d, G, WL, WR) % 10)
    assert worst < 2e-13, worst
    if riemann == 1:
        assert branches == {0, 1, 2, 3, 4, 5}, branches     # every branch of the fan was exercised


def test_hlld_degenerate_cases(shim):
    """P6-style degenerate inputs: identical states, B = 0 (HLLC limit), Bn = 0, B_t = 0 with c_A > a."""
    cases = []
    W = np.array([1.0, 0.3, -0.2, 0.1, 0.6, 0.7, 0.2, -0.3])
    cases.append((W, W.copy()))
    Wh = np.array([1.0, 0.3, -0.2, 0.1, 0.6, 0.0, 0.0, 0.0])
    Wh2 = np.array([0.5, -0.1, 0.2, 0.0, 0.3, 0.0, 0.0, 0.0])
    cases.append((Wh, Wh2)); cases.append((Wh2, Wh))
    Wd = np.array([1.0, 0.1, 0.0, 0.0, 0.1, 1.0, 0.0, 0.0])          # B = (B0,0,0), B0^2/rho > gamma p/rho
    cases.append((Wd, Wd.copy()))
    Wd2 = Wd.copy(); Wd2[0] = 0.7
    cases.append((Wd, Wd2)); cases.append((Wd2, Wd))
    Wn = np.array([1.0, 0.2, 0.1, 0.0, 0.5, 0.0, 0.4, 0.3])           # Bn = 0 along x
    Wn2 = np.array([0.8, -0.2, 0.0, 0.1, 0.4, 0.0, -0.3, 0.2])
    cases.append((Wn, Wn2)); cases.append((Wn2, Wn))
    for WL, WR in cases:
        for d in range(3):
            # permute so that the special structure sits along direction d
            perm = [0] + [1 + (c - d) % 3 for c in range(3)] + [4] + [5 + (c - d) % 3 for c in range(3)]
            wl, wr = WL[perm], WR[perm]
            Fo = oracle.face_flux(1, d, G, wl, wr)
            Fs = shim_flux(shim, 0, 1, d, G, wl, wr)
            assert relerr(Fs, Fo) < 1e-13, (WL, WR, d, Fs, Fo)


def test_hlld_fast_and_general_bodies(shim):
    """The two HLLD bodies of the CUDA path on their own.  The lean body (star-region flux function, one-sided pt*,
    c_f = N rsqrt(N rho)) must agree with the oracle on every face it accepts, and it must hand every supersonic
    or degenerate face (oracle branches 0, 5 and the eps-guarded star states) to the general body, which must agree
    with the oracle everywhere."""
    rng = np.random.default_rng(77)
    worst_fast, worst_gen, nslow, seen = 0.0, 0.0, 0, set()
    Ff, Fg = np.empty(8), np.empty(8)
    for n in range(6000):
        amp = [0.1, 0.5, 2.0, 6.0][n % 4]
        WL, WR = rand_state(rng, amp), rand_state(rng, amp)
        if n % 7 == 0:
            WR = WL + 1e-3 * (rand_state(rng) - 1.0)
            WR[0] = abs(WR[0]) + 0.1; WR[4] = abs(WR[4]) + 0.1
        if n % 11 == 0:
            WL[5:8] *= [1.0, 0.0, 0.0][n % 3]; WR[5:8] = WL[5:8]        # B = 0, or B along one axis on both sides
        d = n % 3
        Fo = oracle.face_flux(1, d, G, WL, WR)
        br = oracle.hlld_branch(d, G, WL, WR) % 10
        slow = shim.shim_hlld_fast(d, G, _p(WL), _p(WR), _p(Ff))
        shim.shim_hlld_general(d, G, _p(WL), _p(WR), _p(Fg))
        worst_gen = max(worst_gen, relerr(Fg, Fo))
        if br in (0, 5):
            assert slow == 1, (n, br)                                   # supersonic faces never stay in the lean body
        if slow:
            nslow += 1
        else:
            seen.add(br)
            worst_fast = max(worst_fast, relerr(Ff, Fo))
    assert worst_gen < 2e-13 and worst_fast < 2e-13, (worst_gen, worst_fast)
    assert seen >= {1, 2, 3, 4}, seen           # both single-star and both double-star branches ran through the lean body
    assert 0 < nslow < 3000, nslow


def test_plm_faces(shim):
    """plm_faces (slope and both face states in one piece) against W -+ slope/2 of the oracle's eq.4: equal up to
    one rounding of the centred difference (c - a against dp + dm), exact zeros where eq.4 gives zero."""
    rng = np.random.default_rng(5)
    lo, hi = C.c_double(), C.c_double()
    for n in range(4000):
        a, b, c = rng.normal(size=3) * [1.0, 1e-3, 1e3][n % 3]
        if n % 5 == 0:
            a = b
        if n % 7 == 0:
            c = 2 * b - a
        if n % 13 == 0:
            a = b = c
        for lim, beta in ((0, 1.0), (1, 1.0), (2, 1.0), (2, 1.3), (2, 2.0), (3, 1.0)):
            shim.shim_plm_faces(lim, 2.0 * beta, a, b, c, C.byref(lo), C.byref(hi))
            so = oracle.slope(2 if lim == 3 else lim, beta, c - b, b - a)
            tol = 4e-16 * max(abs(c - b), abs(b - a)) + 2e-16 * abs(b)
            assert abs(hi.value - (b + 0.5 * so)) <= tol and abs(lo.value - (b - 0.5 * so)) <= tol, (lim, beta, a, b, c)
            if so == 0.0:
                assert hi.value == b and lo.value == b


def test_hall_hll_flux(shim):
    rng = np.random.default_rng(7)
    for n in range(2000):
        WL, WR = rand_state(rng), rand_state(rng)
        J = 3.0 * (2 * rng.random(3) - 1)
        d = n % 3
        Fo = oracle.face_flux(0, d, G, WL, WR, eqset=1, d_i=0.05, dxmin=1.0 / 128, J=J)
        Fs = shim_flux(shim, 1, 0, d, G, WL, WR, d_i=0.05, dxmin=1.0 / 128, J=J)
        assert relerr(Fs, Fo) < 2e-13


def test_brio_wu_hand_flux(shim, golden):
    """The CUDA path's HLL against the paper-derived hand value (tests/golden/brio_wu_hll.txt)."""
    g = golden("brio_wu_hll.txt")
    WL = np.array(g["WL"]); WR = np.array(g["WR"])
    F = shim_flux(shim, 0, 0, 0, g["gamma"][0], WL, WR)
    c = g["c_fast_R"][0]
    assert np.allclose(F, np.array(g["F_LR_coeff_c"]) * c + np.array(g["F_LR_const"]), rtol=1e-14, atol=1e-15)
    F = shim_flux(shim, 0, 0, 0, g["gamma"][0], WR, WL)
    assert np.allclose(F, np.array(g["F_RL_coeff_c"]) * c + np.array(g["F_RL_const"]), rtol=1e-14, atol=1e-15)


def test_cons_to_prim_slope_speed(shim):
    rng = np.random.default_rng(3)
    for n in range(2000):
        W = rand_state(rng)
        U = oracle.prim_to_cons(W, G)
        Wo = oracle.cons_to_prim(U, G)
        Ws = np.empty(8)
        shim.shim_cons_to_prim(G, _p(U), _p(Ws))
        assert relerr(Ws, Wo) < 1e-14
        dp, dm = rng.normal(), rng.normal()
        if n % 5 == 0:
            dm = 0.0
        for lim, beta in ((0, 1.0), (1, 1.0), (2, 1.0), (2, 1.3), (2, 2.0)):
            assert shim.shim_slope(lim, beta, dp, dm) == oracle.slope(lim, beta, dp, dm)
        # A7 per-cell speed = |v| + max_d c_f,d (ideal), and with the whistler speed (Hall)
        vo = np.sqrt(np.sum(W[1:4] ** 2)) + max(oracle.cfast(d, G, W) for d in range(3))
        vs = shim.shim_cell_speed(0, G, 0.0, 1.0, _p(U))
        assert abs(vs - vo) <= 2e-15 * vo      # dt parity budget is 1e-14 relative
        cw = oracle.cwhistler(0.05, 1.0 / 64, W)
        voh = np.sqrt(np.sum(W[1:4] ** 2)) + max(max(oracle.cfast(d, G, W) for d in range(3)), cw)
        vsh = shim.shim_cell_speed(1, G, 0.05, 1.0 / 64, _p(U))
        assert abs(vsh - voh) <= 2e-15 * voh
    Ubad = oracle.prim_to_cons(np.array([1.0, 0, 0, 0, 1.0, 0, 0, 0]), G); Ubad[0] = -1.0
    assert shim.shim_cell_speed(0, G, 0.0, 1.0, _p(Ubad)) < 0


def test_half_slope_and_inline_speed(shim):
    """The kernels' own forms: half_slope (limiter constants folded, minmod variant 3) is half of eq.4 bit for bit;
    cell_speed_inline (straight-line roots in the device build, IEEE here) is the A7 speed."""
    rng = np.random.default_rng(4)
    for n in range(2000):
        dp, dm = rng.normal(), rng.normal()
        if n % 5 == 0:
            dm = 0.0
        if n % 7 == 0:
            dm = dp
        for lim, beta in ((0, 1.0), (1, 1.0), (2, 1.0), (2, 1.3), (2, 2.0)):
            assert shim.shim_half_slope(lim, 0.5 * beta, dp, dm) == 0.5 * oracle.slope(lim, beta, dp, dm)
        assert shim.shim_half_slope(3, 0.5, dp, dm) == 0.5 * oracle.slope(2, 1.0, dp, dm)
        W = rand_state(rng)
        U = oracle.prim_to_cons(W, G)
        vo = np.sqrt(np.sum(W[1:4] ** 2)) + max(oracle.cfast(d, G, W) for d in range(3))
        assert abs(shim.shim_cell_speed_inline(0, G, 0.0, 1.0, _p(U)) - vo) <= 3e-15 * vo
        cw = oracle.cwhistler(0.05, 1.0 / 64, W)
        voh = np.sqrt(np.sum(W[1:4] ** 2)) + max(max(oracle.cfast(d, G, W) for d in range(3)), cw)
        assert abs(shim.shim_cell_speed_inline(1, G, 0.05, 1.0 / 64, _p(U)) - voh) <= 3e-15 * voh


def test_cgl_point_functions(shim):
    """CGL (R24): recovery, HLL flux in all three directions, relaxed A_log and the eq.28 cell speed of the kernels'
    header against the oracle."""
    rng = np.random.default_rng(6)
    def rand9():
        W = np.empty(9)
        W[0] = 0.3 + 2 * rng.random(); W[4] = 0.2 + 2 * rng.random(); W[8] = 0.2 + 2 * rng.random()
        W[1:4] = rng.normal(size=3) * 0.5
        W[5:8] = 0.3 + rng.random(3)
        return W
    for _ in range(500):
        WL, WR = rand9(), rand9()
        U = oracle.cgl_prim_to_cons(WL)
        Ws = np.empty(9)
        shim.shim_cgl_cons_to_prim(_p(U), _p(Ws))
        assert relerr(Ws, oracle.cgl_cons_to_prim(U)) < 1e-14
        for d in range(3):
            F = np.empty(9)
            shim.shim_cgl_face_flux(d, _p(WL), _p(WR), _p(F))
            assert relerr(F, oracle.cgl_face_flux(d, WL, WR)) < 5e-14
        for f in (0.5, 0.99):
            W2 = oracle.cgl_cons_to_prim(U)
            B2 = float(np.sum(W2[5:8] ** 2))
            a, b = oracle.cgl_relax(f, B2, W2[4], W2[8])
            want = W2[0] * np.log((W2[0] ** 2 / (B2 * np.sqrt(B2))) * (b / a))
            assert abs(shim.shim_cgl_relaxed_alog(f, _p(U)) - want) <= 1e-13 * max(1.0, abs(want))
        vo = np.sqrt(np.sum(WL[1:4] ** 2)) + max(oracle.cgl_cfast(d, WL) for d in range(3))
        assert abs(shim.shim_cell_speed_cgl(_p(U)) - vo) <= 5e-15 * vo


def test_cgl_point_functions_nonlog_form(shim):
    """The same point functions with the variable of eq.16 (eqs.24-25; cgl_form = 1) against the oracle."""
    rng = np.random.default_rng(16)
    def rand9():
        W = np.empty(9)
        W[0] = 0.3 + 2 * rng.random(); W[4] = 0.2 + 2 * rng.random(); W[8] = 0.2 + 2 * rng.random()
        W[1:4] = rng.normal(size=3) * 0.5
        W[5:8] = 0.3 + rng.random(3)
        return W
    for _ in range(300):
        WL, WR = rand9(), rand9()
        U = oracle.cgl_prim_to_cons(WL, form=1)
        Ws = np.empty(9)
        shim.shim_cgl_cons_to_prim_form(1, _p(U), _p(Ws))
        assert relerr(Ws, oracle.cgl_cons_to_prim(U, form=1)) < 1e-14
        for d in range(3):
            F = np.empty(9)
            shim.shim_cgl_face_flux_form(1, d, _p(WL), _p(WR), _p(F))
            assert relerr(F, oracle.cgl_face_flux(d, WL, WR, form=1)) < 5e-14
        W2 = oracle.cgl_cons_to_prim(U, form=1)
        B2 = float(np.sum(W2[5:8] ** 2))
        a, b = oracle.cgl_relax(0.99, B2, W2[4], W2[8])
        want = (W2[0] ** 3 / (B2 * np.sqrt(B2))) * (b / a)                           # eq.16 of the relaxed pressures
        assert abs(shim.shim_cgl_relaxed_form(1, 0.99, _p(U)) - want) <= 1e-13 * max(1.0, abs(want))
        vo = np.sqrt(np.sum(WL[1:4] ** 2)) + max(oracle.cgl_cfast(d, WL) for d in range(3))
        assert abs(shim.shim_cell_speed_cgl_form(1, _p(U)) - vo) <= 5e-15 * vo
