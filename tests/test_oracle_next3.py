"""Pins of the oracle's NEXT-3 pieces and of the Hall face current's transverse branch (R15, R27, R28).

P14  the 2-D whistler wave of PAPER.md §4.3 (L312-316) with the sheared zero-gradient ends in y (R28): Table 1's
     "2D test" column (L286-294), second order; the same wave in a doubly periodic box whose sides fit the oblique
     wave vector (no special boundary) gives the same numbers; a random state with the (1,2) translational
     symmetry has an L(U) with that symmetry bit for bit, boundary rows included.
     These runs are the pin of the TRANSVERSE branch of the face current (the average of the two adjacent cells'
     central differences, R15): the wave vector has a component across every face normal, so a wrong factor or
     sign there changes the whistler dispersion and the error stops converging (a factor 2 gives 0.87 / 0.98 at
     n = 16 / 32, a flipped sign 1.06 / 1.21, against 0.365 / 0.095).
P15  RK43 / RK53 (R27): closed-form amplification factor with each scheme's stability polynomial (the terms
     up to z^3 are fixed by third order; z^4, z^5 by composing the stages by hand), and third order in dt on a
     fixed grid.
C10  CGL relaxation on a grid (eqs.31-33): with f = 1 every zone ends inside the firehose,
     mirror and ion-cyclotron bounds, (rho, m, E, B) are bit for bit those of the unrelaxed step, the mean
     pressure is kept, zones that were inside the bounds do not move.
"""
import math

import numpy as np
import pytest

import oracle
import workloads
from conftest import read_golden

G53 = 5.0 / 3.0


# ------------------------------------------------------------------------------------------------
# P14: rotated whistler wave
# ------------------------------------------------------------------------------------------------
def _whistler_2d(n, sheared, threads=4):
    g = read_golden("whistler.txt")
    d_i, B0, lam, db = g["d_i"][0], g["v_A"][0], g["wavelength"][0], g["delta_b"][0]
    k = 2 * math.pi / lam
    vphi = d_i * B0 * k / 2 + math.sqrt(B0 ** 2 + (d_i * B0 * k) ** 2 / 4)          # eq.34
    tau = lam / vphi
    al = math.atan(0.5)                                                              # L312
    ca, sa = math.cos(al), math.sin(al)
    if sheared:
        Lx = Ly = lam / ca                   # L314: x, y in [-100/cos a, 100/cos a]; k_y L_y = pi -> sheared ends
        nx = ny = n
    else:
        Lx, Ly = lam / ca, lam / sa          # k.(L_x, 0) = k.(0, L_y) = 2 pi: doubly periodic, same dx = dy
        nx, ny = n, 2 * n
    dx, dy = Lx / nx, Ly / ny
    x = -Lx / 2 + (np.arange(nx) + 0.5) * dx
    y = -Ly / 2 + (np.arange(ny) + 0.5) * dy
    X, Y = np.meshgrid(x, y)
    ph = k * ca * X + k * sa * Y
    dv = db * B0 / (vphi * 1.0)
    W = np.zeros((8, 1, ny, nx))
    W[0], W[4] = 1.0, 1.0
    W[1, 0], W[2, 0], W[3, 0] = dv * np.cos(ph) * sa, -dv * np.cos(ph) * ca, dv * np.sin(ph)
    W[5, 0] = B0 * ca - db * np.cos(ph) * sa
    W[6, 0] = B0 * sa + db * np.cos(ph) * ca
    W[7, 0] = -db * np.sin(ph)
    U0 = workloads.prim_to_cons(W, G53)
    s = oracle.RefSolver((nx, ny, 1), (dx, dy, 1.0), 2, eqset=oracle.HALL, riemann=oracle.HLL, limiter=2, beta=1.3,
                         rk=2, cfl=0.0, d_i=d_i, bc=(0, 2 if sheared else 0, 0))     # cfl<=0 -> 2-D default 0.45
    s.set_state(U0)
    oracle.set_threads(threads)              # bitwise identical to the serial run (test_threads_bitwise_identical)
    try:
        t = 0.0
        while t < tau * (1 - 1e-13):
            dt = min(s.compute_dt(), tau - t)
            s.step(dt)
            t += dt
    finally:
        oracle.set_threads(1)
    U = s.get_state()
    return np.abs(U[7] - U0[7]).sum() / np.abs(U0[7]).sum()                          # eq.35


def test_p14_whistler_2d_table1():
    g = read_golden("whistler.txt")
    ns = [int(v) for v in g["table1_n"]][:3]             # 16, 32, 64 (128 costs 8x the 64 run; same slope)
    paper = g["table1_2d"][:3]
    errs = [_whistler_2d(n, True) for n in ns]
    for e, pval in zip(errs, paper):
        assert pval / 1.5 < e < pval * 1.5, (errs, paper)
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]
    assert all(1.8 < sl < 2.3 for sl in slopes), slopes


def test_p14_oblique_periodic_whistler_matches_the_sheared_run():
    """No special boundary: the box fits the oblique wave vector.  Same wave, same dx = dy, same dt, so the
    eq.35 errors agree to round-off-driven differences; both converge at second order."""
    errs = [_whistler_2d(n, False) for n in (16, 32)]
    ref = [_whistler_2d(n, True) for n in (16, 32)]
    for a, b in zip(errs, ref):
        assert abs(a - b) < 1e-6 * b, (errs, ref)
    assert 1.8 < math.log2(errs[0] / errs[1]) < 2.3, errs


@pytest.mark.parametrize("eqset", [oracle.IDEAL, oracle.HALL])
def test_p14_sheared_ends_keep_the_translational_symmetry(eqset):
    """U(i, j) = g[(2 i + j) mod 2 nx] is invariant under (i, j) -> (i - 1, j + 2).  With the sheared ends the
    ghost rows continue that pattern, so L(U) has the same symmetry bit for bit in EVERY row; any other rule
    (plain zero-gradient, the shift with the wrong sign, a shift by one row) breaks it in the two rows next to
    each end."""
    nx, ny = 12, 9
    rng = np.random.default_rng(7)
    gtab = rng.uniform(-0.3, 0.3, size=(8, 2 * nx))
    gtab[0] = 1.0 + 0.5 * np.abs(gtab[0]); gtab[4] = 0.6 + np.abs(gtab[4])
    i, j = np.meshgrid(np.arange(nx), np.arange(ny))
    W = gtab[:, (2 * i + j) % (2 * nx)][:, None]
    U0 = workloads.prim_to_cons(W, G53)
    s = oracle.RefSolver((nx, ny, 1), (0.1, 0.1, 1.0), 2, eqset=eqset, riemann=oracle.HLL, limiter=2, beta=1.3,
                         d_i=0.4 if eqset == oracle.HALL else 0.0, bc=(0, 2, 0))
    s.set_state(U0)
    L = s.rhs()
    assert np.abs(L).max() > 1e-3
    for jj in range(ny - 2):
        a = L[:, 0, jj, :]
        b = np.roll(L[:, 0, jj + 2, :], 1, axis=-1)          # b[i] = L(i - 1, j + 2)
        assert np.array_equal(a.view(np.uint64), b.view(np.uint64)), jj
    # and the rule is needed: plain zero-gradient ends do break it
    s2 = oracle.RefSolver((nx, ny, 1), (0.1, 0.1, 1.0), 2, eqset=eqset, riemann=oracle.HLL, limiter=2, beta=1.3,
                          d_i=0.4 if eqset == oracle.HALL else 0.0, bc=(0, 1, 0))
    s2.set_state(U0)
    L2 = s2.rhs()
    assert not np.array_equal(L2[:, 0, 0, :], np.roll(L2[:, 0, 2, :], 1, axis=-1))
    with pytest.raises(oracle.RefError):
        oracle.RefSolver((nx, ny, 1), (0.1, 0.1, 1.0), 2, bc=(1, 2, 0))          # sheared ends need a periodic x


# ------------------------------------------------------------------------------------------------
# P15: RK43 and RK53 (R27)
# ------------------------------------------------------------------------------------------------
def _poly_mul(a, b):
    return np.convolve(a, b)


def _stability_poly(rk):
    """Stability polynomial (ascending coefficients) of the Shu-Osher forms of R27, composed stage by stage for
    dU/dt = lambda U, z = lambda dt."""
    if rk == 4:
        e = np.array([1.0, 0.5])                                                 # 1 + z/2
        u2 = _poly_mul(e, e)
        u3 = np.array([2.0 / 3.0, 0, 0, 0]) + _poly_mul(u2, e) / 3.0
        return _poly_mul(u3, e)
    c = 0.377268915331368
    e = np.array([1.0, c])
    u2 = _poly_mul(e, e)
    u3 = 0.644090224936674 * _poly_mul(u2, e); u3[0] += 0.355909775063327
    u4 = 0.632066208361863 * _poly_mul(u3, e); u4[0] += 0.367933791638137
    u5 = 0.762406163401431 * _poly_mul(u4, e); u5[:3] += 0.237593836598569 * u2
    return u5


@pytest.mark.parametrize("rk", [4, 5])
def test_p15_stability_polynomial_is_third_order(rk):
    p = _stability_poly(rk)
    assert np.allclose(p[:4], [1.0, 1.0, 0.5, 1.0 / 6.0], rtol=0, atol=5e-15)
    if rk == 4:
        assert abs(p[4] - 1.0 / 48.0) < 1e-16 and len(p) == 5


@pytest.mark.parametrize("rk", [4, 5])
@pytest.mark.parametrize("mode", ["alfven+", "entropy"])
def test_p15_linear_eigenmode(rk, mode, monkeypatch):
    """P4's closed form with the scheme's own stability polynomial in place of 1 + z + z^2/2."""
    import test_oracle_pins as tp
    base = tp._amplification

    def amp(lam, sL, sR, hlld, limiter, theta, dt_dx, rk_):
        z = base(lam, sL, sR, hlld, limiter, theta, dt_dx, 1) - 1.0              # rk = 1 returns 1 + z
        return sum(cq * z ** q for q, cq in enumerate(_stability_poly(rk_)))

    monkeypatch.setattr(tp, "_amplification", amp)
    tp.test_p4_linear_eigenmode(oracle.HLLD, 1, mode, 0, rk=rk)
    tp.test_p4_linear_eigenmode(oracle.HLL, 1, mode, 1, rk=rk)


def _smooth_run(rk, nsteps, N=32, T=0.25):
    x = (np.arange(N) + 0.5) / N
    k = 2 * math.pi
    W = np.zeros((8, 1, 1, N))
    W[0] = 1.0 + 0.2 * np.sin(k * x); W[1] = 0.3; W[4] = 0.6; W[5] = 1.0
    W[6, 0, 0], W[7, 0, 0] = 0.1 * np.cos(k * x), 0.1 * np.sin(k * x)
    W[2, 0, 0], W[3, 0, 0] = -W[6, 0, 0], -W[7, 0, 0]
    s = oracle.RefSolver((N, 1, 1), (1.0 / N, 1, 1), 1, riemann=oracle.HLL, limiter=1, rk=rk)
    s.set_state(workloads.prim_to_cons(W, G53))
    for _ in range(nsteps):
        s.step(T / nsteps)
    return s.get_state()


def test_p15_order_in_dt():
    """Fixed grid, smooth data, unlimited slopes: the semi-discrete system is one smooth ODE for every scheme, so
    the error against a finely stepped solution falls as dt^p with p = 2 for SSP-RK22 and 3 for RK33, RK43, RK53;
    at equal dt the error constant shrinks with the stage count."""
    ref = _smooth_run(5, 4096)
    errs = {rk: [np.abs(_smooth_run(rk, n) - ref).max() for n in (32, 64, 128)] for rk in (2, 3, 4, 5)}
    for rk, e in errs.items():
        order = math.log2(e[1] / e[2])
        want = 2 if rk == 2 else 3
        assert abs(order - want) < 0.05, (rk, e)
    assert errs[5][2] < errs[4][2] < errs[3][2] < errs[2][2]


# ------------------------------------------------------------------------------------------------
# C10: CGL relaxation on a grid (eqs.31-33)
# ------------------------------------------------------------------------------------------------
def _cgl_state(n, seed):
    rng = np.random.default_rng(seed)
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x, indexing="xy")
    W = np.zeros((9, 1, n, n))
    W[0] = 1.0 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    W[1] = 0.2 * np.sin(2 * np.pi * Y); W[2] = -0.2 * np.sin(2 * np.pi * X); W[3] = 0.05
    W[5] = 0.5 - 0.3 * np.sin(2 * np.pi * Y); W[6] = 0.3 * np.sin(4 * np.pi * X); W[7] = 0.2
    # anisotropies on both sides of every bound: p_perp / p_par from 0.2 to 5
    W[4] = 0.6 * np.exp(rng.uniform(-0.8, 0.8, size=(n, n)))
    W[8] = W[4] * np.exp(rng.uniform(-1.6, 1.6, size=(n, n)))
    U = np.empty_like(W)
    for j in range(n):
        for i in range(n):
            U[:, 0, j, i] = oracle.cgl_prim_to_cons(W[:, 0, j, i])
    return U


def _bounds(w):
    B2 = w[5] ** 2 + w[6] ** 2 + w[7] ** 2
    dP = w[8] - w[4]
    return dP, -B2, (w[4] / w[8]) * B2 / 2, 0.3 * w[4] * math.sqrt(B2 / (2 * w[4]))      # L236-244, C1 = 0.3, C2 = 0.5


def test_c10_relaxation_on_a_grid():
    n = 16
    U = _cgl_state(n, 11)
    out = {}
    for f in (0.0, 1.0):
        s = oracle.RefSolver(shape=(n, n, 1), dx=(1 / n, 1 / n, 1), ndim=2, eqset=oracle.CGL, riemann=oracle.HLL,
                             beta=1.3, relax=f)
        s.set_state(U)
        s.step(2e-3)
        out[f] = s.get_state()
    free, rel = out[0.0], out[1.0]
    # (rho, m, E, B) are untouched by the relaxation: only A_log moves
    assert np.array_equal(free[:8].view(np.uint64), rel[:8].view(np.uint64))
    hit = {"firehose": 0, "mirror": 0, "ion-cyclotron": 0, "inside": 0}
    for j in range(n):
        for i in range(n):
            w0 = oracle.cgl_cons_to_prim(free[:, 0, j, i])
            w1 = oracle.cgl_cons_to_prim(rel[:, 0, j, i])
            dP0, fh0, mi0, ic0 = _bounds(w0)
            dP1, fh1, mi1, ic1 = _bounds(w1)
            tol = 1e-12 * (abs(w1[4]) + abs(w1[8]))
            assert fh1 - tol <= dP1 <= min(mi1, ic1) + tol, (i, j, dP1, fh1, mi1, ic1)
            # eq.31 with the bounds of the state being relaxed, hard wall (f = 1)
            want = max(fh0, min(dP0, mi0, ic0))
            assert abs(dP1 - want) <= tol, (i, j)
            assert abs((w1[4] + 2 * w1[8]) - (w0[4] + 2 * w0[8])) <= tol                     # mean pressure kept
            if dP0 < fh0:
                hit["firehose"] += 1
            elif dP0 > min(mi0, ic0):
                hit["mirror" if mi0 < ic0 else "ion-cyclotron"] += 1
            else:
                hit["inside"] += 1
                assert abs(rel[8, 0, j, i] - free[8, 0, j, i]) <= 1e-13 * max(1.0, abs(free[8, 0, j, i]))
            # the stored A_log is eq.18 of the relaxed pressures
            B2 = w1[5] ** 2 + w1[6] ** 2 + w1[7] ** 2
            alog = w1[0] * math.log(w1[0] ** 2 * w1[8] / (B2 ** 1.5 * w1[4]))
            assert abs(alog - rel[8, 0, j, i]) <= 1e-12 * max(1.0, abs(alog))
    assert all(v > 0 for v in hit.values()), hit
