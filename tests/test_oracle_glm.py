"""Pins of the oracle's GLM divergence cleaning (NEXT-1; eqs.10-11, constants L142; R22).

The paper gives the equations and the two constants, not the face treatment; R22 fixes it (2x2 linear Riemann problem
for (B_n, psi), c_h = 0.95 v_max(U^n), source integrated exactly after the Runge-Kutta update).  Each pin below checks
the oracle against something other than its own formulas: hand numbers, closed forms from the characteristic
solution of the linear subsystem, invariants, and the reduction to plain ideal MHD.
"""
import numpy as np
import pytest

import oracle

G = 5.0 / 3.0


def cons(W):
    """U from W = (rho, v, p, B[, psi]) -- the definition of the conserved vector (P:L140 with R2)."""
    U = np.array(W, dtype=float, copy=True)
    U[1:4] = W[0] * W[1:4]
    U[4] = W[4] / (G - 1) + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2) + 0.5 * (W[5] ** 2 + W[6] ** 2 + W[7] ** 2)
    return U


def test_g1_face_values_by_hand():
    """Characteristics of dB/dt + dpsi/dx = 0, dpsi/dt + c^2 dB/dx = 0 are B -+ psi/c at speeds -+c.  With c = 2,
    (B, psi)_L = (1, 0.5), (B, psi)_R = (3, -0.5):  B + psi/c comes from the left = 1.25,  B - psi/c from the right =
    3.25  =>  B* = 2.25, psi* = c (1.25 - 3.25)/2 = -2."""
    bn, ps = oracle.glm_face(2.0, 1.0, 3.0, 0.5, -0.5)
    assert bn == 2.25 and ps == -2.0
    # continuous data pass through unchanged
    assert oracle.glm_face(0.7, 0.3, 0.3, -0.2, -0.2) == (0.3, -0.2)


@pytest.mark.parametrize("riemann", [oracle.HLL, oracle.HLLD])
@pytest.mark.parametrize("rk", [1, 2])
def test_g2_uniform_state_decays_exactly(riemann, rk):
    """Uniform state with psi = const: no flux difference anywhere, so the 8 MHD variables stay bitwise fixed and
    psi is multiplied by exp(-dt c_h / 0.18) per step (c_p^2 = 0.18 c_h), c_h = 0.95 v_max."""
    W = np.array([1.3, 0.2, -0.1, 0.05, 0.9, 0.4, -0.3, 0.2, 0.37])
    U = np.tile(cons(W)[:, None, None, None], (1, 1, 12, 10))
    s = oracle.RefSolver(shape=(10, 12, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=oracle.IDEAL_GLM, riemann=riemann, rk=rk)
    s.set_state(U)
    vm = s.vmax()
    psi = 0.37
    for _ in range(3):
        dt = s.step(0.0)
        assert s.glm_ch() == 0.95 * vm
        psi *= np.exp(-dt * 0.95 * vm / 0.18)
    V = s.get_state()
    assert np.array_equal(V[:8], U[:8])
    assert np.allclose(V[8], psi, rtol=1e-15, atol=0)
    assert V[8].min() == V[8].max()


@pytest.mark.parametrize("riemann", [oracle.HLL, oracle.HLLD])
def test_g3_one_dimensional_flow_is_plain_ideal_mhd(riemann):
    """1-D flow along x with uniform B_x has div B = 0 identically: psi stays 0, B_x stays put, and every other
    variable must evolve bit for bit as in the 8-variable ideal solver (shock-tube data)."""
    n = 64
    x = (np.arange(n) + 0.5) / n
    left = np.abs(x - 0.5) < 0.25
    W = np.zeros((9, 1, 1, n))
    W[0] = np.where(left, 1.0, 0.125); W[4] = np.where(left, 1.0, 0.1)
    W[5] = 0.75; W[6] = np.where(left, 1.0, -1.0)
    U9 = np.stack([cons(W[:, 0, 0, i]) for i in range(n)], axis=-1).reshape(9, 1, 1, n)
    kw = dict(shape=(n, 1, 1), dx=(1.0 / n, 1, 1), ndim=1, riemann=riemann, beta=1.3)
    a = oracle.RefSolver(eqset=oracle.IDEAL_GLM, **kw); a.set_state(U9)
    b = oracle.RefSolver(eqset=oracle.IDEAL, **kw); b.set_state(U9[:8])
    for _ in range(12):
        dt = b.step(0.0)
        assert a.step(dt) == dt
    Va, Vb = a.get_state(), b.get_state()
    assert np.array_equal(Va[:8], Vb)
    assert np.all(Va[8] == 0.0)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_g4_linear_glm_wave_closed_form(axis):
    """(B_n, psi) on a uniform fluid at rest, first-order reconstruction, forward Euler: the characteristic
    variables w+- = B_n +- psi/c_h are advected by the first-order upwind scheme, whose amplification factor for
    a Fourier mode is  g+- = 1 - nu (1 - exp(-+ i k dx)),  nu = c_h dt/dx;  then psi decays by exp(-dt c_h/0.18).
    Starting from B_n = B0 + eps cos(kx), psi = 0:  B_hat -> (g+ + g-)/2,  psi_hat -> c_h (g+ - g-)/2 * decay."""
    n, m, eps, B0 = 32, 3, 1e-3, 0.5
    shape = [1, 1, 1]
    ndim = axis + 1
    for d in range(ndim):
        shape[d] = n if d == axis else 4
    dx = tuple(1.0 / shape[d] if d < ndim else 1.0 for d in range(3))
    idx = np.indices((shape[2], shape[1], shape[0]))[2 - axis]           # cell index along `axis`
    xc = (idx + 0.5) / n
    W = np.zeros((9,) + xc.shape)
    W[0] = 1.0; W[4] = 1.0
    W[5 + axis] = B0 + eps * np.cos(2 * np.pi * m * xc)
    U = W.copy(); U[4] = W[4] / (G - 1) + 0.5 * W[5 + axis] ** 2
    s = oracle.RefSolver(shape=tuple(shape), dx=dx, ndim=ndim, eqset=oracle.IDEAL_GLM, riemann=oracle.HLL, limiter=0, rk=1)
    s.set_state(U)
    dt = 0.3 * dx[axis] / s.vmax()
    s.step(dt)
    ch = s.glm_ch()
    V = s.get_state()
    line = [0, 0, 0]; line[2 - axis] = slice(None)
    bhat = np.fft.fft(V[5 + axis][tuple(line)])[m] / (n / 2)
    phat = np.fft.fft(V[8][tuple(line)])[m] / (n / 2)
    ph0 = np.exp(1j * 2 * np.pi * m * 0.5 / n)                          # phase of cos(k x) at cell centres
    nu, th = ch * dt / dx[axis], 2 * np.pi * m / n
    gp, gm = 1 - nu * (1 - np.exp(-1j * th)), 1 - nu * (1 - np.exp(1j * th))
    assert abs(bhat - eps * ph0 * 0.5 * (gp + gm)) <= 1e-13
    assert abs(phat - eps * ph0 * 0.5 * ch * (gp - gm) * np.exp(-dt * ch / 0.18)) <= 1e-13
    # nothing transverse: the other field components stay zero, the field stays uniform across the line
    for c in range(3):
        if c != axis:
            assert np.all(V[5 + c] == 0.0)
    assert np.ptp(V[5 + axis], axis=tuple(a for a in range(3) if a != 2 - axis)).max() == 0.0


def _blob_state(n, div_err):
    """Smooth 2-D state; div_err adds a B_x bump whose central-difference divergence is not zero."""
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x, indexing="xy")
    W = np.zeros((9, 1, n, n))
    W[0] = 1.0 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    W[1] = 0.3 * np.sin(2 * np.pi * Y); W[2] = -0.3 * np.sin(2 * np.pi * X); W[4] = 0.8
    W[5] = -0.4 * np.sin(2 * np.pi * Y); W[6] = 0.4 * np.sin(4 * np.pi * X); W[7] = 0.1
    W[5] += div_err * np.exp(-((X - 0.5) ** 2 + (Y - 0.5) ** 2) / 0.01)
    U = np.empty_like(W)
    for j in range(n):
        for i in range(n):
            U[:, 0, j, i] = cons(W[:, 0, j, i])
    return U


def test_g5_conservation_and_psi_budget():
    """Periodic box: the flux form conserves every variable's sum, psi's included, and the source multiplies psi by
    one number per step -- so sum(psi) after a step = decay * sum(psi) before, and the 8 MHD sums stay put."""
    n = 24
    U = _blob_state(n, 0.05)
    U[8] = 0.02 * np.cos(2 * np.pi * (np.arange(n) + 0.5) / n)[None, None, :] + 0.01
    s = oracle.RefSolver(shape=(n, n, 1), dx=(1 / n, 1 / n, 1), ndim=2, eqset=oracle.IDEAL_GLM, riemann=oracle.HLLD, beta=1.3)
    s.set_state(U)
    sums = U.reshape(9, -1).sum(axis=1)
    for _ in range(5):
        dt = s.step(0.0)
        V = s.get_state().reshape(9, -1).sum(axis=1)
        scale = np.abs(s.get_state()).reshape(9, -1).sum(axis=1) + 1e-300
        assert np.all(np.abs(V[:8] - sums[:8]) <= 1e-13 * scale[:8])
        assert abs(V[8] - sums[8] * np.exp(-dt * s.glm_ch() / 0.18)) <= 1e-13 * scale[8]
        sums = V


def test_g6_divergence_error_is_carried_away_and_damped():
    """What the term is for: a local div B error spreads out at c_h and decays.  The peak of the
    central-difference divergence after 40 steps must be well below the run without cleaning."""
    n = 48
    U = _blob_state(n, 0.05)

    def peak_div(eqset):
        s = oracle.RefSolver(shape=(n, n, 1), dx=(1 / n, 1 / n, 1), ndim=2, eqset=eqset, riemann=oracle.HLL, beta=1.3)
        s.set_state(U if eqset == oracle.IDEAL_GLM else U[:8])
        s.advance(40)
        V = s.get_state()
        div = (np.roll(V[5], -1, axis=2) - np.roll(V[5], 1, axis=2) + np.roll(V[6], -1, axis=1) - np.roll(V[6], 1, axis=1)) * n / 2
        return np.max(np.abs(div))

    assert peak_div(oracle.IDEAL_GLM) < 0.5 * peak_div(oracle.IDEAL)


def test_g7_transposition_symmetry():
    """Swapping x and y (and the x/y components of v and B) must commute with a GLM step: catches a flux written
    to the wrong component in one direction only."""
    n = 16
    U = _blob_state(n, 0.03)
    U[8] = 0.01 * np.sin(2 * np.pi * (np.arange(n) + 0.5) / n)[None, :, None]
    Ut = U.transpose(0, 1, 3, 2)[[0, 2, 1, 3, 4, 6, 5, 7, 8]].copy()
    kw = dict(shape=(n, n, 1), dx=(1 / n, 1 / n, 1), ndim=2, eqset=oracle.IDEAL_GLM, riemann=oracle.HLLD, beta=1.3)
    a = oracle.RefSolver(**kw); a.set_state(U)
    b = oracle.RefSolver(**kw); b.set_state(Ut)
    for _ in range(3):
        dt = a.step(0.0)
        b.step(dt)
    Va = a.get_state()
    Vb = b.get_state().transpose(0, 1, 3, 2)[[0, 2, 1, 3, 4, 6, 5, 7, 8]]
    # a mirror-free transposition changes the handedness: v_z and B_z pick up no sign, so equality is exact up to
    # the order of the x and y flux differences (round-off)
    assert np.max(np.abs(Va - Vb)) <= 1e-13


# ------------------------------------------------------------------------------------------------
# G8: Hall MHD with the GLM scalar (eqset HALL_GLM, R29)
# ------------------------------------------------------------------------------------------------
def test_g8_hall_glm_reduces_to_its_two_parents():
    """(i) d_i = 0: no Hall velocity and c_w = v_A <= c_f, so every bit is that of IDEAL_GLM.  (ii) psi = 0 and a
    constant B_n on a 1-D grid (the paper's whistler setup): B_n* = B_n, psi* = 0 exactly, so the first eight
    variables are bit for bit those of HALL (which P9 ties to Table 1) and psi stays zero."""
    import workloads
    wl = workloads.make_workload(6, n=24)
    a = oracle.RefSolver.from_workload(wl)
    b = oracle.RefSolver.from_workload(wl, eqset=oracle.HALL_GLM, d_i=0.0)
    a.advance(5); b.advance(5)
    assert np.array_equal(a.get_state().view(np.uint64), b.get_state().view(np.uint64))
    n = 32
    x = (np.arange(n) + 0.5) * 200.0 / n
    k = 2 * np.pi / 200.0
    W = np.zeros((8, 1, 1, n)); W[0] = 1; W[4] = 1; W[5] = 100.0
    W[2, 0, 0], W[3, 0, 0] = -6e-4 * np.cos(k * x), 6e-4 * np.sin(k * x)
    W[6, 0, 0], W[7, 0, 0] = 1e-3 * np.cos(k * x), -1e-3 * np.sin(k * x)
    U8 = workloads.prim_to_cons(W, 5.0 / 3.0)
    U9 = np.concatenate([U8, np.zeros((1, 1, 1, n))], axis=0)
    kw = dict(shape=(n, 1, 1), dx=(200.0 / n, 1, 1), ndim=1, riemann=oracle.HLL, beta=1.3, d_i=35.1076)
    h = oracle.RefSolver(eqset=oracle.HALL, **kw); h.set_state(U8)
    g = oracle.RefSolver(eqset=oracle.HALL_GLM, **kw); g.set_state(U9)
    for _ in range(20):
        dt = h.compute_dt()
        assert g.compute_dt() == dt
        h.step(dt); g.step(dt)
    V = g.get_state()
    assert np.array_equal(V[:8].view(np.uint64), h.get_state().view(np.uint64))
    assert np.all(V[8] == 0.0)


def test_g8_hall_glm_conservation_uniform_and_rejections():
    import workloads
    wl = workloads.make_workload(4, n=24)
    rng = np.random.default_rng(3)
    U = np.concatenate([wl.U, 0.01 * rng.standard_normal((1,) + wl.U.shape[1:])], axis=0)
    s = oracle.RefSolver(shape=wl.shape, dx=wl.dx, ndim=2, eqset=oracle.HALL_GLM, riemann=oracle.HLL, beta=1.0, d_i=wl.d_i,
                         cfl=wl.cfl)
    s.set_state(U)
    s0 = U.reshape(9, -1).sum(axis=1)
    s.advance(6)
    V = s.get_state()
    scale = np.abs(V).reshape(9, -1).sum(axis=1) + 1e-300
    assert np.all(np.abs(V.reshape(9, -1).sum(axis=1)[:8] - s0[:8]) <= 1e-13 * scale[:8])      # psi has a source
    assert not np.array_equal(V, U)
    Wc = np.array([1.1, 0.1, 0.2, -0.1, 0.8, 0.3, 0.2, 1.0])
    Uc = np.concatenate([workloads.prim_to_cons(np.tile(Wc[:, None, None, None], (1, 1, 6, 6)), 5.0 / 3.0),
                         np.zeros((1, 1, 6, 6))], axis=0)
    u = oracle.RefSolver(shape=(6, 6, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=oracle.HALL_GLM, riemann=oracle.HLL, d_i=0.5)
    u.set_state(Uc); u.advance(3)
    assert np.array_equal(u.get_state().view(np.uint64), Uc.view(np.uint64))
    with pytest.raises(oracle.RefError):
        oracle.RefSolver(shape=(6, 6, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=oracle.HALL_GLM, riemann=oracle.HLLD)
