"""Pins of the oracle's CGL MHD with the GLM scalar (eqset CGL_GLM; eqs.19-23; R30).

Eqs.22-23 are eqs.10-11 again: the (B_n, psi) subsystem is the same 2x2 linear system, so R30 reuses R22's face rule
(pinned by G1/G4) around CGL's flux (pinned by C1-C11).  What is new is the wiring -- ten variables, psi at index 9, A at
index 8, c_h from eq.28's CGL speeds -- and that is what these pins hold down: the two parents as bit-exact special
cases, the closed form of the linear subsystem, a face-by-face recomposition from the separately pinned pieces,
conservation and the psi budget, and the transposition symmetry.
"""
import numpy as np
import pytest

import oracle


def cgl_glm_cons(W, form=0):
    """U[10] from W = (rho, v, p_par, B, p_perp, psi): CGL's variable change (C1, C11) with psi carried along."""
    return np.concatenate([oracle.cgl_prim_to_cons(np.asarray(W[:9], dtype=float), form), [W[9]]])


def field_cons(W, form=0):
    U = np.empty_like(W)
    for idx in np.ndindex(W.shape[1:]):
        U[(slice(None),) + idx] = cgl_glm_cons(W[(slice(None),) + idx], form)
    return U


@pytest.mark.parametrize("form", [0, 1])
@pytest.mark.parametrize("relax", [0.0, 0.99])
def test_g9_one_dimensional_flow_is_plain_cgl(form, relax):
    """1-D flow along x with uniform B_x and psi = 0: B_n* = B_x and psi* = 0 exactly on every face, so the first nine
    variables evolve bit for bit as in the nine-variable CGL solver (whose runs C4-C6 tie to the paper's numbers), psi
    stays zero, and both choose the same dt.  The state is the paper's firehose setup with a density ripple."""
    n = 48
    x = (np.arange(n) + 0.5) / n
    W = np.zeros((10, 1, 1, n))
    W[0] = 1.0 + 0.1 * np.sin(2 * np.pi * x); W[4] = 104.0; W[8] = 3.0; W[5] = 10.0
    W[2, 0, 0] = 1e-3 * np.sin(2 * np.pi * x); W[6, 0, 0] = 1e-2 * np.cos(2 * np.pi * x)
    U10 = field_cons(W, form)
    kw = dict(shape=(n, 1, 1), dx=(1.0 / n, 1, 1), ndim=1, riemann=oracle.HLL, beta=1.3, relax=relax, cgl_form=form)
    a = oracle.RefSolver(eqset=oracle.CGL_GLM, **kw); a.set_state(U10)
    b = oracle.RefSolver(eqset=oracle.CGL, **kw); b.set_state(U10[:9])
    assert a.nvar == 10 and b.nvar == 9
    for _ in range(10):
        dt = b.compute_dt()
        assert a.compute_dt() == dt
        a.step(dt); b.step(dt)
    Va, Vb = a.get_state(), b.get_state()
    assert np.array_equal(Va[:9].view(np.uint64), Vb.view(np.uint64))
    assert np.all(Va[9] == 0.0)
    assert not np.array_equal(Va[:9], U10[:9])


def test_g9_uniform_state_decays_exactly():
    """Uniform state, psi = const: the nine CGL variables stay bitwise fixed (no relaxation: the state is inside the
    stable band), psi is multiplied by exp(-dt c_h / 0.18) per step, and c_h = 0.95 v_max with eq.28's speed written out:
    |v| + max_d c_d, c_d from eq.29 -- for B along x: parallel max(3 p_par, B^2 + p_perp - p_par)/rho, perpendicular
    (B^2 + 2 p_perp)/rho (C2)."""
    rho, v, ppar, B, pperp, psi = 1.3, np.array([0.2, -0.1, 0.05]), 1.0, 2.0, 1.2, 0.37     # C8's stable state
    W = np.array([rho, *v, ppar, B, 0.0, 0.0, pperp, psi])
    U = np.tile(cgl_glm_cons(W)[:, None, None, None], (1, 1, 9, 10))
    s = oracle.RefSolver(shape=(10, 9, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=oracle.CGL_GLM, riemann=oracle.HLL, relax=0.99)
    s.set_state(U)
    vm = np.sqrt(v @ v) + np.sqrt(max(3 * ppar, B * B + pperp - ppar, B * B + 2 * pperp) / rho)
    assert abs(s.vmax() - vm) <= 1e-14 * vm
    vm0 = s.vmax()
    for _ in range(3):
        dt = s.step(0.0)
        assert s.glm_ch() == 0.95 * vm0
        psi *= np.exp(-dt * s.glm_ch() / 0.18)
    V = s.get_state()
    assert np.array_equal(V[:9].view(np.uint64), U[:9].view(np.uint64))
    assert np.allclose(V[9], psi, rtol=1e-15, atol=0) and V[9].min() == V[9].max()


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_g9_linear_glm_wave_closed_form(axis):
    """G4's closed form holds unchanged: B_n's flux is psi* and psi's is c_h^2 B_n*, whatever the fluid's flux, so
    after one forward-Euler step with first-order states the Fourier amplitudes of (B_n, psi) are those of upwinding
    the characteristic variables B_n +- psi/c_h, with psi damped by exp(-dt c_h/0.18)."""
    n, m, eps, B0 = 32, 3, 1e-3, 0.5
    shape = [1, 1, 1]
    ndim = axis + 1
    for d in range(ndim):
        shape[d] = n if d == axis else 4
    dx = tuple(1.0 / shape[d] if d < ndim else 1.0 for d in range(3))
    idx = np.indices((shape[2], shape[1], shape[0]))[2 - axis]
    xc = (idx + 0.5) / n
    W = np.zeros((10,) + xc.shape)
    W[0] = 1.0; W[4] = 1.0; W[8] = 1.2
    W[5 + axis] = B0 + eps * np.cos(2 * np.pi * m * xc)
    U = field_cons(W)
    s = oracle.RefSolver(shape=tuple(shape), dx=dx, ndim=ndim, eqset=oracle.CGL_GLM, riemann=oracle.HLL, limiter=0, rk=1)
    s.set_state(U)
    dt = 0.3 * dx[axis] / s.vmax()
    s.step(dt)
    ch = s.glm_ch()
    V = s.get_state()
    line = [0, 0, 0]; line[2 - axis] = slice(None)
    bhat = np.fft.fft(V[5 + axis][tuple(line)])[m] / (n / 2)
    phat = np.fft.fft(V[9][tuple(line)])[m] / (n / 2)
    ph0 = np.exp(1j * 2 * np.pi * m * 0.5 / n)
    nu, th = ch * dt / dx[axis], 2 * np.pi * m / n
    gp, gm = 1 - nu * (1 - np.exp(-1j * th)), 1 - nu * (1 - np.exp(1j * th))
    assert abs(bhat - eps * ph0 * 0.5 * (gp + gm)) <= 1e-13
    assert abs(phat - eps * ph0 * 0.5 * ch * (gp - gm) * np.exp(-dt * ch / 0.18)) <= 1e-13
    for c in range(3):
        if c != axis:
            assert np.all(V[5 + c] == 0.0)


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("form", [0, 1])
def test_g9_step_recomposed_from_the_pinned_pieces(axis, form):
    """One forward-Euler step with first-order states along one axis, rebuilt face by face from the two separately
    pinned routines: the face's (B_n*, psi*) from glm_face (G1), CGL's HLL flux (C3, C5, C11) of the two states with
    B_n* on both sides, then F[B_n] = psi*, F[psi] = c_h^2 B_n*;  U' = U - dt (F_{i+1/2} - F_{i-1/2})/dx, and psi times
    the decay.  A wrong index (A and psi swapped, the flux written to a transverse component, c_h not squared) fails."""
    rng = np.random.default_rng(11 + axis)
    n = 12
    shape = [1, 1, 1]
    ndim = axis + 1
    for d in range(ndim):
        shape[d] = n if d == axis else 3
    dx = tuple(0.1 if d < ndim else 1.0 for d in range(3))
    W1 = np.empty((10, n))
    W1[0] = 0.8 + rng.random(n); W1[1:4] = 0.3 * rng.standard_normal((3, n)); W1[4] = 0.5 + rng.random(n)
    W1[5:8] = 0.6 * rng.standard_normal((3, n)) + 0.4; W1[8] = 0.5 + rng.random(n); W1[9] = 0.1 * rng.standard_normal(n)
    U1 = np.stack([cgl_glm_cons(W1[:, i], form) for i in range(n)], axis=1)
    full = [shape[2], shape[1], shape[0]]
    sl = [None, None, None]; sl[2 - axis] = slice(None)
    U = np.broadcast_to(U1[(slice(None),) + tuple(sl)], [10] + full).copy()
    s = oracle.RefSolver(shape=tuple(shape), dx=dx, ndim=ndim, eqset=oracle.CGL_GLM, riemann=oracle.HLL, limiter=0, rk=1,
                         cgl_form=form)
    s.set_state(U)
    dt = 0.4 * dx[axis] / s.vmax()
    s.step(dt)
    ch = s.glm_ch()
    F = np.empty((10, n))                       # F[:, i] = flux through face i-1/2 (periodic)
    for i in range(n):
        L, R = W1[:, i - 1].copy(), W1[:, i].copy()
        bns, pss = oracle.glm_face(ch, L[5 + axis], R[5 + axis], L[9], R[9])
        L[5 + axis] = R[5 + axis] = bns
        F[:9, i] = oracle.cgl_face_flux(axis, L[:9], R[:9], form)
        F[5 + axis, i] = pss
        F[9, i] = ch * ch * bns
    want = U1 - dt * (np.roll(F, -1, axis=1) - F) / dx[axis]
    want[9] *= np.exp(-dt * ch / 0.18)
    line = [0, 0, 0]; line[2 - axis] = slice(None)
    got = s.get_state()[(slice(None),) + tuple(line)]
    scale = np.max(np.abs(want), axis=1, keepdims=True) + 1e-300
    assert np.max(np.abs(got - want) / scale) <= 1e-13
    # and the lines are copies of each other
    assert np.ptp(s.get_state(), axis=tuple(1 + a for a in range(3) if a != 2 - axis)).max() == 0.0


def _state2d(n, div_err, form=0):
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x, indexing="xy")
    W = np.zeros((10, 1, n, n))
    W[0, 0] = 1.0 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    W[1, 0] = 0.3 * np.sin(2 * np.pi * Y); W[2, 0] = -0.3 * np.sin(2 * np.pi * X); W[3, 0] = 0.1 * np.cos(2 * np.pi * (X + Y))
    W[4, 0] = 0.8 + 0.2 * np.cos(2 * np.pi * X); W[8, 0] = 0.6 + 0.3 * np.sin(2 * np.pi * Y)
    W[5, 0] = 0.5 - 0.4 * np.sin(2 * np.pi * Y); W[6, 0] = 0.4 * np.sin(4 * np.pi * X); W[7, 0] = 0.2
    W[5, 0] += div_err * np.exp(-((X - 0.5) ** 2 + (Y - 0.5) ** 2) / 0.01)
    W[9, 0] = 0.02 * np.cos(2 * np.pi * X) + 0.01
    return field_cons(W, form)


@pytest.mark.parametrize("relax", [0.0, 0.99])
def test_g9_conservation_and_psi_budget(relax):
    """Periodic box: flux form conserves every sum; psi's sum is multiplied by the decay factor each step; with the
    relaxation on, A's sum is free and the other eight stay put (the relaxation keeps e_int, C7)."""
    n = 20
    U = _state2d(n, 0.05)
    s = oracle.RefSolver(shape=(n, n, 1), dx=(1 / n, 1 / n, 1), ndim=2, eqset=oracle.CGL_GLM, riemann=oracle.HLL, beta=1.3,
                         relax=relax)
    s.set_state(U)
    sums = U.reshape(10, -1).sum(axis=1)
    for _ in range(5):
        dt = s.step(0.0)
        V = s.get_state()
        S = V.reshape(10, -1).sum(axis=1)
        scale = np.abs(V).reshape(10, -1).sum(axis=1) + 1e-300
        nq = 9 if relax == 0.0 else 8
        assert np.all(np.abs(S[:nq] - sums[:nq]) <= 1e-13 * scale[:nq])
        assert abs(S[9] - sums[9] * np.exp(-dt * s.glm_ch() / 0.18)) <= 1e-13 * scale[9]
        sums = S


def test_g9_divergence_error_is_carried_away_and_damped():
    """What the term is for: the peak central-difference divergence of a local error, ten steps on, is well
    below that of the same run without cleaning (later the flow's own truncation error takes over in both runs)."""
    n = 48
    U = _state2d(n, 0.2)
    U[9] = 0.0

    def peak_div(eqset):
        s = oracle.RefSolver(shape=(n, n, 1), dx=(1 / n, 1 / n, 1), ndim=2, eqset=eqset, riemann=oracle.HLL, beta=1.3)
        s.set_state(U if eqset == oracle.CGL_GLM else U[:9])
        s.advance(10)
        V = s.get_state()
        div = (np.roll(V[5], -1, axis=2) - np.roll(V[5], 1, axis=2) + np.roll(V[6], -1, axis=1) - np.roll(V[6], 1, axis=1)) * n / 2
        return np.max(np.abs(div))

    assert peak_div(oracle.CGL_GLM) < 0.5 * peak_div(oracle.CGL)


def test_g9_transposition_symmetry_and_rejections():
    n = 16
    U = _state2d(n, 0.03)
    perm = [0, 2, 1, 3, 4, 6, 5, 7, 8, 9]
    Ut = U.transpose(0, 1, 3, 2)[perm].copy()
    kw = dict(shape=(n, n, 1), dx=(1 / n, 1 / n, 1), ndim=2, eqset=oracle.CGL_GLM, riemann=oracle.HLL, beta=1.3, relax=0.99)
    a = oracle.RefSolver(**kw); a.set_state(U)
    b = oracle.RefSolver(**kw); b.set_state(Ut)
    for _ in range(3):
        dt = a.step(0.0)
        b.step(dt)
    Va = a.get_state()
    Vb = b.get_state().transpose(0, 1, 3, 2)[perm]
    assert np.max(np.abs(Va - Vb)) <= 1e-13
    with pytest.raises(oracle.RefError):
        oracle.RefSolver(shape=(8, 8, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=oracle.CGL_GLM, riemann=oracle.HLLD)
    with pytest.raises(oracle.RefError):
        oracle.RefSolver(shape=(8, 8, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=oracle.CGL_GLM, riemann=oracle.HLL, relax=1.5)
