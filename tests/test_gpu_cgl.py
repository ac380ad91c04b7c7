"""GPU parity of the CGL path (NEXT-2: eqset CGL, 9 variables, HLL; 2-D strip kernel and 3-D row-owner kernel) against the oracle  (-m gpu).

Bar: relative L-inf per variable <= 1e-12 after one step, <= 1e-9 after the run, dt to 1e-14.  Scale of A_log
(R24): A_log = rho log(...) is a density-weighted logarithm that passes through zero, so it is measured
against max(max|A_log|, max rho)."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

TOL_1, TOL_N, TOL_DT = 1e-12, 1e-9, 1e-14


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    return m


def rel_linf9(Ug, Ur):
    sc = np.empty(9)
    sc[0] = np.max(np.abs(Ur[0])); sc[4] = np.max(np.abs(Ur[4]))
    sc[1:4] = np.max(np.abs(Ur[1:4])); sc[5:8] = np.max(np.abs(Ur[5:8]))
    sc[8] = max(np.max(np.abs(Ur[8])), sc[0])
    return np.array([np.max(np.abs(Ug[q] - Ur[q])) / (sc[q] if sc[q] > 0 else 1.0) for q in range(9)])


def cons_field(W):
    U = np.empty_like(W)
    flat_w = W.reshape(9, -1)
    flat_u = U.reshape(9, -1)
    for i in range(flat_w.shape[1]):
        flat_u[:, i] = oracle.cgl_prim_to_cons(flat_w[:, i])
    return U


def smooth_state(n):
    x = (np.arange(n) + 0.5) / n
    X, Y = np.meshgrid(x, x, indexing="xy")
    W = np.zeros((9, 1, n, n))
    W[0] = 1.0 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    W[1] = 0.3 * np.sin(2 * np.pi * Y); W[2] = -0.3 * np.sin(2 * np.pi * X); W[3] = 0.1 * np.cos(2 * np.pi * (X + Y))
    W[4] = 0.8 + 0.2 * np.cos(2 * np.pi * X); W[8] = 0.6 + 0.3 * np.sin(2 * np.pi * Y)
    W[5] = 0.5 - 0.4 * np.sin(2 * np.pi * Y); W[6] = 0.4 * np.sin(4 * np.pi * X); W[7] = 0.2
    return cons_field(W)


def pair(ag, shape, dx, relax, stage_grid=0, **kw):
    args = dict(shape=shape, dx=dx, ndim=2, riemann=0, limiter=2, beta=1.3, rk=2, relax=relax)
    args.update(kw)
    return oracle.RefSolver(eqset=oracle.CGL, **args), ag.Agate(eqset=ag.CGL, stage_grid=stage_grid, **args)


def march(ref, gpu, steps):
    e1 = None
    for s in range(steps):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr)
        assert gpu.step(0.0) == dtg
        if s == 0:
            e1 = rel_linf9(gpu.get_state(), ref.get_state())
    return e1, rel_linf9(gpu.get_state(), ref.get_state())


@pytest.mark.parametrize("relax", [0.0, 0.99])
@pytest.mark.parametrize("n,grid", [(100, 0), (64, 30)])
def test_cgl_smooth_2d_parity(ag, relax, n, grid):
    """Smooth anisotropic 2-D state, ragged strips (n=100) and short segments (grid=30), with and without the
    relaxation of eqs.31-33 (the state crosses the mirror bound in places, so the relaxation is live)."""
    U = smooth_state(n)
    ref, gpu = pair(ag, (n, n, 1), (1 / n, 1 / n, 1), relax, stage_grid=grid)
    ref.set_state(U); gpu.set_state(U)
    e1, eN = march(ref, gpu, 8)
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    tr, tg = ref.advance(3), gpu.advance(3)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf9(gpu.get_state(), ref.get_state()) <= TOL_N)
    ref.close(); gpu.close()


def test_cgl_firehose_with_relaxation_parity(ag):
    """The paper's firehose state (p_par = 104, p_perp = 3, B_x = 10) as four identical rows, with the
    default relaxation 0.99: the relaxation pulls the anisotropy back to the firehose bound every step."""
    n = 128
    x = -6 + (np.arange(n) + 0.5) * 12 / n
    W = np.zeros((9, 1, 4, n)); W[0] = 1; W[5] = 10; W[4] = 104; W[8] = 3
    W[2] = 0.01 * np.cos(2 * np.pi * x / 6)[None, None, :]
    W[6] = 0.1 * np.cos(2 * np.pi * x / 6 + np.pi / 2)[None, None, :]
    U = cons_field(W)
    ref, gpu = pair(ag, (n, 4, 1), (12 / n, 12 / n, 1), 0.99)
    ref.set_state(U); gpu.set_state(U)
    e1, eN = march(ref, gpu, 10)
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    V = gpu.get_state()
    assert np.ptp(V, axis=2).max() == 0.0                       # the rows stay identical
    ref.close(); gpu.close()


def test_cgl_uniform_state_bitwise_fixed(ag):
    W = np.array([1.1, 0.3, -0.2, 0.1, 0.9, 0.4, 0.2, -0.3, 0.5])
    U = np.tile(oracle.cgl_prim_to_cons(W)[:, None, None, None], (1, 1, 37, 70))
    gpu = ag.Agate(shape=(70, 37, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=ag.CGL, riemann=0, relax=0.0)
    gpu.set_state(U)
    gpu.advance(4)
    assert np.array_equal(gpu.get_state(), U)
    gpu.close()


@pytest.mark.parametrize("relax", [0.0, 0.99])
def test_cgl_3d_parity(ag, relax):
    """CGL through the 3-D row-owner kernel: smooth anisotropic state at 36^3 (ragged tiles: 32 + 4 columns,
    3 x 11 + 3 rows), with and without relaxation."""
    n = 36
    x = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    W = np.zeros((9, n, n, n))
    W[0] = 1.0 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.1 * np.sin(2 * np.pi * Z)
    W[1] = 0.3 * np.sin(2 * np.pi * Y); W[2] = -0.3 * np.sin(2 * np.pi * Z); W[3] = 0.2 * np.cos(2 * np.pi * X)
    W[4] = 0.8 + 0.2 * np.cos(2 * np.pi * (X + Z)); W[8] = 0.6 + 0.3 * np.sin(2 * np.pi * Y)
    W[5] = 0.5 - 0.4 * np.sin(2 * np.pi * Y); W[6] = 0.4 * np.sin(2 * np.pi * Z); W[7] = 0.3 * np.cos(2 * np.pi * X)
    U = cons_field(W)
    args = dict(shape=(n, n, n), dx=(1 / n,) * 3, ndim=3, riemann=0, limiter=2, beta=1.3, rk=2, relax=relax)
    ref = oracle.RefSolver(eqset=oracle.CGL, **args); gpu = ag.Agate(eqset=ag.CGL, **args)
    ref.set_state(U); gpu.set_state(U)
    e1, eN = march(ref, gpu, 4)
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    tr, tg = ref.advance(2), gpu.advance(2)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf9(gpu.get_state(), ref.get_state()) <= TOL_N)
    ref.close(); gpu.close()


def test_cgl_rejected_where_not_built(ag):
    for kw in (dict(shape=(8, 8, 1), dx=(1 / 8, 1 / 8, 1), ndim=2, riemann=1),
               dict(shape=(8, 8, 1), dx=(1 / 8, 1 / 8, 1), ndim=2, riemann=0, relax=1.5)):
        with pytest.raises(ag.AgateError) as ei:
            ag.Agate(eqset=ag.CGL, **kw)
        assert ei.value.code == ag.ERR_ARG


def test_cgl_brio_wu_open_ends(ag):
    """The paper's CGL shock tube (the Brio-Wu states with zero initial anisotropy), four identical rows, open
    in x, default relaxation, run until the fast waves have left: GPU against the oracle."""
    n = 128
    x = (np.arange(n) + 0.5) / n
    left = (x < 0.5)[None, None, :]
    W = np.zeros((9, 1, 4, n))
    W[0] = np.where(left, 1.0, 0.125); W[4] = np.where(left, 1.0, 0.1); W[8] = W[4]
    W[5] = 0.75; W[6] = np.where(left, 1.0, -1.0)
    U = cons_field(W)
    ref, gpu = pair(ag, (n, 4, 1), (1 / n, 1 / n, 1), 0.99, bc=(1, 0, 0))
    ref.set_state(U); gpu.set_state(U)
    tr, tg = ref.advance(300), gpu.advance(300)
    assert abs(tg - tr) <= 1e-12 * tr and tr > 0.15
    assert np.all(rel_linf9(gpu.get_state(), ref.get_state()) <= TOL_N)
    ref.close(); gpu.close()


@pytest.mark.parametrize("seed", range(6))
def test_cgl_random_shapes_and_options(ag, seed):
    """Seeded sweep for the CGL path: ragged 2-D and 3-D shapes, every limiter and RK scheme, relaxation on and off,
    periodic and open ends, default and forced work splits -- 3 steps against the oracle."""
    rng = np.random.default_rng(8000 + seed)
    ndim = int(rng.choice([2, 3]))
    nx, ny = int(rng.choice([29, 31, 33, 61, 64])), int(rng.choice([5, 11, 12, 23]))
    nz = int(rng.choice([4, 9, 17])) if ndim == 3 else 1
    limiter, beta = [(0, 1.0), (1, 1.0), (2, 1.0), (2, 1.3)][int(rng.integers(4))]
    rk = int(rng.choice([1, 2, 3, 4, 5]))
    relax = float(rng.choice([0.0, 0.5, 0.99]))
    bc = tuple(int(b) for b in rng.integers(0, 2, 3))
    sg = int(rng.choice([1, 5, 40])) if rng.random() < 0.5 else 0
    shp = (nz, ny, nx)
    W = np.empty((9,) + shp)
    W[0] = 0.5 + rng.random(shp); W[4] = 0.5 + rng.random(shp); W[8] = 0.5 + rng.random(shp)
    for q in (1, 2, 3):
        W[q] = 0.3 * (2 * rng.random(shp) - 1)
    for q in (5, 6, 7):
        W[q] = 0.4 + 0.3 * (2 * rng.random(shp) - 1)               # |B| bounded away from zero (A_log needs it)
    U = cons_field(W)
    kw = dict(shape=(nx, ny, nz), dx=(1.0 / nx, 1.3 / ny, 0.7 / nz if ndim == 3 else 1.0), ndim=ndim, riemann=0,
              limiter=limiter, beta=beta, rk=rk, bc=bc, relax=relax)
    ref = oracle.RefSolver(eqset=oracle.CGL, **kw); gpu = ag.Agate(eqset=ag.CGL, stage_grid=sg, **kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(3):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr, (kw, s)
        ref.step(0.5 * dtr); gpu.step(0.5 * dtr)
        e = rel_linf9(gpu.get_state(), ref.get_state())
        assert np.all(e <= 1e-11), (kw, s, e)
    ref.close(); gpu.close()


# ---- the non-logarithmic variable of eq.16 (cgl_form = 1) ---------------------------------------------------
def to_form1(U):
    """The same primitive state with A of eq.16 in place of A_log."""
    V = np.empty_like(U)
    fu, fv = U.reshape(9, -1), V.reshape(9, -1)
    for i in range(fu.shape[1]):
        fv[:, i] = oracle.cgl_prim_to_cons(oracle.cgl_cons_to_prim(fu[:, i]), form=1)
    return V


@pytest.mark.parametrize("relax", [0.0, 0.99])
@pytest.mark.parametrize("ndim,n,grid", [(2, 100, 0), (2, 64, 30), (3, 36, 0), (1, 75, 0)])
def test_cgl_nonlog_form_parity(ag, relax, ndim, n, grid):
    if ndim == 2:
        U = to_form1(smooth_state(n)); shape, dx = (n, n, 1), (1 / n, 1 / n, 1)
    elif ndim == 3:
        U2 = to_form1(smooth_state(n))
        U = np.ascontiguousarray(np.repeat(U2, n, axis=1)) * 1.0
        z = (np.arange(n) + 0.5) / n
        U[3] = U[0] * 0.1 * np.sin(2 * np.pi * z)[:, None, None]          # a z-dependent flow so every sweep works
        shape, dx = (n, n, n), (1 / n, 1 / n, 1 / n)
    else:
        U = to_form1(smooth_state(n))[:, :, :1, :].copy(); shape, dx = (n, 1, 1), (1 / n, 1, 1)
    kw = dict(shape=shape, dx=dx, ndim=ndim, riemann=0, limiter=2, beta=1.3, rk=2, relax=relax, cgl_form=1)
    ref = oracle.RefSolver(eqset=oracle.CGL, **kw); gpu = ag.Agate(eqset=ag.CGL, stage_grid=grid, **kw)
    ref.set_state(U); gpu.set_state(U)
    e1, eN = march(ref, gpu, 6)
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    ref.close(); gpu.close()
    with pytest.raises(ag.AgateError):
        ag.Agate(eqset=ag.CGL, shape=(8, 8, 1), dx=(1, 1, 1), ndim=2, riemann=0, cgl_form=2)
