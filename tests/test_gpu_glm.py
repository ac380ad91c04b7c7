"""GPU parity of the GLM path (NEXT-1: eqset IDEAL_GLM, 9 variables; 2-D strip kernel and 3-D row-owner kernel) against the oracle  (-m gpu).

Same bar as the 8-variable path: relative L-inf per variable <= 1e-12 after one step, <= 1e-9 after the run, dt to
1e-14 relative.  Scale of psi (R23): psi / c_h is the quantity that travels with B_n (the characteristic
variables of eqs.10-11 are B_n -+ psi/c_h), and psi is built from differences of B times c_h, so its round-off is
c_h |B| eps however small psi itself is: psi is measured against max(max|psi|, c_h max|B|)."""
import numpy as np
import pytest

import oracle
from workloads import make_workload

pytestmark = pytest.mark.gpu

TOL_1, TOL_N, TOL_DT = 1e-12, 1e-9, 1e-14


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    return m


def rel_linf9(Ug, Ur, ch):
    sc = np.empty(9)
    sc[0] = np.max(np.abs(Ur[0])); sc[4] = np.max(np.abs(Ur[4]))
    sc[1:4] = np.max(np.abs(Ur[1:4])); sc[5:8] = np.max(np.abs(Ur[5:8]))
    sc[8] = max(np.max(np.abs(Ur[8])), ch * sc[5])
    return np.array([np.max(np.abs(Ug[q] - Ur[q])) / (sc[q] if sc[q] > 0 else 1.0) for q in range(9)])


@pytest.mark.parametrize("n,steps,riemann,grid", [(100, 12, None, 0), (64, 6, oracle.HLLD, 0), (100, 4, None, 40),
                                                   (256, 3, None, 0)])
def test_orszag_tang_glm_parity(ag, n, steps, riemann, grid):
    """Config 6 recipe (Orszag-Tang, + GLM) at reduced size: ragged strips (n=100: 3 x 30 + 10), short
    segments (grid=40), HLL (the paper's default) and HLLD."""
    wl = make_workload(6, n=n)
    over = {} if riemann is None else {"riemann": riemann}
    ref = oracle.RefSolver.from_workload(wl, **over)
    gpu = ag.Agate.from_workload(wl, stage_grid=grid, **over)
    e1 = None
    for s in range(steps):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr)
        assert gpu.step(0.0) == dtg
        if s == 0:
            e1 = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    eN = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    assert np.max(np.abs(ref.get_state()[8])) > 0          # the cleaning field is live in this problem
    ref.close(); gpu.close()


@pytest.mark.parametrize("rk", [1, 2])
def test_glm_sequences_and_advance(ag, rk):
    """Host-chosen dt (c_h still 0.95 v_max of the current state), self-timed steps, agate_advance (graph replay)
    and a second set_state, against the oracle doing the same."""
    wl = make_workload(6, n=64)
    U0 = wl.U.copy()
    U0[8] = 0.01 * np.sin(2 * np.pi * (np.arange(64) + 0.5) / 64)[None, :, None]     # start with a live psi
    ref = oracle.RefSolver.from_workload(wl, rk=rk); ref.set_state(U0)
    gpu = ag.Agate.from_workload(wl, rk=rk); gpu.set_state(U0)
    d = ref.compute_dt()
    ref.step(0.5 * d); assert gpu.step(0.5 * d) == 0.5 * d
    d = ref.compute_dt(); assert abs(gpu.compute_dt() - d) <= TOL_DT * d
    ref.step(d); gpu.step(0.0)
    tr, tg = ref.advance(4), gpu.advance(4)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch()) <= TOL_N)
    ref.set_state(wl.U, 0.0); gpu.set_state(wl.U, 0.0)
    tr, tg = ref.advance(2), gpu.advance(2)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch()) <= TOL_N)
    ref.close(); gpu.close()


def test_glm_uniform_state_exact_decay(ag):
    """Pin G2 on the GPU: uniform state with psi = const: the 8 MHD variables stay bitwise fixed, psi is multiplied
    by exp(-dt c_h/0.18) per step."""
    W = np.array([1.3, 0.2, -0.1, 0.05, 0.9, 0.4, -0.3, 0.2, 0.37])
    U1 = W.copy(); U1[1:4] = W[0] * W[1:4]
    U1[4] = W[4] / (5 / 3 - 1) + 0.5 * W[0] * np.sum(W[1:4] ** 2) + 0.5 * np.sum(W[5:8] ** 2)
    U = np.tile(U1[:, None, None, None], (1, 1, 50, 70))
    gpu = ag.Agate(shape=(70, 50, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=ag.IDEAL_GLM, riemann=0, beta=1.3)
    ref = oracle.RefSolver(shape=(70, 50, 1), dx=(0.1, 0.1, 1), ndim=2, eqset=oracle.IDEAL_GLM, riemann=0, beta=1.3)
    gpu.set_state(U); ref.set_state(U)
    vm = ref.vmax()
    psi = 0.37
    for _ in range(3):
        dt = gpu.step(0.0)
        psi *= np.exp(-dt * 0.95 * vm / 0.18)
    V = gpu.get_state()
    assert np.array_equal(V[:8], U[:8])
    assert np.allclose(V[8], psi, rtol=1e-14, atol=0)
    gpu.close(); ref.close()


@pytest.mark.parametrize("riemann", [oracle.HLL, oracle.HLLD])
@pytest.mark.parametrize("grid", [0, 23])
def test_glm_3d_parity(ag, riemann, grid):
    """GLM through the 3-D row-owner kernel: config 3's seeded state at 40^3 (ragged tiles) plus a smooth psi and a
    divergence error in B_x; default segmentation and short segments."""
    wl = make_workload(3, n=40)
    n = 40
    x = (np.arange(n) + 0.5) / n
    U = np.empty((9, n, n, n))
    U[:8] = wl.U
    U[5] += 0.02 * np.exp(-((x[None, None, :] - 0.5) ** 2 + (x[None, :, None] - 0.4) ** 2 + (x[:, None, None] - 0.6) ** 2) / 0.02)
    U[4] = wl.U[4] + 0.5 * (U[5] ** 2 - wl.U[5] ** 2)                    # keep the pressure of the recipe
    U[8] = 0.01 * np.sin(2 * np.pi * x)[None, None, :] * np.cos(2 * np.pi * x)[:, None, None]
    kw = dict(shape=wl.shape, dx=wl.dx, ndim=3, gamma=wl.gamma, riemann=riemann, limiter=2, beta=1.3, rk=2, cfl=wl.cfl)
    ref = oracle.RefSolver(eqset=oracle.IDEAL_GLM, **kw); ref.set_state(U)
    gpu = ag.Agate(eqset=ag.IDEAL_GLM, stage_grid=grid, **kw); gpu.set_state(U)
    e1 = None
    for s_ in range(4):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr)
        assert gpu.step(0.0) == dtg
        if s_ == 0:
            e1 = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    tr, tg = ref.advance(2), gpu.advance(2)
    assert abs(tg - tr) <= 1e-13 * tr
    eN = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    ref.close(); gpu.close()


def test_glm_1d_grid_is_accepted(ag):
    """1-D GLM runs through the strip kernel as one periodic row (parity: tests/test_gpu_next3.py)."""
    g = ag.Agate(shape=(8, 1, 1), dx=(1 / 8, 1, 1), ndim=1, eqset=ag.IDEAL_GLM)
    assert g.nvar == 9
    g.close()


@pytest.mark.parametrize("seed", range(8))
def test_glm_random_shapes_and_options(ag, seed):
    """Seeded sweep for the 9-variable GLM path: ragged 2-D and 3-D shapes, both solvers, every limiter and RK scheme,
    periodic and open ends, default and forced work splits -- 3 steps against the oracle."""
    import workloads
    rng = np.random.default_rng(7000 + seed)
    ndim = int(rng.choice([2, 3]))
    nx, ny = int(rng.choice([29, 31, 33, 61, 64])), int(rng.choice([5, 11, 12, 23]))
    nz = int(rng.choice([4, 9, 17])) if ndim == 3 else 1
    riemann = int(rng.choice([oracle.HLL, oracle.HLLD]))
    limiter, beta = [(0, 1.0), (1, 1.0), (2, 1.0), (2, 1.3)][int(rng.integers(4))]
    rk = int(rng.choice([1, 2, 3, 4, 5]))
    bc = tuple(int(b) for b in rng.integers(0, 2, 3))
    sg = int(rng.choice([1, 5, 40])) if rng.random() < 0.5 else 0
    W, U8 = workloads.random_state(300 + seed, (nx, ny, nz), ndim, amp=0.3)
    U = np.concatenate([U8, 0.05 * rng.standard_normal((1,) + U8.shape[1:])], axis=0)
    kw = dict(shape=(nx, ny, nz), dx=(1.0 / nx, 1.3 / ny, 0.7 / nz if ndim == 3 else 1.0), ndim=ndim, riemann=riemann,
              limiter=limiter, beta=beta, rk=rk, bc=bc)
    ref = oracle.RefSolver(eqset=oracle.IDEAL_GLM, **kw); gpu = ag.Agate(eqset=ag.IDEAL_GLM, stage_grid=sg, **kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(3):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr, (kw, s)
        ref.step(0.5 * dtr); gpu.step(0.5 * dtr)
        e = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
        assert np.all(e <= 1e-11), (kw, s, e)
    ref.close(); gpu.close()


# ---- Hall MHD with the GLM scalar (eqset HALL_GLM, R29): strip kernel, 1-D and 2-D grids ------------------------------
@pytest.mark.parametrize("n,grid,rk", [(64, 0, 2), (100, 0, 2), (100, 37, 3), (64, 5, 5)])
def test_hall_glm_2d_parity(ag, n, grid, rk):
    """Config 4's recipe (2-D Hall, d_i across 51 zones, whistler-limited dt) with a live cleaning field."""
    wl = make_workload(4, n=n)
    x = (np.arange(n) + 0.5) / n
    U = np.concatenate([wl.U, (0.01 * np.sin(2 * np.pi * x)[None, :] * np.cos(4 * np.pi * x)[:, None])[None, None]], axis=0)
    U[5] += 0.02 * np.exp(-((x[None, None, :] - 0.5) ** 2 + (x[None, :, None] - 0.4) ** 2) / 0.01)   # a divergence error
    U[4] = wl.U[4] + 0.5 * (U[5] ** 2 - wl.U[5] ** 2)
    kw = dict(shape=wl.shape, dx=wl.dx, ndim=2, gamma=wl.gamma, riemann=oracle.HLL, limiter=2, beta=1.3, rk=rk, cfl=wl.cfl,
              d_i=wl.d_i)
    ref = oracle.RefSolver(eqset=oracle.HALL_GLM, **kw); ref.set_state(U)
    gpu = ag.Agate(eqset=ag.HALL_GLM, stage_grid=grid, **kw); gpu.set_state(U)
    e1 = None
    for s in range(6):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr)
        assert gpu.step(0.0) == dtg
        if s == 0:
            e1 = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    eN = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    tr, tg = ref.advance(3), gpu.advance(3)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch()) <= TOL_N)
    ref.close(); gpu.close()


def test_hall_glm_1d_and_rejections(ag):
    import workloads
    n = 80
    x = (np.arange(n) + 0.5) / n
    W = np.zeros((8, 1, 1, n))
    W[0] = 1.0 + 0.3 * np.sin(2 * np.pi * x); W[1] = 0.2; W[4] = 0.7
    W[5] = 0.8 + 0.05 * np.sin(4 * np.pi * x)
    W[6, 0, 0], W[7, 0, 0] = 0.3 * np.cos(2 * np.pi * x), 0.3 * np.sin(4 * np.pi * x)
    U = np.concatenate([workloads.prim_to_cons(W, 5 / 3), 0.01 * np.sin(2 * np.pi * x)[None, None, None, :]], axis=0)
    kw = dict(shape=(n, 1, 1), dx=(1.0 / n, 1, 1), ndim=1, riemann=oracle.HLL, beta=1.3, d_i=0.05)
    ref = oracle.RefSolver(eqset=oracle.HALL_GLM, **kw); gpu = ag.Agate(eqset=ag.HALL_GLM, **kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(6):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr); gpu.step(0.0)
    assert np.all(rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch()) <= TOL_N)
    ref.close(); gpu.close()
    with pytest.raises(ag.AgateError):
        ag.Agate(eqset=ag.HALL_GLM, shape=(8, 8, 1), dx=(1, 1, 1), ndim=2, riemann=1)          # Hall + HLLD


@pytest.mark.parametrize("grid,rk", [(0, 2), (23, 3)])
def test_hall_glm_3d_parity(ag, grid, rk):
    """Hall + GLM through the 3-D row-owner kernel (nine variables, three halo-row planes, bulk row copies): config 8's
    recipe at 40^3 (ragged tiles) with a smooth psi and a divergence error in B_x."""
    wl = make_workload(8, n=40)
    n = 40
    x = (np.arange(n) + 0.5) / n
    U = np.empty((9, n, n, n))
    U[:8] = wl.U
    U[5] += 0.02 * np.exp(-((x[None, None, :] - 0.5) ** 2 + (x[None, :, None] - 0.4) ** 2 + (x[:, None, None] - 0.6) ** 2) / 0.02)
    U[4] = wl.U[4] + 0.5 * (U[5] ** 2 - wl.U[5] ** 2)
    U[8] = 0.01 * np.sin(2 * np.pi * x)[None, None, :] * np.cos(2 * np.pi * x)[:, None, None]
    kw = dict(shape=wl.shape, dx=wl.dx, ndim=3, gamma=wl.gamma, riemann=oracle.HLL, limiter=2, beta=1.3, rk=rk, cfl=wl.cfl,
              d_i=wl.d_i)
    ref = oracle.RefSolver(eqset=oracle.HALL_GLM, **kw); ref.set_state(U)
    gpu = ag.Agate(eqset=ag.HALL_GLM, stage_grid=grid, **kw); gpu.set_state(U)
    e1 = None
    for s in range(4):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr)
        assert gpu.step(0.0) == dtg
        if s == 0:
            e1 = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    eN = rel_linf9(gpu.get_state(), ref.get_state(), ref.glm_ch())
    assert np.all(e1 <= TOL_1), e1
    assert np.all(eN <= TOL_N), eN
    ref.close(); gpu.close()
