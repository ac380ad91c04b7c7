"""A8 on 3-D grids (-m gpu): Hall MHD through the row-owner kernel (face current with all three transverse
differences, whistler-limited fused Courant reduction) against the oracle, same metric and bars as the other parity
tests; forced work splits reach every segment prologue; the halo rows' x corners, the third halo-row buffer and the
extra hand-overs are what this variant adds."""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import TOL_1, TOL_DT, TOL_N, assert_parity, rel_linf, run_pair
from workloads import HALL, HLL, make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("n,grid", [(40, 0), (40, 1), (40, 7), (40, 37), (40, 160), (72, 0)])
def test_config8_reduced(ag, n, grid):
    """Config 8 recipe (config 3's 3-D state, Hall, HLL, eq.4 at beta = 1, d_i across 51 zones); n = 40: ragged in x
    (32 + 8) and y (3 x 11 + 7)."""
    wl = make_workload(8, n=n)
    assert_parity(*run_pair(ag, wl, 5 if n == 40 else 2, gpu_kw=dict(stage_grid=grid)))


@pytest.mark.parametrize("over", [dict(rk=3), dict(rk=5, beta=1.3), dict(limiter=1), dict(bc=(1, 0, 1)), dict(bc=(0, 2, 0)),
                                  dict(rk=1, limiter=0)])
def test_options_3d_hall(ag, over):
    wl = make_workload(8, n=36)
    assert_parity(*run_pair(ag, wl, 3, **over))


def test_2d_problem_embedded_in_3d(ag):
    """Config 4's 2-D state copied along z: the 3-D Hall path must reproduce the 2-D strip kernel's run (different
    kernels, same formulas: agreement at round-off, z components of the update included)."""
    wl = make_workload(4, n=48)
    nz = 6
    g2 = ag.Agate.from_workload(wl)
    U3 = np.ascontiguousarray(np.repeat(wl.U, nz, axis=1))
    g3 = ag.Agate(shape=(48, 48, nz), dx=(wl.dx[0], wl.dx[1], wl.dx[0]), ndim=3, gamma=wl.gamma, eqset=HALL, riemann=HLL,
                  limiter=2, beta=wl.beta, rk=2, cfl=wl.cfl, d_i=wl.d_i)
    g3.set_state(U3)
    for s in range(5):
        dt = g2.compute_dt()
        assert abs(g3.compute_dt() - dt) <= TOL_DT * dt
        g2.step(dt); g3.step(dt)
    A, B = g2.get_state(), g3.get_state()
    for k in range(nz):
        assert np.all(rel_linf(B[:, k:k + 1], A) <= 1e-12), k
    g2.close(); g3.close()


@pytest.mark.parametrize("seed", range(8))
def test_random_shapes_3d_hall(ag, seed):
    rng = np.random.default_rng(5000 + seed)
    nx = int(rng.choice([5, 31, 32, 33, 64, 70])); ny = int(rng.choice([3, 10, 11, 12, 23])); nz = int(rng.choice([3, 7, 16]))
    limiter, beta = [(0, 1.0), (1, 1.0), (2, 1.0), (2, 1.3)][int(rng.integers(4))]
    rk = int(rng.choice([1, 2, 3, 4, 5]))
    bc = [int(b) for b in rng.integers(0, 2, 3)]
    if bc[0] == 0 and rng.random() < 0.3:
        bc[1] = 2
    sg = int(rng.choice([1, 3, 17, 80])) if rng.random() < 0.5 else 0
    W, U = workloads.random_state(700 + seed, (nx, ny, nz), 3, amp=0.3)
    kw = dict(shape=(nx, ny, nz), dx=(1.0 / nx, 1.3 / ny, 0.7 / nz), ndim=3, riemann=HLL, limiter=limiter, beta=beta, rk=rk,
              bc=tuple(bc), eqset=HALL, d_i=0.03)
    ref = oracle.RefSolver(**kw); gpu = ag.Agate(stage_grid=sg, **kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(3):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr, (kw, s)
        ref.step(0.5 * dtr); gpu.step(0.5 * dtr)
        e = rel_linf(gpu.get_state(), ref.get_state())
        assert np.all(e <= 1e-11), (kw, s, e)
    ref.close(); gpu.close()


def test_z_slabs_3d_hall(ag):
    """NEXT-4 with Hall: the halo planes travel with their x / y ghosts, so the edge and corner values the face
    current needs arrive with them."""
    from test_gpu_slab import run_slabs
    wl = make_workload(8, n=40)
    kw = dict(shape=wl.shape, dx=wl.dx, ndim=3, gamma=wl.gamma, riemann=HLL, limiter=2, beta=wl.beta, rk=2, cfl=wl.cfl,
              d_i=wl.d_i)
    one = ag.Agate(eqset=HALL, **kw)
    one.set_state(wl.U)
    t1 = one.advance(3)
    U1 = one.get_state()
    one.close()
    U2, ts = run_slabs(ag, kw, wl.U, 3, 3, periodic=True, eqset=HALL)
    assert all(t == t1 for t in ts)
    assert np.array_equal(U1.view(np.uint64), U2.view(np.uint64))
