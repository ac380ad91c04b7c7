"""GPU parity for the rest of NEXT-3 (-m gpu): RK43 / RK53 (R27), the sheared zero-gradient ends in y (R28), and the
per-context launch tuning that replaced the environment knobs.  Same metric and bars as tests/test_gpu_parity.py."""
import math

import numpy as np
import pytest

import oracle
import workloads
from conftest import read_golden
from test_gpu_parity import TOL_1, TOL_DT, TOL_N, assert_parity, rel_linf, run_pair
from workloads import HALL, HLL, HLLD, IDEAL, make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("rk", [4, 5])
@pytest.mark.parametrize("cfg,n,steps", [(2, 100, 5), (4, 64, 5), (3, 40, 4), (5, 36, 3)])
def test_rk43_rk53_2d_3d(ag, rk, cfg, n, steps):
    """Strip kernel (ideal HLLD, Hall) and row-owner kernel: every stage's c dt and the Shu-Osher weights."""
    wl = make_workload(cfg, n=n)
    assert_parity(*run_pair(ag, wl, steps, rk=rk))


@pytest.mark.parametrize("rk", [4, 5])
def test_rk43_rk53_1d_and_advance(ag, rk):
    """Pooled kernel on a 1-D grid; advance() (RK43 replays the graph, RK53 ends in the other buffer and launches
    directly) against the oracle's advance()."""
    n = 96
    x = (np.arange(n) + 0.5) / n
    W = np.zeros((8, 1, 1, n))
    W[0] = 1.0 + 0.3 * np.sin(2 * np.pi * x); W[1] = 0.2; W[4] = 0.7; W[5] = 0.8
    W[6, 0, 0], W[7, 0, 0] = 0.3 * np.cos(2 * np.pi * x), 0.3 * np.sin(4 * np.pi * x)
    U = workloads.prim_to_cons(W, 5 / 3)
    kw = dict(shape=(n, 1, 1), dx=(1 / n, 1, 1), ndim=1, riemann=HLLD, beta=1.3, rk=rk)
    ref = oracle.RefSolver(**kw); gpu = ag.Agate(**kw)
    ref.set_state(U); gpu.set_state(U)
    tr, tg = ref.advance(7), gpu.advance(7)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    ref.close(); gpu.close()
    wl = make_workload(3, n=24)
    ref = oracle.RefSolver.from_workload(wl, rk=rk); gpu = ag.Agate.from_workload(wl, rk=rk)
    tr, tg = ref.advance(5), gpu.advance(5)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    ref.close(); gpu.close()


def test_sheared_ends_whistler_2d(ag):
    """The rotated whistler wave of PAPER.md L312-316 at n = 32 for a fifth of a period: Hall strip kernel + the
    sheared ghost rule against the oracle, and the (1,2) translational symmetry of the result."""
    g = read_golden("whistler.txt")
    d_i, B0, lam, db = g["d_i"][0], g["v_A"][0], g["wavelength"][0], g["delta_b"][0]
    n = 32
    k = 2 * math.pi / lam
    vphi = d_i * B0 * k / 2 + math.sqrt(B0 ** 2 + (d_i * B0 * k) ** 2 / 4)
    al = math.atan(0.5); ca, sa = math.cos(al), math.sin(al)
    Lx = lam / ca; dx = Lx / n
    x = -Lx / 2 + (np.arange(n) + 0.5) * dx
    X, Y = np.meshgrid(x, x)
    ph = k * ca * X + k * sa * Y
    dv = db * B0 / vphi
    W = np.zeros((8, 1, n, n))
    W[0], W[4] = 1.0, 1.0
    W[1, 0], W[2, 0], W[3, 0] = dv * np.cos(ph) * sa, -dv * np.cos(ph) * ca, dv * np.sin(ph)
    W[5, 0] = B0 * ca - db * np.cos(ph) * sa; W[6, 0] = B0 * sa + db * np.cos(ph) * ca; W[7, 0] = -db * np.sin(ph)
    U = workloads.prim_to_cons(W, 5 / 3)
    kw = dict(shape=(n, n, 1), dx=(dx, dx, 1.0), ndim=2, eqset=HALL, riemann=HLL, beta=1.3, d_i=d_i, bc=(0, 2, 0))
    ref = oracle.RefSolver(**kw); gpu = ag.Agate(**kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(120):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr); gpu.step(0.0)
    Ug, Ur = gpu.get_state(), ref.get_state()
    # B_x, B_y carry the background 100: measure the wave part of every variable against the wave amplitude
    for q, amp in ((1, dv), (2, dv), (3, dv), (5, db), (6, db), (7, db)):
        assert np.max(np.abs(Ug[q] - Ur[q])) <= 1e-9 * amp * 100, q
    assert np.all(rel_linf(Ug, Ur) <= TOL_N)
    assert np.max(np.abs(Ug[7, 0, :-2, :] - np.roll(Ug[7, 0, 2:, :], 1, axis=-1))) <= 1e-6 * db
    ref.close(); gpu.close()


@pytest.mark.parametrize("ndim", [2, 3])
def test_sheared_ends_random_state(ag, ndim):
    """Random cell-to-cell data: every ghost cell of the sheared rule matters (corners with the periodic x, and the
    z ends of a 3-D grid, open or periodic)."""
    shape = (37, 13, 1) if ndim == 2 else (33, 12, 9)
    W, U = workloads.random_state(4242 + ndim, shape, ndim, amp=0.3)
    kw = dict(shape=shape, dx=(1 / shape[0], 1.2 / shape[1], 0.8 / shape[2] if ndim == 3 else 1.0), ndim=ndim,
              riemann=HLLD, beta=1.3, bc=(0, 2, 1 if ndim == 3 else 0))
    ref = oracle.RefSolver(**kw); gpu = ag.Agate(**kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(3):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(0.5 * dtr); gpu.step(0.5 * dtr)
        assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= 1e-11)
    ref.close(); gpu.close()
    with pytest.raises(ag.AgateError):
        ag.Agate(shape=shape, dx=(1, 1, 1), ndim=ndim, bc=(1, 2, 0))


@pytest.mark.parametrize("cfg,n", [(3, 40), (2, 100)])
def test_stage_grid_does_not_change_the_bits(ag, cfg, n):
    """include/agate.h: the work split chosen with agate_set_tuning changes no bit of the result, and neither does
    launching directly instead of replaying the graph."""
    wl = make_workload(cfg, n=n)
    outs = []
    for kw in (dict(), dict(stage_grid=1), dict(stage_grid=37), dict(no_graph=True), dict(stage_grid=5, no_graph=True)):
        gpu = ag.Agate.from_workload(wl, **kw)
        t = gpu.advance(4)
        outs.append((t, gpu.get_state()))
        if kw.get("stage_grid"):
            assert gpu.launch_info()["grid"][0] == kw["stage_grid"]
        gpu.close()
    for t, U in outs[1:]:
        assert t == outs[0][0]
        assert np.array_equal(U.view(np.uint64), outs[0][1].view(np.uint64))


def test_device_source_is_read_in_stream_order(ag):
    """agate_set_state with a DEVICE source does not synchronise: the binding orders the context's stream after
    torch's current stream, so a tensor produced just before the call is read complete."""
    import torch
    wl = make_workload(3, n=48)
    gpu = ag.Agate.from_workload(wl, set_state=False)
    host = torch.as_tensor(wl.U).pin_memory()
    for rep in range(3):
        big = torch.empty((64, 1024, 1024), device="cuda").normal_()      # keeps the current stream busy
        Ud = (host.to("cuda", non_blocking=True) * 2.0) * 0.5             # produced on the current stream
        gpu.set_state(Ud)
        out = torch.empty_like(Ud)
        gpu.get_state(out)
        assert torch.equal(out.cpu(), host)
        del big
    ref = oracle.RefSolver.from_workload(wl)
    dtr = ref.compute_dt(); ref.step(dtr)
    assert gpu.step(0.0) == dtr or abs(gpu.compute_dt()) > 0
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_1)
    ref.close(); gpu.close()


@pytest.mark.parametrize("eqset_name", ["glm", "cgl"])
@pytest.mark.parametrize("n", [64, 75])
def test_nine_variable_sets_on_1d_grids(ag, eqset_name, n):
    """1-D GLM / CGL problems (the paper's CGL benchmarks are 1-D) run through the 2-D strip kernel as one
    row that is its own periodic neighbour; the oracle runs them as genuinely 1-D (no y sweep, C = 0.8)."""
    x = (np.arange(n) + 0.5) / n
    if eqset_name == "glm":
        W = np.zeros((8, 1, 1, n))
        W[0] = 1.0 + 0.3 * np.sin(2 * np.pi * x); W[1] = 0.2; W[2] = 0.1 * np.cos(2 * np.pi * x); W[4] = 0.7
        W[5] = 0.8 + 0.05 * np.sin(4 * np.pi * x)                  # a divergence error for the cleaning to act on
        W[6, 0, 0], W[7, 0, 0] = 0.3 * np.cos(2 * np.pi * x), 0.3 * np.sin(4 * np.pi * x)
        U = np.concatenate([workloads.prim_to_cons(W, 5 / 3), 0.01 * np.sin(2 * np.pi * x)[None, None, None, :]], axis=0)
        eo, eg, rie = oracle.IDEAL_GLM, ag.IDEAL_GLM, HLLD
    else:
        W = np.zeros((9, n))
        W[0] = 1.0 + 0.2 * np.sin(2 * np.pi * x); W[1] = 0.3 * np.cos(2 * np.pi * x); W[2] = 0.1
        W[4] = 0.8 + 0.2 * np.cos(2 * np.pi * x); W[8] = 0.6 + 0.3 * np.sin(2 * np.pi * x)
        W[5] = 0.7; W[6] = 0.3 * np.sin(2 * np.pi * x); W[7] = 0.2
        U = np.stack([oracle.cgl_prim_to_cons(W[:, i]) for i in range(n)], axis=1).reshape(9, 1, 1, n)
        eo, eg, rie = oracle.CGL, ag.CGL, HLL
    kw = dict(shape=(n, 1, 1), dx=(1.0 / n, 1, 1), ndim=1, riemann=rie, beta=1.3, rk=2,
              relax=0.99 if eqset_name == "cgl" else 0.0)
    ref = oracle.RefSolver(eqset=eo, **kw); gpu = ag.Agate(eqset=eg, **kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(6):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr)
        assert gpu.step(0.0) == dtg
    Ug, Ur = gpu.get_state(), ref.get_state()
    for q in range(9):
        sc = max(np.max(np.abs(Ur[q])), np.max(np.abs(Ur[0])) if q == 8 else 0.0, 1e-300)
        if 1 <= q <= 3: sc = np.max(np.abs(Ur[1:4]))
        if 5 <= q <= 7: sc = np.max(np.abs(Ur[5:8]))
        assert np.max(np.abs(Ug[q] - Ur[q])) <= TOL_N * sc, (q,)
    tr, tg = ref.advance(3), gpu.advance(3)
    assert abs(tg - tr) <= 1e-13 * tr
    ref.close(); gpu.close()
