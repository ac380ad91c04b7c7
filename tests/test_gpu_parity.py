"""GPU parity tests: the CUDA path (through the C-ABI, via the thin binding) against the CPU oracle, element by
element on the same seeded inputs.  Run on the B200 box with  pytest -m gpu.

Tolerances (BASELINE.json north_star): relative L-inf per conserved variable <= 1e-12 after one
step and <= 1e-9 after the config's step count; dt identical to 1e-14 relative at every step.  The scale of a
momentum / magnetic component is the largest |component| over all three components of that vector, so a component
that is identically zero must also be exactly zero on the GPU.
"""
import os

import numpy as np
import pytest

import oracle
from workloads import HALL, HLL, HLLD, IDEAL, make_workload, random_state

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12
TOL_N = 1e-9
TOL_DT = 1e-14


@pytest.fixture(scope="module")
def ag():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the CUDA path has no CPU fallback")
    import paper_2503_20899_b200 as m
    m.lib()          # raises if the extension cannot be built/loaded
    return m


def rel_linf(Ug, Ur):
    """R19 metric: per-variable max |diff| / scale, vector components share the scale of their vector."""
    err = np.empty(8)
    sc = np.empty(8)
    sc[0] = np.max(np.abs(Ur[0])); sc[4] = np.max(np.abs(Ur[4]))
    sc[1:4] = np.max(np.abs(Ur[1:4])); sc[5:8] = np.max(np.abs(Ur[5:8]))
    for q in range(8):
        d = np.max(np.abs(Ug[q] - Ur[q]))
        err[q] = d / sc[q] if sc[q] > 0 else (0.0 if d == 0 else np.inf)     # R19: exact zeros stay exact zeros
    return err


def run_pair(ag, wl, n_steps, check_each=True, gpu_kw=None, **over):
    """Advance the oracle and the GPU side by side; returns (err after step 1, err after n_steps, worst dt err)."""
    ref = oracle.RefSolver.from_workload(wl, **over)
    gpu = ag.Agate.from_workload(wl, **over, **(gpu_kw or {}))      # gpu_kw: launch tuning (stage_grid)
    worst_dt, e1 = 0.0, None
    for s in range(n_steps):
        dtr = ref.compute_dt()
        dtg = gpu.compute_dt()
        worst_dt = max(worst_dt, abs(dtg - dtr) / dtr)
        ref.step(dtr)
        used = gpu.step(0.0)                       # device-resident dt of the reduction
        assert used == dtg
        if s == 0:
            e1 = rel_linf(gpu.get_state(), ref.get_state())
    eN = rel_linf(gpu.get_state(), ref.get_state())
    ref.close(); gpu.close()
    return e1, eN, worst_dt


def assert_parity(e1, eN, edt):
    assert edt <= TOL_DT, f"dt mismatch {edt}"
    assert np.all(e1 <= TOL_1), f"1-step rel L-inf {e1}"
    assert np.all(eN <= TOL_N), f"n-step rel L-inf {eN}"


# ---- device Riemann solvers against the oracle's, pair by pair ---------------------------------------------
@pytest.mark.parametrize("riemann", [HLL, HLLD])
def test_device_face_flux(ag, riemann):
    rng = np.random.default_rng(11 + riemann)
    n = 20000
    WL = np.empty((8, n)); WR = np.empty((8, n))
    for W in (WL, WR):
        W[0] = 0.2 + 2 * rng.random(n); W[4] = 0.1 + 2 * rng.random(n)
        amp = np.array([0.1, 0.5, 2.0, 6.0])[np.arange(n) % 4]
        for q in (1, 2, 3, 5, 6, 7):
            W[q] = amp * (2 * rng.random(n) - 1)
    WR[:, ::7] = WL[:, ::7] * (1 + 1e-3 * rng.random((8, len(range(0, n, 7)))))     # near-smooth pairs
    WR[:, ::11] = WL[:, ::11]                                                         # identical pairs
    WL[6:8, ::13] = 0.0; WR[6:8, ::13] = 0.0                                          # B_t = 0 (degenerate guard)
    g = 5.0 / 3.0
    for d in range(3):
        Fg = ag.test_face_flux(IDEAL, riemann, d, g, WL, WR)
        idx = rng.choice(n, 1500, replace=False)
        idx = np.concatenate([idx, np.arange(0, n, 91)])
        for i in idx:
            Fo = oracle.face_flux(riemann, d, g, WL[:, i], WR[:, i])
            sc = max(np.max(np.abs(Fo)), 1e-300)
            assert np.max(np.abs(Fg[:, i] - Fo)) <= 5e-13 * sc, (d, i, Fg[:, i], Fo)


def test_device_face_flux_hall(ag):
    rng = np.random.default_rng(5)
    n = 4000
    WL = np.empty((8, n)); WR = np.empty((8, n))
    for W in (WL, WR):
        W[0] = 0.2 + 2 * rng.random(n); W[4] = 0.1 + 2 * rng.random(n)
        for q in (1, 2, 3, 5, 6, 7):
            W[q] = 0.5 * (2 * rng.random(n) - 1)
    J = 3.0 * (2 * rng.random((3, n)) - 1)
    g = 5.0 / 3.0
    for d in range(3):
        Fg = ag.test_face_flux(HALL, HLL, d, g, WL, WR, J=J, d_i=0.05, dxmin=1 / 128)
        for i in range(0, n, 7):
            Fo = oracle.face_flux(HLL, d, g, WL[:, i], WR[:, i], eqset=HALL, d_i=0.05, dxmin=1 / 128, J=J[:, i])
            assert np.max(np.abs(Fg[:, i] - Fo)) <= 5e-13 * np.max(np.abs(Fo))


# ---- the five configs (BASELINE.json); reduced sizes span several tiles and a ragged tail ------------------
def test_config1_full(ag):
    """Config 1 at its full size and step count: 2D ideal 128^2, HLL, minmod, 10 steps."""
    wl = make_workload(1)
    assert_parity(*run_pair(ag, wl, wl.n_steps))


@pytest.mark.parametrize("n,steps,grid", [(100, 12, 0), (256, 4, 0), (100, 4, 1), (100, 4, 5), (100, 4, 40)])
def test_config2_reduced(ag, n, steps, grid):
    """Config 2 recipe (2D HLLD, beta=1.3, shear layer) through the strip kernel.  n=100: 3 full 30-column strips + a
    ragged one of 10.  `grid` CTAs of 6 warps share the (strip, row) pairs evenly: 1 = 16-17 rows per warp, segments
    that cross from one strip into the next; 5 / 40 = ever shorter segments (40: one or two rows each, every row
    through the segment prologue and the closing step); 0 = the library's own choice."""
    wl = make_workload(2, n=n)
    assert_parity(*run_pair(ag, wl, steps, gpu_kw=dict(stage_grid=grid)))


@pytest.mark.parametrize("n,grid", [(40, 0), (40, 1), (40, 7), (40, 37), (40, 160), (72, 0)])
def test_config3_reduced(ag, n, grid):
    """Config 3 recipe (3D HLLD) through the row-owner kernel.  n=40: ragged in x (32+8) and y (3*11+7).  The work
    (tile-planes) is split evenly over `grid` CTAs: 1 = every tile a whole segment of one CTA, 7 / 37 = segments that
    start and end in the middle of a tile column, 160 = one or two planes per segment (every plane through the segment
    prologue and the closing step), 0 = the library's own choice."""
    wl = make_workload(3, n=n)
    assert_parity(*run_pair(ag, wl, 5 if n == 40 else 2, gpu_kw=dict(stage_grid=grid)))


@pytest.mark.parametrize("n", [64, 100])
def test_config4_reduced(ag, n):
    """Config 4 recipe (2D Hall, HLL with Hall electric field, whistler-limited dt); d_i/dx kept at 51.2 cells."""
    wl = make_workload(4, n=n)
    assert_parity(*run_pair(ag, wl, 10))


def test_config5_reduced(ag):
    wl = make_workload(5, n=48)
    assert_parity(*run_pair(ag, wl, 4))


def test_advance_matches_oracle_advance(ag):
    """agate_advance (CUDA graph, device-resident dt, no host sync) against the oracle's advance: state and t."""
    wl = make_workload(2, n=128)
    ref = oracle.RefSolver.from_workload(wl)
    gpu = ag.Agate.from_workload(wl)
    tr = ref.advance(20)
    tg = gpu.advance(20)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    assert abs(gpu.t - tr) <= 1e-13 * tr


@pytest.mark.parametrize("rk", [1, 2, 3])
def test_fused_dt_sequences_3d(ag, rk):
    """3-D path: the Courant reduction of step n+1 runs inside the last stage of step n (A7 fused).  Every way into a
    step must see the right v_max: after set_state (stand-alone reduction), after a self-timed step (fused), after a
    step with a host-chosen dt (fused, restarted from zero), inside agate_advance (graph replay), after a second
    set_state (stale value dropped).  dt and t against the oracle at every point."""
    wl = make_workload(3, n=40)
    ref = oracle.RefSolver.from_workload(wl, rk=rk)
    gpu = ag.Agate.from_workload(wl, rk=rk)

    def same_dt():
        dr, dg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dg - dr) <= TOL_DT * dr
        return dr

    d = same_dt()
    ref.step(d); assert abs(gpu.step(0.0) - d) <= TOL_DT * d              # stand-alone reduction feeds step 1
    d = same_dt()
    ref.step(d); assert abs(gpu.step(0.0) - d) <= TOL_DT * d              # fused reduction of step 1 feeds step 2
    ref.step(0.4 * d); assert gpu.step(0.4 * d) == 0.4 * d                # host-chosen dt
    d = same_dt()
    ref.step(d); assert abs(gpu.step(0.0) - d) <= TOL_DT * d              # fused reduction after a host-chosen dt
    tr = ref.advance(3); tg = gpu.advance(3)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    U0 = wl.U.copy()
    ref.set_state(U0, 0.0); gpu.set_state(U0, 0.0)                        # v_max of the old state must not leak
    tr = ref.advance(2); tg = gpu.advance(2)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    ref.close(); gpu.close()


def test_fused_dt_flags_unphysical_3d(ag):
    """R14 through the fused reduction: a step that drives a cell to negative pressure must be reported by the next
    synchronising call (the stage that stores the value also evaluates its speed)."""
    wl = make_workload(3, n=24)
    gpu = ag.Agate.from_workload(wl)
    d = gpu.compute_dt()
    gpu.step(400.0 * d, sync=False)            # far beyond the Courant limit
    with pytest.raises(ag.AgateError) as ei:
        gpu.poll()
        gpu.step(0.0)
    assert ei.value.code == ag.ERR_UNPHYSICAL
    gpu.close()


def test_3d_run_to_run_bitwise(ag):
    """The 3-D kernel hands data between warps through phase counters instead of CTA barriers; a lost ordering would
    show up as run-to-run differences.  Same input, same launch configuration, 8 steps, three runs: bitwise equal
    (dt included), on a grid with ragged tiles and several segments per CTA."""
    wl = make_workload(5, n=72)
    outs = []
    for _ in range(3):
        gpu = ag.Agate.from_workload(wl)
        t = gpu.advance(8)
        outs.append((t, gpu.get_state()))
        gpu.close()
    for t, U in outs[1:]:
        assert t == outs[0][0]
        assert np.array_equal(U, outs[0][1])


@pytest.mark.parametrize("cfg,n", [(2, 100), (4, 64), (1, 32)])
def test_ssp_rk33_2d(ag, cfg, n):
    """SSP-RK33 (NEXT-3, R25) through the 2-D strip kernel (ideal HLLD, Hall HLL) -- three stages, third state copy,
    weights (3/4, 1/4) and (1/3, 2/3), A7 fused into the third stage."""
    wl = make_workload(cfg, n=n)
    assert_parity(*run_pair(ag, wl, 6, rk=3))
    ref = oracle.RefSolver.from_workload(wl, rk=3)
    gpu = ag.Agate.from_workload(wl, rk=3)
    tr, tg = ref.advance(5), gpu.advance(5)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    assert gpu.launch_info()["launches_per_step"] == 7
    ref.close(); gpu.close()


def test_ssp_rk33_1d_pooled_kernel(ag):
    wl = make_workload(1, n=32)
    U = wl.U[:, :, :1, :].copy()
    kw = dict(shape=(32, 1, 1), dx=(1 / 32, 1, 1), ndim=1, riemann=HLLD, beta=1.3, rk=3)
    ref = oracle.RefSolver(**kw); gpu = ag.Agate(**kw)
    ref.set_state(U); gpu.set_state(U)
    tr, tg = ref.advance(8), gpu.advance(8)
    assert abs(tg - tr) <= 1e-13 * tr
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    ref.close(); gpu.close()


# ---- solver options and edge cases --------------------------------------------------------------------------
@pytest.mark.parametrize("riemann", [HLL, HLLD])
@pytest.mark.parametrize("limiter,beta", [(0, 1.0), (1, 1.0), (2, 1.0), (2, 2.0)])
@pytest.mark.parametrize("rk", [1, 2, 3])
def test_options_3d(ag, riemann, limiter, beta, rk):
    W, U = random_state(21, (20, 14, 9), 3, amp=0.3)
    dx = (1 / 20, 1 / 14, 1 / 9)
    kw = dict(shape=(20, 14, 9), dx=dx, ndim=3, riemann=riemann, limiter=limiter, beta=beta, rk=rk, cfl=0.2)
    ref = oracle.RefSolver(**kw); ref.set_state(U)
    gpu = ag.Agate(**kw); gpu.set_state(U)
    for s in range(3):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr); gpu.step(dtr)
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= 1e-11)


@pytest.mark.parametrize("shape,ndim", [((4, 4, 1), 2), ((4, 4, 4), 3), ((1, 1, 1), 1), ((3, 1, 1), 1),
                                        ((37, 1, 1), 1), ((33, 7, 1), 2), ((2, 5, 3), 3), ((65, 13, 5), 3)])
@pytest.mark.parametrize("riemann", [HLL, HLLD])
def test_tiny_and_ragged_grids(ag, shape, ndim, riemann):
    W, U = random_state(sum(shape), shape, ndim, amp=0.3)
    dx = tuple(1.0 / s for s in shape)
    kw = dict(shape=shape, dx=dx, ndim=ndim, riemann=riemann, limiter=2, beta=1.3, rk=2, cfl=0.2)
    ref = oracle.RefSolver(**kw); ref.set_state(U)
    gpu = ag.Agate(**kw); gpu.set_state(U)
    for s in range(2):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr); gpu.step(dtr)
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= 1e-11)


def test_hall_1d_and_options(ag):
    W, U = random_state(3, (48, 1, 1), 1, amp=0.2)
    kw = dict(shape=(48, 1, 1), dx=(1 / 48, 1.0, 1.0), ndim=1, eqset=HALL, riemann=HLL, limiter=2, beta=1.3, rk=2,
              cfl=0.3, d_i=0.3)
    ref = oracle.RefSolver(**kw); ref.set_state(U)
    gpu = ag.Agate(**kw); gpu.set_state(U)
    for s in range(5):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr); gpu.step(dtr)
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= 1e-11)


@pytest.mark.parametrize("riemann", [HLL, HLLD])
def test_uniform_state_is_bitwise_fixed(ag, riemann):
    """P1 on the GPU, incl. the HLLD-degenerate state B=(B0,0,0), B0^2/rho > gamma p/rho."""
    for Wc in ([1.0, 0.3, -0.2, 0.1, 0.6, 0.7, 0.2, -0.3], [1.0, 0.1, 0.0, 0.0, 0.1, 1.0, 0.0, 0.0]):
        shape = (40, 16, 6)
        W = np.empty((8,) + shape[::-1]); W[:] = np.array(Wc)[:, None, None, None]
        from workloads import prim_to_cons
        U = prim_to_cons(W, 5.0 / 3.0)
        gpu = ag.Agate(shape=shape, dx=(1 / 40, 1 / 16, 1 / 6), ndim=3, riemann=riemann, beta=1.3)
        gpu.set_state(U)
        gpu.advance(5)
        assert np.array_equal(gpu.get_state(), U)


def test_conservation_on_gpu(ag):
    """P2 on the GPU: periodic => sums of all 8 variables conserved to round-off."""
    wl = make_workload(3, n=36)
    gpu = ag.Agate.from_workload(wl)
    s0 = wl.U.reshape(8, -1).sum(axis=1)
    gpu.advance(10)
    s1 = gpu.get_state().reshape(8, -1).sum(axis=1)
    scale = np.abs(wl.U).reshape(8, -1).sum(axis=1)
    assert np.all(np.abs(s1 - s0) <= 1e-13 * scale)


def test_unphysical_state_is_flagged(ag):
    wl = make_workload(1, n=32)
    U = wl.U.copy(); U[0, 0, 5, 7] = -1.0
    gpu = ag.Agate.from_workload(wl, set_state=False)
    gpu.set_state(U)
    with pytest.raises(ag.AgateError) as ei:
        gpu.compute_dt()
    assert ei.value.code == ag.ERR_UNPHYSICAL
    gpu.set_state(wl.U)                 # a fresh state clears the flag
    assert gpu.compute_dt() > 0


def test_device_resident_state_roundtrip(ag):
    import torch
    wl = make_workload(1, n=64)
    gpu = ag.Agate.from_workload(wl, set_state=False)
    Ud = torch.as_tensor(wl.U, device="cuda")
    gpu.set_state(Ud)
    out = torch.empty_like(Ud)
    gpu.get_state(out)
    gpu.poll()
    assert torch.equal(out, Ud)
    assert np.array_equal(gpu.get_state(), wl.U)


def test_call_order_and_bad_args(ag):
    wl = make_workload(1, n=32)
    gpu = ag.Agate.from_workload(wl, set_state=False)
    with pytest.raises(ag.AgateError) as ei:
        gpu.compute_dt()
    assert ei.value.code == ag.ERR_STATE
    with pytest.raises(ag.AgateError):
        ag.Agate(shape=(32, 32, 1), dx=(1, 1, 1), ndim=2, eqset=HALL, riemann=HLLD)


# ---- NEXT-3 (R26): zero-gradient / open boundaries ------------------------------------------------------------
@pytest.mark.parametrize("riemann", [HLL, HLLD])
def test_open_boundaries_brio_wu(ag, riemann):
    """The paper's Brio-Wu tube (gamma = 2) as four identical rows, open in x and periodic in y, run until
    the fast waves have left through both ends: GPU against the oracle, ghost rule included."""
    n = 128
    x = (np.arange(n) + 0.5) / n
    W = np.zeros((8, 1, 4, n))
    left = (x < 0.5)[None, None, :]
    W[0] = np.where(left, 1.0, 0.125); W[4] = np.where(left, 1.0, 0.1); W[5] = 0.75; W[6] = np.where(left, 1.0, -1.0)
    import workloads
    U = workloads.prim_to_cons(W, 2.0)
    kw = dict(shape=(n, 4, 1), dx=(1 / n, 1 / n, 1), ndim=2, gamma=2.0, riemann=riemann, beta=1.3, bc=(1, 0, 0))
    ref = oracle.RefSolver(**kw); gpu = ag.Agate(**kw)
    ref.set_state(U); gpu.set_state(U)
    tr, tg = ref.advance(450), gpu.advance(450)
    assert abs(tg - tr) <= 1e-12 * tr and tr > 0.3
    assert np.all(rel_linf(gpu.get_state(), ref.get_state()) <= TOL_N)
    assert abs(gpu.get_state()[0].sum() - U[0].sum()) > 1e-3 * U[0].sum()        # mass has left the tube
    ref.close(); gpu.close()


def test_open_boundaries_3d(ag):
    """Open in z and x, periodic in y, on the 3-D kernel (config 3 recipe at 40^3)."""
    wl = make_workload(3, n=40)
    assert_parity(*run_pair(ag, wl, 4, bc=(1, 0, 1)))


# ---- seeded sweep over shapes, options and work splits ----------------------------------------------------------
@pytest.mark.parametrize("seed", range(24))
def test_random_shapes_and_options(ag, seed):
    """Ragged sizes around the tile / strip / segment boundaries (nx around 30, 32, 60, 64; ny around 11, 22; small nz),
    every solver option, periodic and open ends, default and forced work splits -- 3 steps against the oracle."""
    rng = np.random.default_rng(9000 + seed)
    ndim = int(rng.choice([2, 3]))
    nx = int(rng.choice([5, 29, 30, 31, 32, 33, 59, 61, 64, 65, 70]))
    ny = int(rng.choice([3, 10, 11, 12, 21, 23, 34]))
    nz = int(rng.choice([3, 7, 16, 19])) if ndim == 3 else 1
    hall = ndim == 2 and rng.random() < 0.25
    riemann = HLL if hall else int(rng.choice([HLL, HLLD]))
    limiter, beta = [(0, 1.0), (1, 1.0), (2, 1.0), (2, 1.3), (2, 2.0)][int(rng.integers(5))]
    rk = int(rng.choice([1, 2, 3, 4, 5]))
    bc = [int(b) for b in rng.integers(0, 2, 3)]
    if bc[0] == 0 and rng.random() < 0.4:
        bc[1] = 2                               # sheared zero-gradient ends in y (R28)
    bc = tuple(bc)
    sg = int(rng.choice([1, 3, 17, 80])) if rng.random() < 0.5 else 0
    import workloads
    W, U = workloads.random_state(100 + seed, (nx, ny, nz), ndim, amp=0.3)
    kw = dict(shape=(nx, ny, nz), dx=(1.0 / nx, 1.3 / ny, 0.7 / nz if ndim == 3 else 1.0), ndim=ndim, riemann=riemann,
              limiter=limiter, beta=beta, rk=rk, bc=bc, eqset=(ag.HALL if hall else ag.IDEAL), d_i=(0.02 if hall else 0.0))
    ref = oracle.RefSolver(**kw); gpu = ag.Agate(stage_grid=sg, **kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(3):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr, (kw, s)
        ref.step(0.5 * dtr)                     # random cell-to-cell data: half the Courant step keeps it physical
        gpu.step(0.5 * dtr)
        e = rel_linf(gpu.get_state(), ref.get_state())
        assert np.all(e <= 1e-11), (kw, s, e)
    ref.close(); gpu.close()
