"""The allocation-free entry point agate_cfl_static (include/agate.h; csrc/agate_noalloc.cu) against the existing Courant
reduction of a context (agate_get_vmax / agate_compute_dt)  (-m gpu).

Collected last on purpose (the suite runs with pytest -x).  The entry point keeps its scratch in a static __device__
array that every call shares and that keeps the previous call's contents, so every case makes two or more calls in a
row on different inputs and checks each; the file passes alone in a fresh process and after the rest of the suite.

Bar: the tests' dt tolerance, 1e-14 relative (tests/test_gpu_parity.py); the two paths use the same device functions
and max is exact, so the values are in fact expected to be equal."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

TOL = 1e-14


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    m.cfl_static_setup()
    return m


def mhd_state(rng, nv, full, rho0=1.0, cgl=False, form=0):
    """Random positive state [nv, nz, ny, nx]: conserved variables through the oracle's point functions."""
    import workloads
    W = np.empty((nv,) + full)
    W[0] = rho0 * (0.6 + 0.8 * rng.random(full)); W[1:4] = 0.4 * rho0 ** -0.5 * rng.standard_normal((3,) + full)
    W[4] = 0.5 + rng.random(full); W[5:8] = 0.3 + 0.3 * rng.standard_normal((3,) + full)
    if cgl:
        W[8] = 0.5 + rng.random(full)
        U = np.empty_like(W)
        fw, fu = W.reshape(nv, -1), U.reshape(nv, -1)
        for i in range(fw.shape[1]):
            fu[:9, i] = oracle.cgl_prim_to_cons(fw[:9, i], form)
        if nv == 10:
            U[9] = 0.05 * rng.standard_normal(full)
        return U
    if nv == 9:
        W[8] = 0.05 * rng.standard_normal(full)
    return workloads.prim_to_cons(W, 5.0 / 3.0)


CASES = [
    # eqset name, nv, shape, ndim, extra
    ("IDEAL", 8, (200, 150, 1), 2, {}),
    ("IDEAL", 8, (2500, 1, 1), 1, {}),                       # three segments of one row, the last one ragged
    ("HALL", 8, (40, 25, 13), 3, {"d_i": 0.7}),
    ("IDEAL_GLM", 9, (70, 33, 1), 2, {}),
    ("HALL_GLM", 9, (33, 17, 9), 3, {"d_i": 0.3}),
    ("CGL", 9, (90, 41, 1), 2, {"cgl_form": 0}),
    ("CGL_GLM", 10, (36, 20, 11), 3, {"cgl_form": 1}),
]


@pytest.mark.parametrize("name,nv,shape,ndim,extra", CASES)
def test_cfl_static_matches_the_context_path_on_calls_in_a_row(ag, name, nv, shape, ndim, extra):
    import torch
    eqset = getattr(ag, name)
    cgl = name.startswith("CGL")
    nx, ny, nz = shape
    dx = tuple([0.11, 0.07, 0.13][d] if d < ndim else 1.0 for d in range(3))
    rng = np.random.default_rng(sum(map(ord, name)) + ndim)
    # three states of very different v_max, largest first: a partial maximum left over from an earlier call would win
    states = [mhd_state(rng, nv, (nz, ny, nx), rho0, cgl, extra.get("cgl_form", 0)) for rho0 in (0.01, 1.0, 100.0)]
    kw = dict(shape=shape, dx=dx, ndim=ndim, eqset=eqset, riemann=0, d_i=extra.get("d_i", 0.0),
              cgl_form=extra.get("cgl_form", 0))
    ctx = ag.Agate(**kw)
    want = []
    for U in states:
        ctx.set_state(U)
        want.append((ctx.get_vmax(), ctx.compute_dt()))
    assert want[0][0] > 3 * want[1][0] and want[1][0] > 3 * want[2][0]
    Ud = [torch.from_numpy(U).cuda() for U in states]
    outs = [torch.full((3,), -1.0, dtype=torch.float64, device="cuda") for _ in states]
    # back to back on one stream, no synchronisation in between; then once more in reverse order
    for U, out in zip(Ud, outs):
        ag.cfl_static(U, out, shape, dx, ndim, eqset=eqset, d_i=kw["d_i"], cgl_form=kw["cgl_form"])
    torch.cuda.synchronize()
    for (vm, dt), out in zip(want, outs):
        got = out.cpu().numpy()
        assert abs(got[0] - vm) <= TOL * vm and abs(got[1] - dt) <= TOL * dt, (got, vm, dt)
        assert got[2] == 0.0
    for U, out, (vm, dt) in reversed(list(zip(Ud, outs, want))):
        out.fill_(-1.0)
        ag.cfl_static(U, out, shape, dx, ndim, eqset=eqset, d_i=kw["d_i"], cgl_form=kw["cgl_form"])
        got = out.cpu().numpy()
        assert abs(got[0] - vm) <= TOL * vm and abs(got[1] - dt) <= TOL * dt, (got, vm, dt)
    ctx.close()


def test_cfl_static_matches_the_oracle_and_honours_cfl(ag):
    """Against the oracle too (the definition: max over zones of |v| + c_f; dt = C dx_min / v_max), with a caller's
    Courant number, on a side stream."""
    import torch
    import workloads
    wl = workloads.make_workload(1, n=96)
    ref = oracle.RefSolver.from_workload(wl, cfl=0.3)
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    U = torch.from_numpy(wl.U).cuda()
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    for _ in range(2):
        ag.cfl_static(U, out, wl.shape, wl.dx, wl.ndim, eqset=ag.IDEAL, cfl=0.3, stream=st)
    st.synchronize()
    got = out.cpu().numpy()
    assert abs(got[0] - ref.vmax()) <= 1e-13 * ref.vmax()
    assert abs(got[1] - ref.compute_dt()) <= 1e-13 * got[1]
    ref.close()


def test_cfl_static_flags_unphysical_zones_and_recovers(ag):
    import torch
    rng = np.random.default_rng(7)
    shape, dx = (64, 20, 1), (0.1, 0.1, 1.0)
    U = mhd_state(rng, 8, (1, 20, 64))
    bad = U.copy()
    bad[0, 0, 5, 17] = -1.0                                   # rho < 0 in one zone (R14)
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    ag.cfl_static(torch.from_numpy(bad).cuda(), out, shape, dx, 2)
    assert out.cpu().numpy()[2] == 1.0
    ctx = ag.Agate(shape=shape, dx=dx, ndim=2, riemann=0)
    ctx.set_state(U)
    vm = ctx.get_vmax()
    ag.cfl_static(torch.from_numpy(U).cuda(), out, shape, dx, 2)           # the flag of the last call must not stick
    got = out.cpu().numpy()
    assert got[2] == 0.0 and abs(got[0] - vm) <= TOL * vm
    ctx.close()


def test_cfl_static_rejects_sizes_beyond_the_static_array(ag):
    import ctypes as C
    import torch
    L = ag.lib()
    mx = int(L.agate_cfl_static_max_segments())
    assert mx == 65536
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    dummy = torch.zeros(8, dtype=torch.float64, device="cuda")             # never read: the size check comes first
    cfg = ag.SolverCfg(0, 2, 1.3, 2, 0.0, 0.0)
    p = lambda t: C.c_void_p(t.data_ptr())
    for grid in (ag.Grid(2, 4, mx + 1, 1, 1.0, 1.0, 1.0), ag.Grid(3, 512, 512, 512, 1.0, 1.0, 1.0),
                 ag.Grid(3, 1025, 256, 256, 1.0, 1.0, 1.0)):
        rc = L.agate_cfl_static(C.byref(grid), 5.0 / 3.0, ag.IDEAL, C.byref(cfg), p(dummy), p(out), None)
        assert rc == 6
    assert b"static array" in L.agate_strerror(6)
    with pytest.raises(ag.AgateError) as e:
        big = torch.zeros(8 * 4 * (mx + 1), dtype=torch.float64, device="cuda")
        ag.cfl_static(big, out, (4, mx + 1, 1), (1.0, 1.0, 1.0), 2)
    assert e.value.code == 6
    # exactly at the limit it runs: 4 x 65536 zones of a uniform state
    W = np.array([1.0, 0.1, 0.0, 0.0, 0.6, 0.5, 0.0, 0.0])
    import workloads
    U1 = workloads.prim_to_cons(W.reshape(8, 1, 1, 1), 5.0 / 3.0).reshape(8)
    U = torch.from_numpy(np.repeat(U1, 4 * mx)).cuda()
    ag.cfl_static(U, out, (4, mx, 1), (1.0, 1.0, 1.0), 2)
    cf = np.sqrt((5.0 / 3.0 * 0.6 + 0.25) / 1.0)                           # B along x: c_f = max(a, v_A) along x, sqrt(a^2 + v_A^2) across
    assert abs(out.cpu().numpy()[0] - (0.1 + cf)) <= 1e-13
    # argument errors
    assert L.agate_cfl_static(C.byref(ag.Grid(2, 8, 8, 1, 1.0, 1.0, 1.0)), 5.0 / 3.0, ag.IDEAL, C.byref(cfg), None, p(out), None) == 1
    assert L.agate_cfl_static(C.byref(ag.Grid(2, 8, 8, 1, 1.0, 1.0, 1.0)), 5.0 / 3.0, 9, C.byref(cfg), p(dummy), p(out), None) == 1
