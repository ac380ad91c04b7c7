"""NEXT-4 on ONE GPU (-m gpu): two (or three) contexts hold the slabs of one problem, exchange their halos by device
copies every stage and take the maximum of their v_max every step; they must reproduce the undivided run bit for bit
(dt included), on 3-D grids (z slabs) and 2-D grids (y slabs), for ideal, Hall, GLM, CGL and CGL + GLM, periodic and open
ends."""
import numpy as np
import pytest

import workloads
from workloads import HALL, HLL, HLLD, IDEAL, make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    return m


def run_slabs(ag, kw, U, nslab, steps, periodic, eqset=0, use_device_vmax=False):
    from paper_2503_20899_b200 import slab
    import torch
    ndim = kw["ndim"]
    nx, ny, nz = kw["shape"]
    ncut = nz if ndim == 3 else ny
    parts = slab.split(ncut, nslab)
    ctxs, bufs, cuts = [], [], []
    for r, (s0, cnt) in enumerate(parts):
        k = dict(kw)
        k["shape"] = (nx, ny, cnt) if ndim == 3 else (nx, cnt, 1)
        c = ag.Agate(eqset=eqset, **k)
        lo, hi = slab.neighbours(r, nslab, periodic)
        c.set_slab(lo is not None, hi is not None)
        Us = U[:, s0:s0 + cnt] if ndim == 3 else U[:, :, s0:s0 + cnt]
        c.set_state(np.ascontiguousarray(Us))
        ctxs.append(c); bufs.append(c.halo_buffers()); cuts.append((lo, hi))
    rk = kw.get("rk", 2)
    dts = []
    for step in range(steps):
        vm = max(c.get_vmax() for c in ctxs)
        for c in ctxs:
            c.set_vmax(vm)
            c.step_begin(0.0)
        for s in range(rk):
            for c, b, (lo, hi) in zip(ctxs, bufs, cuts):
                c.stage_pre(s, b[0] if lo is not None else None, b[1] if hi is not None else None)
            torch.cuda.synchronize()
            for r, (lo, hi) in enumerate(cuts):
                if hi is not None:
                    bufs[hi][2].copy_(bufs[r][1])          # my send_hi -> upper neighbour's recv_lo
                if lo is not None:
                    bufs[lo][3].copy_(bufs[r][0])          # my send_lo -> lower neighbour's recv_hi
            torch.cuda.synchronize()
            for c, b, (lo, hi) in zip(ctxs, bufs, cuts):
                c.stage_post(s, b[2] if lo is not None else None, b[3] if hi is not None else None)
    outs = [c.get_state() for c in ctxs]
    ts = [c.t for c in ctxs]
    for c in ctxs:
        c.close()
    return np.concatenate(outs, axis=1 if ndim == 3 else 2), ts


@pytest.mark.parametrize("rk,riemann,nslab,bcz", [(2, HLLD, 2, 0), (3, HLL, 3, 0), (5, HLLD, 2, 1), (4, HLLD, 2, 0)])
def test_z_slabs_reproduce_the_undivided_run_3d(ag, rk, riemann, nslab, bcz):
    wl = make_workload(3, n=40)
    U = wl.U[:, :, :, :]
    shape = (40, 40, 40)
    kw = dict(shape=shape, dx=wl.dx, ndim=3, gamma=wl.gamma, riemann=riemann, limiter=2, beta=1.3, rk=rk, cfl=wl.cfl,
              bc=(0, 0, bcz))
    one = ag.Agate(**kw)
    one.set_state(U)
    t1 = one.advance(3)
    U1 = one.get_state()
    one.close()
    U2, ts = run_slabs(ag, kw, U, nslab, 3, periodic=(bcz == 0))
    assert all(t == t1 for t in ts), (ts, t1)
    assert np.array_equal(U1.view(np.uint64), U2.view(np.uint64))


def test_y_slabs_reproduce_the_undivided_run_2d_hall(ag):
    """Hall needs the edge / corner ghosts: the halo rows travel with their own x ghosts."""
    wl = make_workload(4, n=64)
    kw = dict(shape=wl.shape, dx=wl.dx, ndim=2, gamma=wl.gamma, riemann=HLL, limiter=2, beta=wl.beta, rk=2, cfl=wl.cfl,
              d_i=wl.d_i)
    one = ag.Agate(eqset=HALL, **kw)
    one.set_state(wl.U)
    t1 = one.advance(4)
    U1 = one.get_state()
    one.close()
    U2, ts = run_slabs(ag, kw, wl.U, 3, 4, periodic=True, eqset=HALL)
    assert all(t == t1 for t in ts)
    assert np.array_equal(U1.view(np.uint64), U2.view(np.uint64))


def test_glm_slabs_share_ch(ag):
    """GLM: c_h = 0.95 x the GLOBAL v_max enters every face flux, so it must be the all-reduced value."""
    wl = make_workload(6, n=64)
    kw = dict(shape=wl.shape, dx=wl.dx, ndim=2, gamma=wl.gamma, riemann=wl.riemann, limiter=2, beta=wl.beta, rk=2,
              cfl=wl.cfl)
    one = ag.Agate(eqset=ag.IDEAL_GLM, **kw)
    one.set_state(wl.U)
    t1 = one.advance(4)
    U1 = one.get_state()
    one.close()
    U2, ts = run_slabs(ag, kw, wl.U, 2, 4, periodic=True, eqset=ag.IDEAL_GLM)
    assert all(t == t1 for t in ts)
    assert np.array_equal(U1.view(np.uint64), U2.view(np.uint64))


@pytest.mark.parametrize("cfg,ndim,n,nslab", [(7, 2, 64, 2), (9, 2, 66, 3), (9, 3, 24, 2)])
def test_cgl_and_cgl_glm_slabs(ag, cfg, ndim, n, nslab):
    """CGL and CGL + GLM: kernels without the fused reduction, so every step's v_max (and with it c_h) goes through
    agate_get_vmax / agate_set_vmax; relaxation and the psi source act in the last stage of every slab alike."""
    wl = make_workload(cfg, n=n)
    U = wl.U
    shape, dx = wl.shape, wl.dx
    if ndim == 3:                         # the Orszag-Tang rows stacked along z with a z-dependent flow on top
        z = (np.arange(n) + 0.5) / n
        U = np.ascontiguousarray(np.repeat(U, n, axis=1))
        U[3] = U[0] * 0.2 * np.sin(2 * np.pi * z)[:, None, None]
        U[4] = U[4] + 0.5 * U[3] ** 2 / U[0]
        shape, dx = (n, n, n), (1.0 / n,) * 3
    kw = dict(shape=shape, dx=dx, ndim=ndim, gamma=wl.gamma, riemann=wl.riemann, limiter=2, beta=wl.beta, rk=2,
              cfl=wl.cfl if ndim == 2 else 0.325, relax=wl.relax)
    one = ag.Agate(eqset=wl.eqset, **kw)
    one.set_state(U)
    t1 = one.advance(4)
    U1 = one.get_state()
    one.close()
    U2, ts = run_slabs(ag, kw, U, nslab, 4, periodic=True, eqset=wl.eqset)
    assert all(t == t1 for t in ts)
    assert np.array_equal(U1.view(np.uint64), U2.view(np.uint64))
    assert not np.array_equal(U1, U)


def test_single_rank_stepper_periodic_self_exchange(ag):
    """SlabStepper with one rank and a periodic dimension: the slab is its own neighbour (the path bench.py --decomp
    times at N = 1), with the device-resident v_max from the second step on."""
    from paper_2503_20899_b200 import slab
    wl = make_workload(3, n=40)
    one = ag.Agate.from_workload(wl)
    t1 = one.advance(4)
    U1 = one.get_state()
    one.close()
    c = ag.Agate.from_workload(wl)
    st = slab.SlabStepper(c, 0, 1, True)
    for _ in range(4):
        st.step()
    U2 = c.get_state()
    assert c.t == t1
    assert np.array_equal(U1.view(np.uint64), U2.view(np.uint64))
    # call order is checked
    with pytest.raises(ag.AgateError):
        c.advance(1)                       # a slab steps through stage_pre / stage_post
    with pytest.raises(ag.AgateError):
        c.stage_post(0, st.recv_lo, st.recv_hi)
    c.close()
