"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times  (-m gpu).

The oracle cannot advance 2048^2 / 256^3 / 512^3 zones in seconds, but it can compute any output zone on its own: a
zone after n SSP-RK2 steps depends on the input within 4n zones (two per stage: PLM needs i-1..i+2 around a face,
the Hall current the same cells plus their transverse neighbours).  So the GPU advances the whole config-sized state,
and the oracle advances small periodic boxes cut out of the SAME input around seeded sample points, with the dt the
GPU used; zones of a box farther than the dependence radius from its edge never see the box's wrap-around and must
equal the GPU's zones.  Boxes are placed on tile, segment and domain boundaries as well as at random.

dt at full size is pinned to the Courant formula itself (readings R3-R5), evaluated here with numpy
in slabs -- a closed form, independent of the oracle's code and of the CUDA path.
"""
import numpy as np
import pytest

import oracle
from workloads import make_workload

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12      # north_star: relative L-inf per conserved variable after one step
TOL_DT = 1e-14     # north_star: dt


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    return m


def rel_linf(Ug, Ur):
    """R19 metric: per-variable max |diff| / scale, vector components share the scale of their vector."""
    sc = np.empty(8)
    sc[0] = np.max(np.abs(Ur[0])); sc[4] = np.max(np.abs(Ur[4]))
    sc[1:4] = np.max(np.abs(Ur[1:4])); sc[5:8] = np.max(np.abs(Ur[5:8]))
    err = np.empty(8)
    for q in range(8):
        d = np.max(np.abs(Ug[q] - Ur[q]))
        err[q] = d / sc[q] if sc[q] > 0 else d
    return err


def courant_dt(wl):
    """C dx_min / max(|v| + max(max_d c_f,d, c_w))  (R4, R5; eq.12 as R3; eq.13 with k_max = pi/dx_min), in z slabs."""
    U = wl.U
    g = wl.gamma
    act = wl.dx[:wl.ndim]
    dxmin = min(act)
    vmax = 0.0
    nz = U.shape[1]
    step = max(1, (1 << 22) // (U.shape[2] * U.shape[3]))
    for k in range(0, nz, step):
        rho, mx, my, mz, E, bx, by, bz = (U[q, k:k + step] for q in range(8))
        v2 = (mx * mx + my * my + mz * mz) / (rho * rho)
        B2 = bx * bx + by * by + bz * bz
        p = (g - 1.0) * (E - 0.5 * rho * v2 - 0.5 * B2)
        a2 = g * p / rho
        sm = a2 + B2 / rho
        bmin2 = np.minimum(np.minimum(bx * bx, by * by), bz * bz)
        c = np.sqrt(0.5 * (sm + np.sqrt(np.maximum(sm * sm - 4.0 * a2 * bmin2 / rho, 0.0))))
        if wl.eqset == oracle.HALL:
            aw = wl.d_i * np.pi * np.sqrt(B2) / (2.0 * rho * dxmin)
            c = np.maximum(c, aw + np.sqrt(aw * aw + B2 / rho))
        vmax = max(vmax, float(np.max(np.sqrt(v2) + c)))
    cfl = wl.cfl if wl.cfl > 0 else {1: 0.8, 2: 0.45, 3: 0.325}[wl.ndim]
    return cfl * dxmin / vmax


def sample_points(shape, ndim, n_random, seed):
    """Box centres (x, y, z): the domain corner (periodic wrap), tile / row-block seams of the kernels, random ones."""
    nx, ny, nz = shape
    pts = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (32, 11, nz // 2), (nx // 2 + 31, 6, 1), (31, ny // 2, nz - 2)]
    rng = np.random.default_rng(seed)
    for _ in range(n_random):
        pts.append((int(rng.integers(nx)), int(rng.integers(ny)), int(rng.integers(nz))))
    if ndim < 3:
        pts = [(x, y, 0) for (x, y, _) in pts]
    return pts


@pytest.mark.parametrize("cfg,n_steps", [(2, 2), (3, 2), (4, 2), (5, 1)])
def test_full_size_sampled(ag, cfg, n_steps):
    wl = make_workload(cfg)
    wl.W = None
    nx, ny, nz = wl.shape
    gpu = ag.Agate.from_workload(wl)
    dt_closed = courant_dt(wl)
    dts = []
    for s in range(n_steps):
        dtg = gpu.compute_dt()
        if s == 0:
            assert abs(dtg - dt_closed) <= TOL_DT * dt_closed, (dtg, dt_closed)
        used = gpu.step(0.0)                      # the path bench.py times: device-resident dt, fused stages
        assert used == dtg
        dts.append(used)
    Ug = gpu.get_state()
    gpu.close()

    rad = 4 * n_steps                             # dependence radius of n SSP-RK2 steps
    core = 6 if wl.ndim == 3 else 16
    half = core // 2 + rad + 1
    worst = np.zeros(8)
    for (cx, cy, cz) in sample_points(wl.shape, wl.ndim, 6 if wl.ndim == 3 else 10, 1000 + cfg):
        ix = np.arange(cx - half, cx + half) % nx
        iy = np.arange(cy - half, cy + half) % ny
        iz = (np.arange(cz - half, cz + half) % nz) if wl.ndim == 3 else np.array([0])
        box = np.ascontiguousarray(wl.U[:, iz][:, :, iy][:, :, :, ix])
        ref = oracle.RefSolver(shape=(len(ix), len(iy), len(iz)), dx=wl.dx, ndim=wl.ndim, gamma=wl.gamma,
                               eqset=wl.eqset, riemann=wl.riemann, limiter=wl.limiter, beta=wl.beta, rk=wl.rk,
                               cfl=wl.cfl, d_i=wl.d_i)
        ref.set_state(box)
        for d in dts:
            ref.step(d)
        Ur = ref.get_state().reshape(box.shape)
        ref.close()
        lo, hi = rad + 1, 2 * half - rad - 1
        kz = slice(lo, hi) if wl.ndim == 3 else slice(0, 1)
        got = Ug[:, iz[kz]][:, :, iy[lo:hi]][:, :, :, ix[lo:hi]]
        want = Ur[:, kz, lo:hi, lo:hi]
        worst = np.maximum(worst, rel_linf(got, want))
    tol = TOL_1 if n_steps == 1 else 1e-11       # two steps: between the 1-step and the 100-step (1e-9) bounds
    assert np.all(worst <= tol), f"config {cfg}: rel L-inf on sampled boxes {worst}"
