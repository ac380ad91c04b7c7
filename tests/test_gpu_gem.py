"""The GEM reconnection setup of PAPER.md §4.6 (L336-358) on the GPU against the oracle (-m gpu): Harris sheet
B_x = tanh 2y, rho = 0.2 + sech^2 2y, p = rho / 2 on [-12.8, 12.8] x [-6.4, 6.4], the flux perturbation of eq.36 with
delta_B = 0.1, periodic in x, zero-gradient ends in y (R26), for ideal, Hall (d_i = 1) and CGL MHD (isotropic
start, relaxation 0.99).  Reduced grid (same aspect), a few dozen steps: this checks that the path the paper's
last benchmark needs (Hall with open ends, CGL with relaxation and open ends) runs through the kernels and matches."""
import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import TOL_DT, TOL_N, rel_linf

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ag():
    import paper_2503_20899_b200 as m
    m.lib()
    return m


def gem_prims(nx, ny):
    Lx, Ly, dB = 25.6, 12.8, 0.1
    x = -Lx / 2 + (np.arange(nx) + 0.5) * Lx / nx
    y = -Ly / 2 + (np.arange(ny) + 0.5) * Ly / ny
    X, Y = np.meshgrid(x, y)
    W = np.zeros((8, 1, ny, nx))
    W[0, 0] = 0.2 + 1.0 / np.cosh(2 * Y) ** 2
    W[4, 0] = 0.5 * W[0, 0]
    W[5, 0] = np.tanh(2 * Y) - dB * (np.pi / Ly) * np.cos(2 * np.pi * X / Lx) * np.sin(np.pi * Y / Ly)      # eq.36
    W[6, 0] = dB * (2 * np.pi / Lx) * np.sin(2 * np.pi * X / Lx) * np.cos(np.pi * Y / Ly)
    return W, (Lx / nx, Ly / ny, 1.0)


@pytest.mark.parametrize("kind", ["ideal", "hall", "cgl"])
def test_gem_setup_parity(ag, kind):
    nx, ny = 128, 64
    W, dx = gem_prims(nx, ny)
    kw = dict(shape=(nx, ny, 1), dx=dx, ndim=2, riemann=oracle.HLL, limiter=2, beta=1.3, rk=2, bc=(0, 1, 0))
    if kind == "cgl":
        W9 = np.concatenate([W, W[4:5]], axis=0)                       # p_par = p_perp = p
        U = np.empty_like(W9)
        fw, fu = W9.reshape(9, -1), U.reshape(9, -1)
        for i in range(fw.shape[1]):
            fu[:, i] = oracle.cgl_prim_to_cons(fw[:, i])
        eo, eg = oracle.CGL, ag.CGL
        kw["relax"] = 0.99
    else:
        U = workloads.prim_to_cons(W, 5.0 / 3.0)
        eo, eg = (oracle.HALL, ag.HALL) if kind == "hall" else (oracle.IDEAL, ag.IDEAL)
        if kind == "hall":
            kw["d_i"] = 1.0
    ref = oracle.RefSolver(eqset=eo, **kw); gpu = ag.Agate(eqset=eg, **kw)
    ref.set_state(U); gpu.set_state(U)
    for s in range(40):
        dtr, dtg = ref.compute_dt(), gpu.compute_dt()
        assert abs(dtg - dtr) <= TOL_DT * dtr
        ref.step(dtr)
        assert gpu.step(0.0) == dtg
    Ug, Ur = gpu.get_state(), ref.get_state()
    assert np.all(rel_linf(Ug[:8], Ur[:8]) <= TOL_N)
    if kind == "cgl":
        sc = max(np.max(np.abs(Ur[8])), np.max(np.abs(Ur[0])))
        assert np.max(np.abs(Ug[8] - Ur[8])) <= TOL_N * sc
    # the reconnected flux of P:L360, -int_{-Lx/2}^{0} B_y dx along the sheet, agrees as well
    j0 = ny // 2
    flux = lambda V: -0.5 * (V[6, 0, j0 - 1, : nx // 2] + V[6, 0, j0, : nx // 2]).sum() * dx[0]
    assert abs(flux(Ug) - flux(Ur)) <= 1e-12 * max(abs(flux(Ur)), 1e-3)
    ref.close(); gpu.close()
