"""Seeded synthetic workloads for the five BASELINE.json configs (SURVEY.md §8(d) generator).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2503_20899_b200/`): both consume the arrays produced here through their own `set_state`.
It holds none of the method's arithmetic (no reconstruction, no Riemann solver, no time stepping).
The single physics-flavoured line is the *definition* of the conserved vector from the primitive one,
U = (rho, rho v, p/(gamma-1) + rho v^2/2 + B^2/2, B)   (with the (gamma-1) typo fix R2),
which is input construction, not a step of the path; the oracle's own cons<->prim maps are pinned
separately against hand values (tests/test_oracle_pins.py, P3).

Recipe: unit box, cell centres x=(i+1/2)/n.
    S_M^K(x) = (1/M) sum_{m=1..M} cos(2 pi k_m.x + phi_m),
each component of the integer vector k_m uniform in {-K..K} (redrawn if k_m = 0), phi_m uniform in
[0, 2 pi).  RNG = splitmix64 seeded with 2503208990 + config_id; u = (next>>11) 2^-53; integer =
floor(u (2K+1)) - K; draw order = fields in the order listed per config, per mode kx, ky[, kz] then phi.
curl_c = periodic central-difference curl of potentials point-sampled at cell centres, so the
central-difference div B is zero to round-off.

The configs stand in for the paper's 2D/3D periodic runs (Orszag-Tang-like turbulence);
the paper measures on a problem, not a dataset.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# Variable order: conserved U = (rho, mx, my, mz, E, Bx, By, Bz),
#                                primitive W = (rho, vx, vy, vz, p, Bx, By, Bz).
NVAR = 8
IDEAL, HALL = 0, 1
IDEAL_GLM = 3          # 9 variables per cell: the GLM scalar psi behind the 8 MHD ones
CGL = 2                # 9 variables per cell: U = (rho, m, E, B, A_log), W = (rho, v, p_par, B, p_perp)
CGL_GLM = 5            # 10 variables per cell: CGL's nine, then the GLM scalar psi (eqs.19-23)
HLL, HLLD = 0, 1
GAMMA = 5.0 / 3.0
SEED_BASE = 2503208990
_MASK = (1 << 64) - 1


class SplitMix64:
    """splitmix64 counter-based generator (public-domain algorithm by S. Vigna), pure Python ints."""

    def __init__(self, seed: int):
        self.s = seed & _MASK

    def next(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & _MASK
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return (self.next() >> 11) * 2.0 ** -53

    def integer(self, K: int) -> int:
        return int(math.floor(self.uniform() * (2 * K + 1))) - K


@dataclasses.dataclass
class Workload:
    """One seeded problem: the interior-only SoA state plus the solver settings of its config."""
    config_id: int
    ndim: int
    shape: tuple          # (nx, ny, nz); inactive dims are 1
    dx: tuple             # (dx, dy, dz)
    gamma: float
    eqset: int            # IDEAL / HALL
    riemann: int          # HLL / HLLD
    limiter: int          # 2 = eq.4
    beta: float
    rk: int
    cfl: float
    d_i: float
    n_steps: int
    W: np.ndarray         # [8, nz, ny, nx] float64, primitive
    U: np.ndarray         # [8, nz, ny, nx] float64, conserved (x fastest)
    name: str = ""
    relax: float = 0.0    # CGL: dt/(dt+tau) of eqs.32-33

    @property
    def zones(self) -> int:
        return int(self.shape[0]) * int(self.shape[1]) * int(self.shape[2])


def draw_modes(rng: SplitMix64, M: int, K: int, ndim: int):
    """Draw M modes: per mode kx, ky[, kz] (redraw the whole vector if it is zero) then phi."""
    ks = np.zeros((M, 3), dtype=np.int64)
    phis = np.zeros(M)
    for m in range(M):
        while True:
            k = [rng.integer(K) for _ in range(ndim)]
            if any(k):
                break
        ks[m, :ndim] = k
        phis[m] = 2.0 * math.pi * rng.uniform()
    return ks, phis


def mode_sum(ks, phis, shape) -> np.ndarray:
    """S(x) = (1/M) sum_m cos(2 pi k_m.x + phi_m) on cell centres; returns [nz, ny, nx].

    Evaluated through the separable form cos(a+b+c) -> real/imag products of 1-D tables and one
    real matrix product over z, so the 512^3 case costs ~17 GFLOP instead of 4e9 cosines per field."""
    nx, ny, nz = shape
    M = len(phis)
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    z = (np.arange(nz) + 0.5) / nz
    tp = 2.0 * math.pi
    ex = np.exp(1j * tp * np.outer(ks[:, 0], x))                      # [M, nx]
    ey = np.exp(1j * (tp * np.outer(ks[:, 1], y) + phis[:, None]))    # [M, ny] (phase folded in)
    ez = np.exp(1j * tp * np.outer(ks[:, 2], z))                      # [M, nz]
    A = (ey[:, :, None] * ex[:, None, :]).reshape(M, ny * nx)         # [M, ny*nx] complex
    # Re( sum_m ez[m,k] A[m,:] ) = ez_re^T A_re - ez_im^T A_im
    L = np.concatenate([ez.real.T, -ez.imag.T], axis=1)               # [nz, 2M]
    R = np.concatenate([A.real, A.imag], axis=0)                      # [2M, ny*nx]
    out = (L @ R).reshape(nz, ny, nx) / M
    return np.ascontiguousarray(out)


def _field(rng, M, K, ndim, shape):
    ks, phis = draw_modes(rng, M, K, ndim)
    return mode_sum(ks, phis, shape)


def _d(f, axis, h):
    """Periodic central difference along array axis (0=z,1=y,2=x)."""
    return (np.roll(f, -1, axis=axis) - np.roll(f, 1, axis=axis)) / (2.0 * h)


def curl_c(Ax, Ay, Az, dx, ndim):
    """Periodic central-difference curl; derivatives along inactive dimensions are zero."""
    hx, hy, hz = dx
    zero = np.zeros_like(Az)
    dAz_dy = _d(Az, 1, hy) if ndim >= 2 else zero
    dAz_dx = _d(Az, 2, hx)
    dAy_dx = _d(Ay, 2, hx) if Ay is not None else zero
    dAx_dy = _d(Ax, 1, hy) if (Ax is not None and ndim >= 2) else zero
    dAy_dz = _d(Ay, 0, hz) if (Ay is not None and ndim >= 3) else zero
    dAx_dz = _d(Ax, 0, hz) if (Ax is not None and ndim >= 3) else zero
    return dAz_dy - dAy_dz, dAx_dz - dAz_dx, dAy_dx - dAx_dy


def _rms(*comps):
    return math.sqrt(float(np.mean(sum(c * c for c in comps))))


def prim_to_cons(W: np.ndarray, gamma: float) -> np.ndarray:
    """Definition of the conserved vector (PAPER.md L140 with R2: p/(gamma-1))."""
    rho, vx, vy, vz, p, bx, by, bz = W[:8]
    U = np.empty_like(W)
    if W.shape[0] > 8:
        U[8:] = W[8:]                 # the GLM scalar is its own conserved variable
    U[0] = rho
    U[1] = rho * vx
    U[2] = rho * vy
    U[3] = rho * vz
    U[4] = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bx * bx + by * by + bz * bz)
    U[5] = bx
    U[6] = by
    U[7] = bz
    return U


# Full-size grids and solver settings per config (BASELINE.json configs).
def prim_to_cons_cgl(W: np.ndarray) -> np.ndarray:
    """Definition of the CGL conserved vector from W = (rho, v, p_par, B, p_perp): E = rho v^2/2 + B^2/2 + p_par/2 +
    p_perp, A_log = rho log[(rho^2/B^3)(p_perp/p_par)] (eq.18)."""
    rho, vx, vy, vz, ppar, bx, by, bz, pperp = W[:9]
    b2 = bx * bx + by * by + bz * bz
    U = np.empty_like(W)
    if W.shape[0] > 9:
        U[9:] = W[9:]                 # the GLM scalar is its own conserved variable
    U[0] = rho; U[1] = rho * vx; U[2] = rho * vy; U[3] = rho * vz
    U[4] = 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * b2 + 0.5 * ppar + pperp
    U[5] = bx; U[6] = by; U[7] = bz
    U[8] = rho * np.log((rho * rho / (b2 * np.sqrt(b2))) * (pperp / ppar))
    return U


_CONFIGS = {
    1: dict(ndim=2, n=128,  eqset=IDEAL, riemann=HLL,  beta=1.0, cfl=0.4,   d_i=0.0,  n_steps=10,
            name="cfg1: 2D ideal 128^2 HLL minmod"),
    2: dict(ndim=2, n=2048, eqset=IDEAL, riemann=HLLD, beta=1.3, cfl=0.45,  d_i=0.0,  n_steps=100,
            name="cfg2: 2D ideal 2048^2 HLLD MC"),
    3: dict(ndim=3, n=256,  eqset=IDEAL, riemann=HLLD, beta=1.3, cfl=0.325, d_i=0.0,  n_steps=50,
            name="cfg3: 3D ideal 256^3 HLLD MC"),
    4: dict(ndim=2, n=1024, eqset=HALL,  riemann=HLL,  beta=1.0, cfl=0.45,  d_i=0.05, n_steps=50,
            name="cfg4: 2D Hall 1024^2 HLL minmod"),
    5: dict(ndim=3, n=512,  eqset=IDEAL, riemann=HLLD, beta=1.3, cfl=0.325, d_i=0.0,  n_steps=20,
            name="cfg5: 3D ideal 512^3 HLLD MC (headline)"),
    # NEXT-1, not a BASELINE.json config: the workload of the paper's Table 2 -- Orszag-Tang vortex
    # (IC printed at P:L282) with GLM divergence cleaning, "default settings": PLM + eq.4 beta=1.3, HLL, C=0.45.
    6: dict(ndim=2, n=2048, eqset=IDEAL_GLM, riemann=HLL, beta=1.3, cfl=0.45,  d_i=0.0,  n_steps=100,
            name="cfg6: 2D Orszag-Tang + GLM 2048^2 HLL MC (paper Table 2 workload)"),
    # NEXT-2, not a BASELINE.json config: the Orszag-Tang vortex in CGL MHD ("In the CGL MHD version, we set
    # the initial anisotropy to zero"), HLL, default relaxation dt/(dt+tau) = 0.99
    7: dict(ndim=2, n=2048, eqset=CGL, riemann=HLL, beta=1.3, cfl=0.45, d_i=0.0, n_steps=100, relax=0.99,
            name="cfg7: 2D Orszag-Tang CGL 2048^2 HLL MC"),
    # not a BASELINE.json config: config 4's setting (Hall MHD, HLL, eq.4 at beta = 1, d_i across ~50 zones) on config
    # 3's three-dimensional recipe, for the 3-D Hall path of the row-owner kernel
    8: dict(ndim=3, n=256, eqset=HALL, riemann=HLL, beta=1.0, cfl=0.325, d_i=0.2, n_steps=50,
            name="cfg8: 3D Hall 256^3 HLL minmod"),
    # not a BASELINE.json config: config 7 with the GLM scalar, i.e. the whole of eqs.19-23 on the Orszag-Tang vortex
    9: dict(ndim=2, n=2048, eqset=CGL_GLM, riemann=HLL, beta=1.3, cfl=0.45, d_i=0.0, n_steps=100, relax=0.99,
            name="cfg9: 2D Orszag-Tang CGL + GLM 2048^2 HLL MC"),
}


def config_settings(config_id: int) -> dict:
    return dict(_CONFIGS[config_id])


def make_workload(config_id: int, n: int | None = None, n_steps: int | None = None,
                  scale_d_i: bool = True) -> Workload:
    """Build config `config_id` (1..5: BASELINE.json; 6: Orszag-Tang + GLM, the paper's Table 2 workload). `n` overrides the per-dimension resolution (reduced-size
    parity cases use the same recipe and seed); for config 4, d_i is rescaled with n so that d_i/dx
    stays 51.2 cells (`scale_d_i`)."""
    c = config_settings(config_id)
    ndim = c["ndim"]
    nfull = c["n"]
    n = nfull if n is None else int(n)
    shape = (n, n, n if ndim == 3 else 1)
    dx = (1.0 / n, 1.0 / n, 1.0 / n if ndim == 3 else 1.0)
    rng = SplitMix64(SEED_BASE + config_id)
    g = GAMMA
    nx, ny, nz = shape
    W = np.empty((NVAR + {IDEAL_GLM: 1, CGL: 1, CGL_GLM: 2}.get(c["eqset"], 0), nz, ny, nx))
    F = lambda M, K: _field(rng, M, K, ndim, shape)

    if config_id in (6, 7, 9):
        # rho = 25/(36 pi), p = 5/(12 pi), v = (-sin 2 pi y, sin 2 pi x, 0), B = B0 (-sin 2 pi y, sin 4 pi x, 0),
        # B0 = 1/sqrt(4 pi), unit box, cell centres; psi = 0
        xc = ((np.arange(nx) + 0.5) / nx)[None, None, :]
        yc = ((np.arange(ny) + 0.5) / ny)[None, :, None]
        B0 = 1.0 / math.sqrt(4.0 * math.pi)
        W[0] = 25.0 / (36.0 * math.pi)
        W[4] = 5.0 / (12.0 * math.pi)
        W[1] = -np.sin(2.0 * math.pi * yc) + 0.0 * xc
        W[2] = np.sin(2.0 * math.pi * xc) + 0.0 * yc
        W[3] = 0.0
        W[5] = -B0 * np.sin(2.0 * math.pi * yc) + 0.0 * xc
        W[6] = B0 * np.sin(4.0 * math.pi * xc) + 0.0 * yc
        W[7] = 0.0
        W[8] = 0.0 if config_id == 6 else W[4]      # GLM: psi = 0;  CGL: p_perp = p_par = p
        if config_id == 9:
            W[9] = 0.0
    elif config_id in (1, 4):
        W[0] = 1.0 + 0.1 * F(4, 4)
        W[1] = 0.1 * F(4, 4)
        W[2] = 0.1 * F(4, 4)
        W[3] = 0.1 * F(4, 4)
        Az = F(4, 4)
        bx, by, _ = curl_c(None, None, Az, dx, ndim)
        amp = 0.1 / max(float(np.max(np.abs(bx))), float(np.max(np.abs(by))))
        W[5] = bx * amp
        W[6] = by * amp
        bz = 0.1 * F(4, 4)                    # drawn for both configs so the draw order is shared
        W[7] = bz if config_id == 1 else 1.0  # config 4: uniform guide field
        W[4] = 1.0
    elif config_id == 2:
        W[0] = 1.0 + 0.5 * F(16, 8)
        yc = ((np.arange(ny) + 0.5) / ny)[None, :, None]
        W[1] = 0.5 * np.tanh((yc - 0.5) / 0.05) + 0.01 * F(4, 8)
        W[2] = 0.01 * F(4, 8)
        W[3] = 0.0
        Az = F(16, 8)
        bx, by, _ = curl_c(None, None, Az, dx, ndim)
        s = 0.2 / _rms(bx, by)
        W[5] = bx * s + 0.1
        W[6] = by * s
        W[7] = 0.0
        W[4] = 1.0
    elif config_id in (3, 8):
        W[0] = 1.0 + 0.2 * F(8, 4)
        Px, Py, Pz = F(8, 4), F(8, 4), F(8, 4)
        vx, vy, vz = curl_c(Px, Py, Pz, dx, ndim)
        s = 0.3 / _rms(vx, vy, vz)
        W[1], W[2], W[3] = vx * s, vy * s, vz * s
        del Px, Py, Pz, vx, vy, vz
        Ax, Ay, Az = F(8, 4), F(8, 4), F(8, 4)
        bx, by, bz = curl_c(Ax, Ay, Az, dx, ndim)
        s = 0.2 / _rms(bx, by, bz)
        W[5], W[6], W[7] = bx * s + 0.1, by * s, bz * s
        W[4] = 0.6
    elif config_id == 5:
        gfield = math.sqrt(2.0 * 32) * F(32, 8)
        W[0] = np.exp(0.3 * gfield - 0.045)
        del gfield
        Px, Py, Pz = F(32, 8), F(32, 8), F(32, 8)
        vx, vy, vz = curl_c(Px, Py, Pz, dx, ndim)
        s = 0.5 / _rms(vx, vy, vz)
        W[1], W[2], W[3] = vx * s, vy * s, vz * s
        del Px, Py, Pz, vx, vy, vz
        Ax, Ay, Az = F(32, 8), F(32, 8), F(32, 8)
        bx, by, bz = curl_c(Ax, Ay, Az, dx, ndim)
        s = 0.3 / _rms(bx, by, bz)
        W[5], W[6], W[7] = bx * s, by * s, bz * s
        W[4] = 1.0
    else:
        raise ValueError(f"unknown config {config_id}")

    d_i = c["d_i"]
    if config_id in (4, 8) and scale_d_i and n != nfull:
        d_i = d_i * nfull / n
    U = prim_to_cons_cgl(W) if c["eqset"] in (CGL, CGL_GLM) else prim_to_cons(W, g)
    return Workload(config_id=config_id, ndim=ndim, shape=shape, dx=dx, gamma=g, eqset=c["eqset"],
                    riemann=c["riemann"], limiter=2, beta=c["beta"], rk=2, cfl=c["cfl"], d_i=d_i,
                    n_steps=c["n_steps"] if n_steps is None else n_steps, W=W, U=U, relax=c.get("relax", 0.0),
                    name=c["name"] + (f" @n={n}" if n != nfull else ""))


def random_state(seed: int, shape, ndim: int, gamma: float = GAMMA, amp: float = 0.3):
    """Random strictly positive state for brute-force / tiny-grid tests: rho, p in [0.5, 1.5],
    v and B components uniform in [-amp, amp].  Returns (W, U) as [8, nz, ny, nx]."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = shape
    W = np.empty((NVAR, nz, ny, nx))
    W[0] = 0.5 + rng.random((nz, ny, nx))
    W[4] = 0.5 + rng.random((nz, ny, nx))
    for q in (1, 2, 3, 5, 6, 7):
        W[q] = amp * (2.0 * rng.random((nz, ny, nx)) - 1.0)
    return W, prim_to_cons(W, gamma)
