"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests) and the CUDA path. It holds none of the
method's arithmetic (no stencils, no Z4c terms, no RK update, no enforcement): it only writes
initial data -- closed-form expressions evaluated at cell centres -- and parameter sets.

Layout of every array returned: float64 [22][Nz][Ny][Nx] in GLOBAL (block-free) cell order,
x fastest; cell centres x_i = xmin + (i + 1/2) dx (cell-centred grid).

Field order (BASELINE.json north_star (a)): 0 chi; 1-6 gt_xx,xy,xz,yy,yz,zz; 7 Khat;
8-13 At_xx..zz; 14-16 Gamt^x,y,z; 17 Theta; 18 alpha; 19-21 beta^x,y,z.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Tuple

import numpy as np

NF = 22
CHI, GXX, GXY, GXZ, GYY, GYZ, GZZ, KHAT = range(8)
AXX, AXY, AXZ, AYY, AYZ, AZZ = range(8, 14)
GAMX, GAMY, GAMZ, THETA, ALPHA, BETAX, BETAY, BETAZ = range(14, 22)
FIELD_NAMES = ["chi", "gxx", "gxy", "gxz", "gyy", "gyz", "gzz", "Khat",
               "Axx", "Axy", "Axz", "Ayy", "Ayz", "Azz", "Gamx", "Gamy", "Gamz",
               "Theta", "alpha", "betax", "betay", "betaz"]


@dataclass(frozen=True)
class Z4cParams:
    """Mirror of `z4c_params` in include/z4c.h (same member order)."""
    n: int = 16                       # interior cells per block edge
    ng: int = 3                       # ghosts (4th order: PAPER.md:124 rule, reading Q1)
    nb: Tuple[int, int, int] = (1, 1, 1)   # block lattice (x, y, z)
    xmin: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    dx: float = 0.1
    bc: int = 0                       # 0 periodic, 1 outflow-copy
    cfl: float = 0.25
    kappa1: float = 0.02
    kappa2: float = 0.0
    lapse_oplog: float = 2.0          # 1+log
    lapse_harmonic: float = 0.0
    lapse_advect: float = 1.0
    shift_gamma: float = 1.0          # Q6
    shift_eta: float = 2.0
    shift_advect: float = 1.0
    ko_eps: float = 0.5
    chi_floor: float = 1e-6           # Q8

    @property
    def N(self) -> Tuple[int, int, int]:
        return (self.n * self.nb[0], self.n * self.nb[1], self.n * self.nb[2])

    @property
    def ncells(self) -> int:
        N = self.N
        return N[0] * N[1] * N[2]

    @property
    def nblocks(self) -> int:
        return self.nb[0] * self.nb[1] * self.nb[2]

    @property
    def dt(self) -> float:
        return self.cfl * self.dx


def cell_centres(p: Z4cParams):
    """(z, y, x) broadcastable coordinate arrays of the cell centres."""
    N = p.N
    x = p.xmin[0] + (np.arange(N[0], dtype=np.float64) + 0.5) * p.dx
    y = p.xmin[1] + (np.arange(N[1], dtype=np.float64) + 0.5) * p.dx
    z = p.xmin[2] + (np.arange(N[2], dtype=np.float64) + 0.5) * p.dx
    return z[:, None, None], y[None, :, None], x[None, None, :]


def minkowski(p: Z4cParams) -> np.ndarray:
    N = p.N
    u = np.zeros((NF, N[2], N[1], N[0]), dtype=np.float64)
    u[CHI] = 1.0
    u[GXX] = 1.0
    u[GYY] = 1.0
    u[GZZ] = 1.0
    u[ALPHA] = 1.0
    return u


# ---- configs 1 and 5: Minkowski + seeded uniform noise --------------------------------
def params_noise(n: int = 16, nb=(1, 1, 1), dx: float = 0.1) -> Z4cParams:
    """1+log slicing, Gamma-driver eta=2, KO 0.5, CFL 0.25, periodic (BASELINE.json configs[0], [4])."""
    return Z4cParams(n=n, nb=tuple(nb), dx=dx, bc=0, shift_eta=2.0)


def noise_data(p: Z4cParams, seed: int = 1234, amplitude: float = 1e-10) -> np.ndarray:
    """Uniform noise in [-amplitude, amplitude] on all 22 fields, PCG64(seed), drawn in
    [F][z][y][x] order (O8)."""
    N = p.N
    rng = np.random.Generator(np.random.PCG64(seed))
    noise = rng.uniform(-amplitude, amplitude, size=(NF, N[2], N[1], N[0]))
    return minkowski(p) + noise


def tiled_noise_data(p: Z4cParams, tile_nb=(2, 2, 2), seed: int = 1000,
                     amplitude: float = 1e-10) -> np.ndarray:
    """Config 5 at scale: an (tile_nb * n)^3 noise problem repeated periodically to fill the pack
    (periodic-tiling invariance)."""
    small = replace(p, nb=tuple(tile_nb))
    base = noise_data(small, seed, amplitude)
    reps = (1, p.nb[2] // tile_nb[2], p.nb[1] // tile_nb[1], p.nb[0] // tile_nb[0])
    assert all(p.nb[a] % tile_nb[a] == 0 for a in range(3))
    return np.tile(base, reps)


# ---- config 2: linear gravitational wave along x -----------------------------------------
def params_linear_wave(N: int = 64, n: int = 16) -> Z4cParams:
    """Harmonic lapse, frozen zero shift, periodic unit cube (BASELINE.json configs[1])."""
    assert N % n == 0
    nb = N // n
    return Z4cParams(n=n, nb=(nb, nb, nb), xmin=(0.0, 0.0, 0.0), dx=1.0 / N, bc=0,
                     lapse_oplog=0.0, lapse_harmonic=1.0, lapse_advect=0.0,
                     shift_gamma=0.0, shift_eta=0.0, shift_advect=0.0)


def linear_wave_data(p: Z4cParams, t: float = 0.0, A: float = 1e-8, lam: float = 1.0) -> np.ndarray:
    """TT plane wave b = A sin(2 pi (x - t)/lam): gamma_ij = diag(1, 1+b, 1-b),
    K_ij = -1/2 d_t gamma_ij, alpha = 1, beta = 0, converted exactly to conformal variables (O8).
    Evaluated at time t this is also the analytic solution (to O(A^2))."""
    _, _, x = cell_centres(p)
    N = p.N
    shape = (N[2], N[1], N[0])
    ph = 2.0 * math.pi * (x - t) / lam
    b = A * np.sin(ph)
    db = A * (2.0 * math.pi / lam) * np.cos(ph)       # db/dx ; d_t b = -db
    det = 1.0 - b * b
    chi = det ** (-1.0 / 3.0)
    Kyy = 0.5 * db                                     # K_yy = -1/2 d_t(1+b) = +1/2 db/dx
    Kzz = -0.5 * db
    K = Kyy / (1.0 + b) + Kzz / (1.0 - b)
    u = np.zeros((NF,) + shape, dtype=np.float64)
    u[CHI] = np.broadcast_to(chi, shape)
    u[GXX] = np.broadcast_to(chi, shape)
    u[GYY] = np.broadcast_to(chi * (1.0 + b), shape)
    u[GZZ] = np.broadcast_to(chi * (1.0 - b), shape)
    u[KHAT] = np.broadcast_to(K, shape)
    u[AXX] = np.broadcast_to(chi * (-K / 3.0), shape)
    u[AYY] = np.broadcast_to(chi * (Kyy - (1.0 + b) * K / 3.0), shape)
    u[AZZ] = np.broadcast_to(chi * (Kzz - (1.0 - b) * K / 3.0), shape)
    # Gamt^x = -d_x gt^xx = -d_x (1/chi) = 2/3 b b' (1-b^2)^(-2/3)
    u[GAMX] = np.broadcast_to((2.0 / 3.0) * b * db * det ** (-2.0 / 3.0), shape)
    u[ALPHA] = 1.0
    return u


# ---- configs 3 and 4: punctures --------------------------------------------------------
def params_puncture(N: int = 128, n: int = 32, half_width: float = 16.0, eta: float = 2.0) -> Z4cParams:
    """1+log, Gamma-driver, outflow-copy (BASELINE.json configs[2]; configs[3] with N=256, 24, eta=1)."""
    assert N % n == 0
    nb = N // n
    return Z4cParams(n=n, nb=(nb, nb, nb), xmin=(-half_width,) * 3, dx=2.0 * half_width / N, bc=1,
                     shift_eta=eta)


def puncture_data(p: Z4cParams, masses=(1.0,), positions=((0.0, 0.0, 0.0),)) -> np.ndarray:
    """Brill-Lindquist psi = 1 + sum m_i / (2 r_i); chi = psi^-4, gt = delta, alpha = psi^-2 (O8)."""
    z, y, x = cell_centres(p)
    psi = 1.0
    for m, c in zip(masses, positions):
        r = np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2)
        psi = psi + m / (2.0 * r)
    u = minkowski(p)
    u[CHI] = psi ** -4.0
    u[ALPHA] = psi ** -2.0
    return u


def config(idx: int):
    """(params, initial data, nsteps) of BASELINE.json configs[idx] at full size."""
    if idx == 0:
        p = params_noise(16, (1, 1, 1), 0.1)
        return p, noise_data(p, 1234), 10
    if idx == 1:
        p = params_linear_wave(64, 16)
        return p, linear_wave_data(p), 100
    if idx == 2:
        p = params_puncture(128, 32, 16.0, 2.0)
        return p, puncture_data(p, (1.0,), ((0.0, 0.0, 0.0),)), 200
    if idx == 3:
        p = params_puncture(256, 32, 24.0, 1.0)
        return p, puncture_data(p, (0.5, 0.5), ((3.0, 0.0, 0.0), (-3.0, 0.0, 0.0))), 100
    raise ValueError("config 4 (load sweep) is parameterised: use params_noise + tiled_noise_data")


# ---- generic strong-field test data (parity tests; not a BASELINE config) ------------------
def smooth_random_data(p: Z4cParams, seed: int = 7, amplitude: float = 0.1, nmodes: int = 3) -> np.ndarray:
    """Minkowski + a few random Fourier modes of the given amplitude on every field (periodic over the
    domain, so usable with either boundary condition). All nonlinear terms, both upwind directions and all
    tensor components are exercised; det(gt) stays > 0 for amplitude <~ 0.2."""
    rng = np.random.Generator(np.random.PCG64(seed))
    z, y, x = cell_centres(p)
    N = p.N
    L = [N[a] * p.dx for a in range(3)]
    xs = [(x - p.xmin[0]) / L[0], (y - p.xmin[1]) / L[1], (z - p.xmin[2]) / L[2]]
    u = minkowski(p)
    for f in range(NF):
        acc = np.zeros((N[2], N[1], N[0]))
        for _ in range(nmodes):
            k = rng.integers(-2, 3, size=3)
            ph = rng.uniform(0.0, 2.0 * math.pi)
            c = rng.uniform(-1.0, 1.0)
            acc = acc + c * np.sin(2.0 * math.pi * (k[0] * xs[0] + k[1] * xs[1] + k[2] * xs[2]) + ph)
        u[f] += (amplitude / nmodes) * acc
    return u
