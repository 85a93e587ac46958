"""Seeded synthetic inputs for the coupled ACM lattice-Boltzmann step.

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench).
It holds none of the method's arithmetic: it only builds the initial phase field
phi and velocity u that are handed to ``acm_init`` / ``oracle_init``, plus the
table of scalar parameters of each workload.

The workloads stand in for the paper's own simulation set-ups (PAPER.md P:283
"gas bubble in the middle ... R = 65", P:388 rising bubble 256x1024x256, R=16,
P:433 bubble field with R=16 +- R/5); no external dataset is involved.

Recipe (restated in DESIGN.md):
  * cell (i,j,k) has its centre at (i+1/2, j+1/2, k+1/2); distances use the
    minimal image on periodic axes;
  * a sphere of radius R: phi = 1/2 -+ 1/2 tanh(2 (d-R)/xi)  (the paper's
    equilibrium profile eq. 3 P:70 used as an initial condition; '-' outside
    sign for a heavy droplet (phi=1 inside), '+' for a light bubble (phi=0 inside));
  * bubble sets: numpy PCG64 seed 2012; draw c~U[0,L)^3, R~U[Rmin,Rmax]; accept
    iff distance to every accepted centre >= R+Rj+2 xi;
    phi = 1/2 + 1/2 tanh(2 min_b(d_b - R_b)/xi);
  * velocity noise: numpy PCG64 seed 6144, each component i.i.d. U[-1e-3,1e-3].

Array layout handed to the ABI: x fastest, i.e. numpy shape (nz, ny, nx) for phi
and (3, nz, ny, nx) for u (component-major), C-contiguous float64.
"""
from __future__ import annotations

import dataclasses
from typing import Optional, Sequence, Tuple

import numpy as np

WALL_X, WALL_Y, WALL_Z = 1, 2, 4
SEED_BUBBLES = 2012
SEED_VELOCITY = 6144


@dataclasses.dataclass(frozen=True)
class Params:
    """Scalar arguments of acm_create (PAPER.md P:283 benchmark parameters)."""
    nx: int
    ny: int
    nz: int
    stencil_phase: int = 15
    stencil_hydro: int = 19
    rho_H: float = 1.0
    rho_L: float = 1.0e-3
    sigma: float = 1.0e-4
    xi: float = 5.0
    M: float = 0.02
    nu_H: float = 1.0 / 60.0
    nu_L: float = 1.0 / 60.0
    gravity: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    wall_flags: int = 0
    phase_srt: bool = False      # SRT phase-field collision (the paper's benchmark scheme)

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def ncells(self):
        return self.nx * self.ny * self.nz

    def replace(self, **kw):
        return dataclasses.replace(self, **kw)


def cell_centres(p: Params):
    """Coordinates of the cell centres as broadcastable (nz,ny,nx) arrays."""
    x = (np.arange(p.nx, dtype=np.float64) + 0.5)[None, None, :]
    y = (np.arange(p.ny, dtype=np.float64) + 0.5)[None, :, None]
    z = (np.arange(p.nz, dtype=np.float64) + 0.5)[:, None, None]
    return x, y, z


def _distance(p: Params, centre: Sequence[float]):
    """Distance of every cell centre to `centre`, minimal image on periodic axes."""
    x, y, z = cell_centres(p)
    d2 = 0.0
    for coord, c, L, wall in ((x, centre[0], p.nx, p.wall_flags & WALL_X),
                              (y, centre[1], p.ny, p.wall_flags & WALL_Y),
                              (z, centre[2], p.nz, p.wall_flags & WALL_Z)):
        d = np.abs(coord - c)
        if not wall:
            d = np.minimum(d, L - d)
        d2 = d2 + d * d
    return np.sqrt(d2)


def sphere_phi(p: Params, centre: Sequence[float], R: float, heavy_inside: bool):
    """Single sphere with the tanh profile of eq. 3."""
    d = _distance(p, centre)
    s = np.tanh(2.0 * (d - R) / p.xi)
    phi = 0.5 - 0.5 * s if heavy_inside else 0.5 + 0.5 * s
    return np.ascontiguousarray(np.broadcast_to(phi, p.shape), dtype=np.float64)


def bubble_set(p: Params, count: int, r_min: float, r_max: float, seed: int = SEED_BUBBLES):
    """Seeded non-overlapping light bubbles; returns (centres[count,3], radii[count])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    L = np.array([p.nx, p.ny, p.nz], dtype=np.float64)
    centres, radii = [], []
    tries = 0
    while len(centres) < count:
        tries += 1
        if tries > 1000 * count:
            raise RuntimeError("bubble_set: rejection sampling did not converge")
        c = rng.uniform(0.0, 1.0, size=3) * L
        R = rng.uniform(r_min, r_max)
        ok = True
        for cj, Rj in zip(centres, radii):
            d = np.abs(c - cj)
            d = np.minimum(d, L - d)
            if np.sqrt((d * d).sum()) < R + Rj + 2.0 * p.xi:
                ok = False
                break
        if ok:
            centres.append(c)
            radii.append(R)
    return np.array(centres), np.array(radii)


def bubbles_phi(p: Params, centres, radii):
    """phi = 1/2 + 1/2 tanh(2 min_b(d_b - R_b)/xi): light bubbles in heavy liquid.

    Each bubble only touches the cells within R + 12 xi of its centre: beyond that
    tanh(2 (d-R)/xi) = tanh(24) rounds to exactly 1.0 in fp64, which is also what the
    untouched cells get (min over an empty set = +inf), so the result equals the full min."""
    dmin = np.full(p.shape, np.inf)
    n = (p.nx, p.ny, p.nz)
    for c, R in zip(centres, radii):
        reach = R + 12.0 * p.xi
        idx, dist2 = [], []
        for a in range(3):
            lo, hi = int(np.floor(c[a] - reach)) - 1, int(np.ceil(c[a] + reach)) + 1
            if hi - lo >= n[a]:
                lo, hi = 0, n[a]
            ia = np.arange(lo, hi) % n[a]
            d = np.abs(ia + 0.5 - c[a])
            d = np.minimum(d, n[a] - d)
            idx.append(ia)
            dist2.append(d * d)
        sub = np.ix_(idx[2], idx[1], idx[0])
        d = np.sqrt(dist2[2][:, None, None] + dist2[1][None, :, None] + dist2[0][None, None, :]) - R
        dmin[sub] = np.minimum(dmin[sub], d)
    return 0.5 + 0.5 * np.tanh(2.0 * dmin / p.xi)


def velocity_noise(p: Params, amplitude: float = 1.0e-3, seed: int = SEED_VELOCITY):
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(-amplitude, amplitude, size=(3,) + p.shape)


def zeros_u(p: Params):
    return np.zeros((3,) + p.shape, dtype=np.float64)


# ----------------------------------------------------------------------------
# The five BASELINE.json configurations (and scaled-down variants for parity).
# ----------------------------------------------------------------------------

def config1(n: int = 32, R: Optional[float] = None):
    """Static heavy droplet, fully periodic, D3Q15 phase + D3Q19 hydro."""
    p = Params(nx=n, ny=n, nz=n)
    R = n / 4.0 if R is None else R
    phi = sphere_phi(p, (n / 2.0, n / 2.0, n / 2.0), R, heavy_inside=True)
    return p, phi, zeros_u(p)


def config2(nx: int = 128, ny: int = 512, nz: int = 128, R: float = 16.0, gy: float = -1.0e-6,
            centre: Optional[Sequence[float]] = None):
    """Rising light bubble between half-way bounce-back walls in y, gravity in -y."""
    p = Params(nx=nx, ny=ny, nz=nz, gravity=(0.0, gy, 0.0), wall_flags=WALL_Y)
    centre = (nx / 2.0, 64.0 * ny / 512.0, nz / 2.0) if centre is None else centre
    phi = sphere_phi(p, centre, R, heavy_inside=False)
    return p, phi, zeros_u(p)


def config3(n: int = 256, count: int = 64, r_min: float = 8.0, r_max: float = 14.0,
            stencil_phase: int = 15, stencil_hydro: int = 19, noise: float = 1.0e-3):
    """Headline: seeded bubble field + seeded velocity noise, fully periodic."""
    p = Params(nx=n, ny=n, nz=n, stencil_phase=stencil_phase, stencil_hydro=stencil_hydro)
    c, r = bubble_set(p, count, r_min, r_max)
    phi = bubbles_phi(p, c, r)
    u = velocity_noise(p, noise) if noise > 0 else zeros_u(p)
    return p, phi, u


def config4(n: int = 512, count: int = 512):
    p = Params(nx=n, ny=n, nz=n)
    c, r = bubble_set(p, count, 10.0, 16.0)
    return p, bubbles_phi(p, c, r), zeros_u(p)


def config5(n: int = 256, count: int = 64):
    return config3(n=n, count=count, stencil_phase=27, stencil_hydro=27)


def paper_benchmark(n: int = 260, R: Optional[float] = None):
    """The paper's own single-GPU benchmark: n^3 = 260^3 cells, fully periodic, one gas bubble
    (rho_L = 0.001) of radius 65 in the middle of liquid (rho_H = 1), M = 0.02, xi = 5, sigma = 1e-4,
    "relaxation time tau = 0.53" (read as the usual tau including the 1/2: nu = (0.53 - 0.5)/3 = 0.01,
    SURVEY A21), no force, D3Q15 SRT phase field + D3Q27 MRT hydrodynamics."""
    R = n / 4.0 if R is None else R
    p = Params(nx=n, ny=n, nz=n, stencil_phase=15, stencil_hydro=27, nu_H=0.01, nu_L=0.01, phase_srt=True)
    phi = sphere_phi(p, (n / 2.0, n / 2.0, n / 2.0), R, heavy_inside=False)
    return p, phi, zeros_u(p)


def disc2d(n: int = 4096, count: int = 64, r_min: float = 40.0, r_max: float = 80.0, noise: float = 1.0e-3):
    """Two-dimensional instance (D2Q9 + D2Q9, one plane; the paper's Fig. 5 measures D2Q9): seeded light
    discs in heavy liquid on an n x n periodic grid, same recipe as config 3 (centres in the plane z = 1/2)."""
    p = Params(nx=n, ny=n, nz=1, stencil_phase=9, stencil_hydro=9)
    rng = np.random.Generator(np.random.PCG64(SEED_BUBBLES))
    centres, radii = [], []
    while len(centres) < count:
        c = np.array([rng.uniform(0, n), rng.uniform(0, n), 0.5])
        R = rng.uniform(r_min, r_max)
        d = np.abs(np.array(centres).reshape(-1, 3) - c)[:, :2] if centres else np.zeros((0, 2))
        d = np.minimum(d, n - d)
        if all(np.sqrt((d * d).sum(1)) >= R + np.array(radii) + 2.0 * p.xi):
            centres.append(c)
            radii.append(R)
    phi = bubbles_phi(p, np.array(centres), np.array(radii))
    u = velocity_noise(p, noise) if noise > 0 else zeros_u(p)
    u[2] = 0.0
    return p, phi, u


def scaled_config3(n: int, stencil_phase: int = 15, stencil_hydro: int = 19):
    """Config-3-like input on a small grid: bubble count and radii scaled so that
    the volume fraction and the interface structure stay comparable."""
    count = max(1, int(round(64 * (n / 256.0) ** 3 * 8)))  # radii are halved below => x8 in count
    return config3(n=n, count=count, r_min=4.0, r_max=7.0,
                   stencil_phase=stencil_phase, stencil_hydro=stencil_hydro)
