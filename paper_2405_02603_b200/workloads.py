"""Seeded synthetic inputs shaped like the paper's workloads and the
BASELINE.json configs.  Shared by the tests, the oracle legs and bench.py.

This module holds NONE of the method's arithmetic (no Green's function, no FFT, no convolution):
it only samples analytic charge densities on the mesh.  numpy only; everything is fp64 and
deterministic given the seed (numpy ``default_rng`` = PCG64).  Recipe stated in DESIGN.md
("Input recipe").

Sampling: cell centres, x_i = x_min + (i + 1/2) h   (reading R3).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    name: str
    N: tuple            # (Nx, Ny, Nz)
    lo: tuple           # lower corner of the box
    hi: tuple           # upper corner of the box
    rho: np.ndarray     # (Nx, Ny, Nz) fp64, C order
    # parameters of the analytic density, so tests can build the closed-form potential:
    # list of (amplitude, centre(3), sigma(3)) for whole Gaussians; noise is not in the list.
    gaussians: list = field(default_factory=list)
    noise_rel: float = 0.0
    seed: int | None = None

    @property
    def h(self):
        return tuple((b - a) / n for a, b, n in zip(self.lo, self.hi, self.N))


def cell_centres(N, lo, hi):
    """Three 1-D coordinate vectors of the cell centres."""
    return tuple(lo[d] + (np.arange(N[d], dtype=np.float64) + 0.5) * ((hi[d] - lo[d]) / N[d])
                 for d in range(3))


def gaussian_density(N, lo, hi, centre, sigma, amplitude=1.0):
    """amplitude * normalised 3-D Gaussian exp(-sum (x-c)^2/(2 s^2)) / ((2 pi)^{3/2} sx sy sz).

    DESIGN.md reading R1 of PAPER.md Eq. 4 (normalised, positive).  Separable, so built from three
    1-D factors.
    """
    sig = np.broadcast_to(np.asarray(sigma, dtype=np.float64), (3,))
    xs = cell_centres(N, lo, hi)
    f = [np.exp(-((xs[d] - centre[d]) ** 2) / (2.0 * sig[d] ** 2)) / (math.sqrt(2.0 * math.pi) * sig[d])
         for d in range(3)]
    return amplitude * f[0][:, None, None] * f[1][None, :, None] * f[2][None, None, :]


def config1(N=16):
    """16^3 (or N^3), unit cube [-1/2,1/2]^3, one normalised Gaussian at the origin, sigma = 0.05."""
    N3, lo, hi = (N, N, N), (-0.5,) * 3, (0.5,) * 3
    g = [(1.0, (0.0, 0.0, 0.0), (0.05,) * 3)]
    rho = gaussian_density(N3, lo, hi, g[0][1], g[0][2])
    return Workload(f"gaussian_{N}^3", N3, lo, hi, np.ascontiguousarray(rho), g)


def config2(N=64, seed=1):
    """64^3 unit cube; sum of 4 Gaussians; centres U[-0.2,0.2]^3, sigma U[0.03,0.08], amplitude
    U[0.5,1.5] x random sign.  Draw order: centres, sigmas, magnitudes, signs."""
    rng = np.random.default_rng(seed)
    N3, lo, hi = (N, N, N), (-0.5,) * 3, (0.5,) * 3
    centres = rng.uniform(-0.2, 0.2, size=(4, 3))
    sigmas = rng.uniform(0.03, 0.08, size=4)
    mags = rng.uniform(0.5, 1.5, size=4)
    signs = rng.choice([-1.0, 1.0], size=4)
    rho = np.zeros(N3, dtype=np.float64)
    gs = []
    for c, s, m, sg in zip(centres, sigmas, mags, signs):
        gs.append((float(m * sg), tuple(float(v) for v in c), (float(s),) * 3))
        rho += gaussian_density(N3, lo, hi, c, s, m * sg)
    return Workload(f"multigauss_{N}^3_seed{seed}", N3, lo, hi, np.ascontiguousarray(rho), gs, seed=seed)


def config3(N=256, seed=4, noise_rel=1e-6):
    """256^3 unit cube; Gaussian sigma = 0.05 plus uniform noise U[-1,1) * 1e-6 * max(rho) per cell."""
    w = config1(N)
    rng = np.random.default_rng(seed)
    peak = float(w.rho.max())
    # generated plane by plane to bound the temporary
    for i in range(N):
        w.rho[i] += (rng.random((N, N)) * 2.0 - 1.0) * (noise_rel * peak)
    w.name, w.noise_rel, w.seed = f"gaussian+noise_{N}^3_seed{seed}", noise_rel, seed
    return w


def config4(N=(128, 128, 512)):
    """Anisotropic grid, box [-1/2,1/2]^2 x [-2,2]; beam-like Gaussian sx = sy = 0.05, sz = 0.5."""
    lo, hi = (-0.5, -0.5, -2.0), (0.5, 0.5, 2.0)
    g = [(1.0, (0.0, 0.0, 0.0), (0.05, 0.05, 0.5))]
    rho = gaussian_density(N, lo, hi, g[0][1], g[0][2])
    return Workload(f"beam_{N[0]}x{N[1]}x{N[2]}", tuple(N), lo, hi, np.ascontiguousarray(rho), g)


def config5(N=512):
    """512^3 unit cube, Gaussian sigma = 0.05."""
    return config1(N)


def random_density(N, seed=0):
    """Dense U[-1,1) field on a unit-spacing-agnostic box (for brute-force parity on small grids,
    including ragged / non-cubic shapes).  Box is [0,1]^3 scaled so that h is not 1."""
    rng = np.random.default_rng(seed)
    N = tuple(int(v) for v in N)
    rho = rng.random(N) * 2.0 - 1.0
    return Workload(f"random_{N[0]}x{N[1]}x{N[2]}_seed{seed}", N, (0.0,) * 3, (1.0, 1.25, 0.75),
                    np.ascontiguousarray(rho), [], seed=seed)
