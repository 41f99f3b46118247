"""Closed-form potentials used as pins (test-side mathematics, independent of oracle and CUDA path).

PAPER.md:108-116: potential of a normalised Gaussian charge (Delta phi = -rho, eps0 = 1):
    phi(r) = erf(r / (sqrt(2) sigma)) / (4 pi r),   phi(0) = sqrt(2/pi) / (4 pi sigma).
Anisotropic Gaussian (not in the paper; standard one-dimensional integral):
    phi(x) = (1/4pi) (2/sqrt(pi)) int_0^inf prod_d (1 + 2 s_d^2 t^2)^(-1/2)
                                   exp(-t^2 x_d^2 / (1 + 2 s_d^2 t^2)) dt.
"""
import math

import numpy as np
from scipy.special import erf

from paper_2405_02603_b200 import workloads as W


def gaussian_potential_iso(w: W.Workload) -> np.ndarray:
    """Superposition of isotropic-Gaussian closed forms for every Gaussian listed in the workload."""
    xs = W.cell_centres(w.N, w.lo, w.hi)
    phi = np.zeros(w.N, dtype=np.float64)
    for amp, c, sig in w.gaussians:
        assert sig[0] == sig[1] == sig[2]
        r = np.sqrt((xs[0][:, None, None] - c[0]) ** 2 + (xs[1][None, :, None] - c[1]) ** 2
                    + (xs[2][None, None, :] - c[2]) ** 2)
        with np.errstate(divide="ignore", invalid="ignore"):
            p = erf(r / (math.sqrt(2.0) * sig[0])) / (4.0 * math.pi * r)
        p = np.where(r == 0.0, math.sqrt(2.0 / math.pi) / (4.0 * math.pi * sig[0]), p)
        phi += amp * p
    return phi


def gaussian_potential_aniso_points(sig, pts: np.ndarray, nquad: int = 4000) -> np.ndarray:
    """The 1-D integral above at a list of points (npts, 3), Gauss-Legendre on t = u/(1-u)."""
    u, wu = np.polynomial.legendre.leggauss(nquad)
    u = 0.5 * (u + 1.0)
    wu = 0.5 * wu
    t = u / (1.0 - u)
    dt = wu / (1.0 - u) ** 2
    out = np.empty(len(pts))
    for i, x in enumerate(pts):
        f = np.ones_like(t)
        for d in range(3):
            q = 1.0 + 2.0 * sig[d] ** 2 * t ** 2
            f *= np.exp(-(t ** 2) * x[d] ** 2 / q) / np.sqrt(q)
        out[i] = (1.0 / (4.0 * math.pi)) * (2.0 / math.sqrt(math.pi)) * np.sum(f * dt)
    return out


def rel_l2(a: np.ndarray, b: np.ndarray) -> float:
    """PAPER.md:135 'relative error L2 norm': ||a-b||_2 / ||b||_2 over all points."""
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def rel_max(a: np.ndarray, b: np.ndarray) -> float:
    """Max-norm relative error max|a-b| / max|b| (reading R14)."""
    return float(np.abs(a - b).max() / np.abs(b).max())


def gaussian_field_iso(w: W.Workload) -> np.ndarray:
    """E = -grad phi of the closed form above (Eq. A.1), shape (3, Nx, Ny, Nz):
        E(r) = (x / r) [ erf(r / (sqrt(2) s)) / r^2 - sqrt(2/pi) exp(-r^2 / (2 s^2)) / (s r) ] / (4 pi),  E(0) = 0.
    """
    xs = W.cell_centres(w.N, w.lo, w.hi)
    E = np.zeros((3,) + tuple(w.N), dtype=np.float64)
    for amp, c, sig in w.gaussians:
        assert sig[0] == sig[1] == sig[2]
        s = sig[0]
        d = [xs[0][:, None, None] - c[0], xs[1][None, :, None] - c[1], xs[2][None, None, :] - c[2]]
        r = np.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2)
        with np.errstate(divide="ignore", invalid="ignore"):
            er = (erf(r / (math.sqrt(2.0) * s)) / r ** 2
                  - math.sqrt(2.0 / math.pi) * np.exp(-r ** 2 / (2.0 * s * s)) / (s * r)) / (4.0 * math.pi)
            for a in range(3):
                E[a] += amp * np.where(r == 0.0, 0.0, er * d[a] / r)
    return E
