"""ctypes marshalling for ``fsp_oracle.c`` (TEST INFRASTRUCTURE -- see ``oracle/__init__.py``).

Every function but one checks shapes, hands contiguous numpy fp64 arrays to the C oracle and returns the
result.  The exception is ``field_of_point_charges``: an FFT-free, point-by-point numpy evaluation of the field
of a few point charges (oracle-side arithmetic, pinned in tests/test_oracle_pins.py against orc_solve_field).
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
import threading

import numpy as np

HOCKNEY, VICO, VICO_2 = 0, 1, 2  # PAPER.md:199 solver names HOCKNEY / VICO / VICO_2
VICO_SAFE = 3  # VICO_2 with per-axis oversampling m_d >= 1 + L/L_d (R17)
G0_DEFAULT = 1.0 / (4.0 * math.pi)  # DESIGN.md reading R5
ALPHA_DEFAULT = 1.1

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fsp_oracle.c")
_LIB = os.path.join(_HERE, "libfsp_oracle.so")
_lock = threading.Lock()
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_lp = ctypes.POINTER(ctypes.c_long)


def build(force: bool = False) -> str:
    """Compile fsp_oracle.c with gcc (-O2 -fopenmp).  Returns the path of the shared object."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        L, I, D = ctypes.c_long, ctypes.c_int, ctypes.c_double
        lib.orc_num_threads.restype = I
        lib.orc_set_num_threads.argtypes = [I]
        lib.orc_set_num_threads.restype = None
        lib.orc_fft1d.argtypes = [L, _dp, _dp, I, I]
        lib.orc_fft3d.argtypes = [L, L, L, _dp, I, I]
        lib.orc_dct1.argtypes = [L, L, _dp, _dp, I]
        lib.orc_vg_window.argtypes = [L, L, L, _dp, D]
        lib.orc_vg_window.restype = D
        lib.orc_green_table_he.argtypes = [L, L, L, _dp, D, _dp]
        lib.orc_green_table_vg.argtypes = [L, L, L, _dp, D, I, _dp]
        lib.orc_green_table_vg2.argtypes = [L, L, L, _dp, D, I, _dp]
        lib.orc_green_table_vgm.argtypes = [L, L, L, _dp, D, I, _lp, _dp]
        lib.orc_vg_safe_factors.argtypes = [L, L, L, _dp, D, _lp]
        lib.orc_green_spectrum.argtypes = [L, L, L, _dp, I, _dp]
        lib.orc_solve.argtypes = [L, L, L, _dp, _dp, I, _dp, _dp]
        lib.orc_solve_field.argtypes = [L, L, L, _dp, _dp, I, _dp, _dp, _dp]
        lib.orc_direct_sum.argtypes = [L, L, L, _dp, _dp, _dp, L, _lp, _dp]
        lib.orc_green_table_vg_entries.argtypes = [L, L, L, _dp, D, _lp, L, _lp, _dp]
        _ip = ctypes.POINTER(ctypes.c_int)
        lib.orc_solve_mixed.argtypes = [L, L, L, _dp, _dp, _ip, I, _dp, _dp]
        lib.orc_direct_sum_mixed.argtypes = [L, L, L, _dp, _dp, _ip, _dp, L, _lp, _dp]
        _lib = lib
    return _lib


def _check(rc: int, what: str) -> None:
    if rc == -2:
        raise MemoryError(f"oracle {what}: out of memory")
    if rc != 0:
        raise ValueError(f"oracle {what}: invalid argument (rc={rc})")


def _d(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _h3(h) -> np.ndarray:
    h = np.ascontiguousarray(np.broadcast_to(np.asarray(h, dtype=np.float64), (3,)))
    return h


def num_threads() -> int:
    return int(_load().orc_num_threads())


def set_num_threads(n: int) -> None:
    _load().orc_set_num_threads(int(n))


def fft1d(x: np.ndarray, sign: int = -1, method: int = 0) -> np.ndarray:
    """Unscaled 1-D DFT of a complex vector; method 0 = radix-2 (direct if not 2^k), 1 = direct."""
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    _check(_load().orc_fft1d(x.size, _d(x.view(np.float64)), _d(out.view(np.float64)), sign, method),
           "fft1d")
    return out


def fft3d(a: np.ndarray, sign: int = -1, method: int = 0) -> np.ndarray:
    """Unscaled separable 3-D DFT (returns a new array)."""
    a = np.array(a, dtype=np.complex128, order="C", copy=True)
    assert a.ndim == 3
    _check(_load().orc_fft3d(a.shape[0], a.shape[1], a.shape[2], _d(a.view(np.float64)), sign, method),
           "fft3d")
    return a


def dct1(x: np.ndarray, nout: int | None = None, method: int = 1) -> np.ndarray:
    """Un-normalised DCT-I (REDFT00 convention) of n+1 reals, first nout outputs."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    n = x.size - 1
    nout = n + 1 if nout is None else nout
    out = np.empty(nout, dtype=np.float64)
    _check(_load().orc_dct1(n, nout, _d(x), _d(out), method), "dct1")
    return out


def vg_window(N, h, alpha: float = ALPHA_DEFAULT) -> float:
    h = _h3(h)
    return float(_load().orc_vg_window(N[0], N[1], N[2], _d(h), alpha))


def vg_safe_factors(N, h, alpha: float = ALPHA_DEFAULT):
    """Per-axis oversampling factors of VICO_SAFE: 4, doubled while m_d < 1 + L/L_d (R17)."""
    h = _h3(h)
    m = np.zeros(3, dtype=np.int64)
    _check(_load().orc_vg_safe_factors(int(N[0]), int(N[1]), int(N[2]), _d(h), alpha, m.ctypes.data_as(_lp)),
           "vg_safe_factors")
    return tuple(int(v) for v in m)


def green_table_vgm(N, h, m, alpha: float = ALPHA_DEFAULT, method: int = 0) -> np.ndarray:
    """VG table from the lattice with per-axis oversampling factors m (even); m = (4,4,4) is VICO_2."""
    Nx, Ny, Nz = (int(v) for v in N)
    h = _h3(h)
    mm = np.asarray(m, dtype=np.int64)
    T = np.empty((Nx + 1, Ny + 1, Nz + 1), dtype=np.float64)
    _check(_load().orc_green_table_vgm(Nx, Ny, Nz, _d(h), alpha, method, mm.ctypes.data_as(_lp), _d(T)),
           "green_table_vgm")
    return T


def green_table_vg_entries(N, h, m, entries, alpha: float = ALPHA_DEFAULT) -> np.ndarray:
    """Entries T[dx, dy, dz] of the VG table (oversampling factors m, (4,4,4) = the paper's) by the explicit
    triple cosine sum of PAPER.md:100-102, one entry at a time, no transform.  entries: (npts, 3) integers."""
    Nx, Ny, Nz = (int(v) for v in N)
    h = _h3(h)
    mm = np.ascontiguousarray(m, dtype=np.int64)
    d = np.ascontiguousarray(entries, dtype=np.int64).reshape(-1, 3)
    assert ctypes.sizeof(ctypes.c_long) == 8
    assert (d >= 0).all() and (d <= np.array([Nx, Ny, Nz])).all()
    out = np.empty(d.shape[0], dtype=np.float64)
    _check(_load().orc_green_table_vg_entries(Nx, Ny, Nz, _d(h), alpha, mm.ctypes.data_as(_lp), d.shape[0],
                                              d.ctypes.data_as(_lp), _d(out)), "green_table_vg_entries")
    return out


def green_table(algorithm: int, N, h, g0: float = G0_DEFAULT, alpha: float = ALPHA_DEFAULT,
                method: int = 0) -> np.ndarray:
    """Real-space kernel table T of shape (Nx+1, Ny+1, Nz+1) for HOCKNEY / VICO / VICO_2 / VICO_SAFE."""
    if algorithm == VICO_SAFE:
        return green_table_vgm(N, h, vg_safe_factors(N, h, alpha), alpha, method)
    Nx, Ny, Nz = (int(v) for v in N)
    h = _h3(h)
    T = np.empty((Nx + 1, Ny + 1, Nz + 1), dtype=np.float64)
    lib = _load()
    if algorithm == HOCKNEY:
        rc = lib.orc_green_table_he(Nx, Ny, Nz, _d(h), g0, _d(T))
    elif algorithm == VICO:
        rc = lib.orc_green_table_vg(Nx, Ny, Nz, _d(h), alpha, method, _d(T))
    elif algorithm == VICO_2:
        rc = lib.orc_green_table_vg2(Nx, Ny, Nz, _d(h), alpha, method, _d(T))
    else:
        raise ValueError("unknown algorithm")
    _check(rc, "green_table")
    return T


def green_spectrum(T: np.ndarray, method: int = 0) -> np.ndarray:
    """F{G2}: unscaled 3-D DFT of the mirrored table on the doubled grid, complex (2Nx,2Ny,2Nz)."""
    T = np.ascontiguousarray(T, dtype=np.float64)
    Nx, Ny, Nz = (s - 1 for s in T.shape)
    G = np.empty((2 * Nx, 2 * Ny, 2 * Nz), dtype=np.complex128)
    _check(_load().orc_green_spectrum(Nx, Ny, Nz, _d(T), method, _d(G.view(np.float64))),
           "green_spectrum")
    return G


def solve_with_spectrum(Ghat: np.ndarray, h, rho: np.ndarray, method: int = 0) -> np.ndarray:
    """Steps 1-5 of PAPER.md:67-82 with a precomputed F{G2}."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    Nx, Ny, Nz = rho.shape
    Ghat = np.ascontiguousarray(Ghat, dtype=np.complex128)
    assert Ghat.shape == (2 * Nx, 2 * Ny, 2 * Nz)
    h = _h3(h)
    phi = np.empty_like(rho)
    _check(_load().orc_solve(Nx, Ny, Nz, _d(h), _d(Ghat.view(np.float64)), method, _d(rho), _d(phi)),
           "solve")
    return phi


def solve_field_with_spectrum(Ghat: np.ndarray, h, rho: np.ndarray, method: int = 0):
    """phi and E = -grad phi (Eq. A.1) by the spectral gradient on the doubled grid
    (R18).  Returns (phi, E) with E of shape (3, Nx, Ny, Nz)."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    Nx, Ny, Nz = rho.shape
    Ghat = np.ascontiguousarray(Ghat, dtype=np.complex128)
    assert Ghat.shape == (2 * Nx, 2 * Ny, 2 * Nz)
    h = _h3(h)
    phi = np.empty_like(rho)
    E = np.empty((3,) + rho.shape, dtype=np.float64)
    _check(_load().orc_solve_field(Nx, Ny, Nz, _d(h), _d(Ghat.view(np.float64)), method, _d(rho),
                                   _d(phi), _d(E)), "solve_field")
    return phi, E


def field_of_point_charges(T: np.ndarray, h, charges, points) -> np.ndarray:
    """E = -grad phi (R18) of a few point charges, point by point, WITHOUT any FFT: usable at any mesh size.

    With rho = sum_p q_p delta[y_p], phi2[x] = hx hy hz sum_p q_p G2[x - y_p] on the doubled periodic grid
    (PAPER.md:72-80), and the spectral derivative along axis d of a periodic sequence of L = 2 N_d points is
    the circular convolution with S[n] = (pi / (L h_d)) (-1)^n cot(pi n / L), S[0] = 0 (the derivative of the
    real trigonometric interpolant).  So
        E_d[x] = -hx hy hz sum_p q_p sum_{i'} S[x_d - y_pd - i'] G2[.., i', ..].
    charges: list of ((ix, iy, iz), q);  points: (npts, 3) integer mesh indices.  Returns (npts, 3)."""
    T = np.ascontiguousarray(T, dtype=np.float64)
    N = tuple(n - 1 for n in T.shape)
    h = _h3(h)
    w = float(h[0] * h[1] * h[2])
    points = np.asarray(points, dtype=np.int64)
    out = np.zeros((len(points), 3), dtype=np.float64)
    mir = [np.minimum(np.arange(2 * n), 2 * n - np.arange(2 * n)) for n in N]   # 8-case mirror
    for d in range(3):
        L = 2 * N[d]
        n = np.arange(L)
        for (y, q) in charges:
            for ip, x in enumerate(points):
                disp = [int(x[a] - y[a]) % (2 * N[a]) for a in range(3)]
                sel = [mir[a][disp[a]] for a in range(3)]
                sel[d] = mir[d]                       # the whole line of G2 along axis d
                line = T[sel[0], sel[1], sel[2]]      # G2[.., i', ..], i' = 0 .. L-1
                m = (disp[d] - n) % L
                with np.errstate(divide="ignore", invalid="ignore"):
                    S = (np.pi / (L * h[d])) * np.where(m % 2 == 0, 1.0, -1.0) / np.tan(np.pi * m / L)
                S[m == 0] = 0.0
                out[ip, d] -= w * q * float(np.dot(S, line))
    return out


def direct_sum(T: np.ndarray, h, rho: np.ndarray, idx: np.ndarray | None = None) -> np.ndarray:
    """Def. O1: the plain O(V^2) discrete convolution, at all points or at flat indices ``idx``."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    T = np.ascontiguousarray(T, dtype=np.float64)
    Nx, Ny, Nz = rho.shape
    assert T.shape == (Nx + 1, Ny + 1, Nz + 1)
    h = _h3(h)
    lib = _load()
    if idx is None:
        out = np.empty(rho.size, dtype=np.float64)
        _check(lib.orc_direct_sum(Nx, Ny, Nz, _d(h), _d(T), _d(rho), rho.size, None, _d(out)),
               "direct_sum")
        return out.reshape(rho.shape)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    assert ctypes.sizeof(ctypes.c_long) == 8
    out = np.empty(idx.size, dtype=np.float64)
    _check(lib.orc_direct_sum(Nx, Ny, Nz, _d(h), _d(T), _d(rho), idx.size, idx.ctypes.data_as(_lp),
                              _d(out)), "direct_sum")
    return out


def _mask3(periodic):
    m = (ctypes.c_int * 3)(*[int(bool(v)) for v in periodic])
    return m


def solve_mixed(T: np.ndarray, h, rho: np.ndarray, periodic, method: int = 0) -> np.ndarray:
    """PAPER.md:67-82 with step 1 taken literally: only the non-periodic directions are doubled; along a periodic
    direction G is the nearest-image kernel of period N_d h_d (R20).  periodic: three booleans."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    T = np.ascontiguousarray(T, dtype=np.float64)
    Nx, Ny, Nz = rho.shape
    assert T.shape == (Nx + 1, Ny + 1, Nz + 1)
    h = _h3(h)
    phi = np.empty_like(rho)
    _check(_load().orc_solve_mixed(Nx, Ny, Nz, _d(h), _d(T), _mask3(periodic), int(method), _d(rho), _d(phi)),
           "solve_mixed")
    return phi


def direct_sum_mixed(T: np.ndarray, h, rho: np.ndarray, periodic, idx: np.ndarray | None = None) -> np.ndarray:
    """Def. O1 with the nearest image along the periodic directions, at all points or at flat indices ``idx``."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    T = np.ascontiguousarray(T, dtype=np.float64)
    Nx, Ny, Nz = rho.shape
    assert T.shape == (Nx + 1, Ny + 1, Nz + 1)
    h = _h3(h)
    lib = _load()
    if idx is None:
        out = np.empty(rho.size, dtype=np.float64)
        _check(lib.orc_direct_sum_mixed(Nx, Ny, Nz, _d(h), _d(T), _mask3(periodic), _d(rho), rho.size, None, _d(out)),
               "direct_sum_mixed")
        return out.reshape(rho.shape)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    out = np.empty(idx.size, dtype=np.float64)
    _check(lib.orc_direct_sum_mixed(Nx, Ny, Nz, _d(h), _d(T), _mask3(periodic), _d(rho), idx.size,
                                    idx.ctypes.data_as(_lp), _d(out)), "direct_sum_mixed")
    return out


class OraclePlan:
    """plan / precompute_green / solve on host arrays, mirroring the product's four calls.

    PAPER.md:65 (mesh, spacings), :199 (algorithm names), :98 (Green's function computed once and
    reused every solve).
    """

    def __init__(self, N, h, algorithm: int, g0: float = G0_DEFAULT, alpha: float = ALPHA_DEFAULT,
                 method: int = 0):
        self.N = tuple(int(v) for v in N)
        self.h = _h3(h).copy()
        self.algorithm = int(algorithm)
        self.g0, self.alpha, self.method = float(g0), float(alpha), int(method)
        self.T = None
        self.Ghat = None

    def precompute_green(self, keep_spectrum: bool = True):
        self.T = green_table(self.algorithm, self.N, self.h, self.g0, self.alpha, self.method)
        self.Ghat = green_spectrum(self.T, self.method) if keep_spectrum else None
        return self

    def solve(self, rho: np.ndarray) -> np.ndarray:
        if self.T is None:
            raise RuntimeError("solve before precompute_green")
        if self.Ghat is None:
            self.Ghat = green_spectrum(self.T, self.method)
        return solve_with_spectrum(self.Ghat, self.h, rho, self.method)

    def solve_field(self, rho: np.ndarray):
        if self.T is None:
            raise RuntimeError("solve_field before precompute_green")
        if self.Ghat is None:
            self.Ghat = green_spectrum(self.T, self.method)
        return solve_field_with_spectrum(self.Ghat, self.h, rho, self.method)

    def direct_sum(self, rho: np.ndarray, idx=None) -> np.ndarray:
        return direct_sum(self.T, self.h, rho, idx)
