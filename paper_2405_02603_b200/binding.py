"""Thin ctypes binding of libfsp.so (include/fsp.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels behind the C ABI.  There is no CPU fallback -- if the library is
missing or no B200 is present the calls raise.

Module-level functions carry the C names without the ``fsp_`` prefix (``plan_create``,
``precompute_green``, ``solve``, ``destroy`` ...); ``Plan`` is a small RAII convenience around them.
Device buffers are torch CUDA tensors (torch is used for device memory and streams only) or raw
integer device pointers.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

HOCKNEY, VICO, VICO_2, VICO_SAFE = 0, 1, 2, 3           # include/fsp.h, PAPER.md:199 (+ DESIGN.md R17)
PARAM_G0, PARAM_ALPHA, PARAM_CHUNK_PLANES, PARAM_K3_VARIANT, PARAM_K2_VARIANT, PARAM_PERIODIC, PARAM_PERIODIC_FAST_Z = 0, 1, 2, 3, 4, 5, 6
NUM_SOLVE_KERNELS = 5
ERRORS = {0: "FSP_OK", -1: "FSP_ERR_INVALID_ARG", -2: "FSP_ERR_NOT_PRECOMPUTED",
          -3: "FSP_ERR_OUT_OF_MEMORY", -4: "FSP_ERR_CUDA", -5: "FSP_ERR_NO_DEVICE"}

_HERE = os.path.dirname(os.path.abspath(__file__))
# the in-tree library; FSP_LIB selects another build of the SAME library (A/B measurements of kernel variants), never a fallback
LIB_PATH = os.environ.get("FSP_LIB", os.path.join(_HERE, "libfsp.so"))
_lib = None

# every symbol include/fsp.h declares, with its ctypes signature
_c = ctypes
_vp, _dp, _i, _d, _sz = _c.c_void_p, _c.POINTER(_c.c_double), _c.c_int, _c.c_double, _c.c_size_t
SIGNATURES = {
    "fsp_plan_create": (_i, [_c.POINTER(_vp), _i, _i, _i, _dp, _i, _vp]),
    "fsp_plan_set_param": (_i, [_vp, _i, _d]),
    "fsp_plan_set_spacing": (_i, [_vp, _dp]),
    "fsp_precompute_green": (_i, [_vp]),
    "fsp_solve": (_i, [_vp, _vp, _vp]),
    "fsp_solve_host": (_i, [_vp, _vp, _vp]),
    "fsp_solve_host_batch": (_i, [_vp, _i, _c.POINTER(_vp), _c.POINTER(_vp)]),
    "fsp_solve_field": (_i, [_vp, _vp, _vp, _vp]),
    "fsp_solve_field_host": (_i, [_vp, _vp, _vp, _vp]),
    "fsp_model_bytes_per_field_solve": (_d, [_vp, _i]),
    "fsp_destroy": (_i, [_vp]),
    "fsp_plan_bytes": (_sz, [_vp]),
    "fsp_precompute_peak_bytes": (_sz, [_vp]),
    "fsp_model_bytes_per_solve": (_d, [_vp, _dp]),
    "fsp_get_vg_factors": (_i, [_vp, _c.POINTER(_i)]),
    "fsp_vg_lattice_is_safe": (_i, [_vp, _c.POINTER(_i)]),
    "fsp_get_green_table": (_i, [_vp, _dp]),
    "fsp_get_green_spectrum": (_i, [_vp, _dp]),
    "fsp_green_spectrum_static": (_i, [_vp, _vp, _i, _i, _i, _vp]),
    "fsp_ubench_fp64": (_i, [_i, _i, _c.POINTER(_d)]),
    "fsp_set_profiling": (_i, [_vp, _i]),
    "fsp_get_kernel_times": (_i, [_vp, _c.POINTER(_c.c_float), _c.POINTER(_i)]),
    "fsp_shard_planes": (_i, [_i, _i, _i, _c.POINTER(_i), _c.POINTER(_i)]),
    "fsp_shard_block": (_i, [_i, _i, _i, _i, _i, _i, _i, _c.POINTER(_c.c_longlong)]),
    "fsp_sharded_create": (_i, [_c.POINTER(_vp), _i, _i, _i, _dp, _i, _vp, _i, _i]),
    "fsp_sharded_set_param": (_i, [_vp, _i, _d]),
    "fsp_sharded_precompute_green": (_i, [_vp]),
    "fsp_sharded_buffers": (_i, [_vp, _c.POINTER(_vp), _c.POINTER(_vp), _c.POINTER(_sz), _c.POINTER(_sz)]),
    "fsp_sharded_set_peers": (_i, [_vp, _c.POINTER(_vp), _c.POINTER(_vp)]),
    "fsp_sharded_solve_phase": (_i, [_vp, _i, _vp, _vp]),
    "fsp_sharded_bytes": (_sz, [_vp]),
    "fsp_sharded_destroy": (_i, [_vp]),
    "fsp_ipc_get_handle": (_i, [_vp, _vp]),
    "fsp_ipc_open_handle": (_i, [_vp, _c.POINTER(_vp)]),
    "fsp_ipc_close_handle": (_i, [_vp]),
    "fsp_kernel_name": (_c.c_char_p, [_i]),
    "fsp_strerror": (_c.c_char_p, [_i]),
    "fsp_version": (_i, []),
}


class FspError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = lib().fsp_strerror(code).decode() if _lib is not None else ""
        super().__init__(f"{where}: {ERRORS.get(code, code)} ({msg})")


def lib():
    """Loads libfsp.so (raises if it has not been built -- no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2405_02603_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _chk(code: int, where: str) -> None:
    if code != 0:
        raise FspError(code, where)


def _ptr(x) -> int:
    """Device (or host) address of a torch tensor / numpy array / int."""
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return int(x.data_ptr())


def version() -> int:
    return int(lib().fsp_version())


def strerror(code: int) -> str:
    return lib().fsp_strerror(code).decode()


def kernel_name(i: int) -> str:
    return lib().fsp_kernel_name(i).decode()


def plan_create(Nx: int, Ny: int, Nz: int, h, algorithm: int, cuda_stream: int = 0) -> int:
    """fsp_plan_create.  Returns the opaque plan handle (an integer address)."""
    hh = (ctypes.c_double * 3)(*[float(v) for v in np.broadcast_to(np.asarray(h, dtype=np.float64), (3,))])
    out = ctypes.c_void_p()
    _chk(lib().fsp_plan_create(ctypes.byref(out), Nx, Ny, Nz, hh, algorithm, ctypes.c_void_p(cuda_stream)),
         "fsp_plan_create")
    return out.value


def plan_set_param(plan: int, which: int, value: float) -> None:
    _chk(lib().fsp_plan_set_param(plan, which, value), "fsp_plan_set_param")


def plan_set_spacing(plan: int, h) -> None:
    hh = (ctypes.c_double * 3)(*[float(v) for v in np.broadcast_to(np.asarray(h, dtype=np.float64), (3,))])
    _chk(lib().fsp_plan_set_spacing(plan, hh), "fsp_plan_set_spacing")


def precompute_green(plan: int) -> None:
    _chk(lib().fsp_precompute_green(plan), "fsp_precompute_green")


def solve(plan: int, rho_dev, phi_dev) -> None:
    _chk(lib().fsp_solve(plan, _ptr(rho_dev), _ptr(phi_dev)), "fsp_solve")


def solve_host(plan: int, rho_host, phi_host) -> None:
    _chk(lib().fsp_solve_host(plan, _ptr(rho_host), _ptr(phi_host)), "fsp_solve_host")


def solve_host_batch(plan: int, rho_hosts, phi_hosts) -> None:
    """fsp_solve_host_batch: sequences of host buffers (numpy arrays or pinned torch CPU tensors)."""
    n = len(rho_hosts)
    assert len(phi_hosts) == n
    ra = (ctypes.c_void_p * max(n, 1))(*[_ptr(x) for x in rho_hosts])
    pa = (ctypes.c_void_p * max(n, 1))(*[_ptr(x) for x in phi_hosts])
    _chk(lib().fsp_solve_host_batch(plan, n, ra, pa), "fsp_solve_host_batch")


def solve_field(plan: int, rho_dev, phi_dev, E_dev) -> None:
    """fsp_solve_field; phi_dev may be None."""
    _chk(lib().fsp_solve_field(plan, _ptr(rho_dev), None if phi_dev is None else _ptr(phi_dev), _ptr(E_dev)),
         "fsp_solve_field")


def solve_field_host(plan: int, rho_host, phi_host, E_host) -> None:
    _chk(lib().fsp_solve_field_host(plan, _ptr(rho_host), None if phi_host is None else _ptr(phi_host),
                                    _ptr(E_host)), "fsp_solve_field_host")


def model_bytes_per_field_solve(plan: int, with_phi: bool = True) -> float:
    return float(lib().fsp_model_bytes_per_field_solve(plan, int(bool(with_phi))))


def destroy(plan: int) -> None:
    _chk(lib().fsp_destroy(plan), "fsp_destroy")


def plan_bytes(plan: int) -> int:
    return int(lib().fsp_plan_bytes(plan))


def precompute_peak_bytes(plan: int) -> int:
    return int(lib().fsp_precompute_peak_bytes(plan))


def model_bytes_per_solve(plan: int):
    per = (ctypes.c_double * NUM_SOLVE_KERNELS)()
    tot = float(lib().fsp_model_bytes_per_solve(plan, per))
    return tot, [float(v) for v in per]


def get_vg_factors(plan: int):
    m = (_i * 3)()
    _chk(lib().fsp_get_vg_factors(plan, m), "fsp_get_vg_factors")
    return tuple(int(v) for v in m)


def vg_lattice_is_safe(plan: int) -> bool:
    ok = _i(0)
    _chk(lib().fsp_vg_lattice_is_safe(plan, ctypes.byref(ok)), "fsp_vg_lattice_is_safe")
    return bool(ok.value)


def get_green_table(plan: int, N) -> np.ndarray:
    T = np.empty(tuple(n + 1 for n in N), dtype=np.float64)
    _chk(lib().fsp_get_green_table(plan, T.ctypes.data_as(_dp)), "fsp_get_green_table")
    return T


def get_green_spectrum(plan: int, N) -> np.ndarray:
    G = np.empty(tuple(n + 1 for n in N), dtype=np.float64)
    _chk(lib().fsp_get_green_spectrum(plan, G.ctypes.data_as(_dp)), "fsp_get_green_spectrum")
    return G


STATIC_MAX_DOUBLES = 274625   # FSP_STATIC_MAX_DOUBLES (65^3)
ERR_STATIC_CAPACITY = -6


def green_spectrum_static(T_dev, Ghat_dev, N, stream: int = 0) -> None:
    """fsp_green_spectrum_static: T -> spectrum octant on the current device, scratch in the library's static device
    array, no allocation.  T_dev, Ghat_dev: contiguous fp64 CUDA tensors of shape (Nx+1, Ny+1, Nz+1)."""
    _chk(lib().fsp_green_spectrum_static(_ptr(T_dev), _ptr(Ghat_dev), int(N[0]), int(N[1]), int(N[2]),
                                         ctypes.c_void_p(int(stream) or None)), "fsp_green_spectrum_static")


def ubench_fp64(mode: int, warps_per_sm: int = 8) -> float:
    """fsp_ubench_fp64: clocks per fp64 warp-instruction and scheduler (mode 0: DFMA with three new register sources,
    1 / 2: with two / one source repeated, 3: DADD)."""
    v = ctypes.c_double()
    _chk(lib().fsp_ubench_fp64(int(mode), int(warps_per_sm), ctypes.byref(v)), "fsp_ubench_fp64")
    return float(v.value)


def set_profiling(plan: int, on: bool) -> None:
    _chk(lib().fsp_set_profiling(plan, int(bool(on))), "fsp_set_profiling")


def get_kernel_times(plan: int):
    ms = (ctypes.c_float * NUM_SOLVE_KERNELS)()
    n = ctypes.c_int()
    _chk(lib().fsp_get_kernel_times(plan, ms, ctypes.byref(n)), "fsp_get_kernel_times")
    return [float(v) for v in ms], int(n.value)


class Plan:
    """plan -> precompute_green -> solve* -> destroy, on the current torch CUDA stream by default."""

    def __init__(self, N, h, algorithm: int, stream: int | None = None, g0: float | None = None,
                 alpha: float | None = None, periodic=None):
        self.N = tuple(int(v) for v in N)
        self.h = tuple(float(v) for v in np.broadcast_to(np.asarray(h, dtype=np.float64), (3,)))
        self.algorithm = int(algorithm)
        if stream is None:
            import torch
            stream = int(torch.cuda.current_stream().cuda_stream)
        self.stream = stream
        self.handle = plan_create(*self.N, self.h, self.algorithm, stream)
        if g0 is not None:
            plan_set_param(self.handle, PARAM_G0, g0)
        if alpha is not None:
            plan_set_param(self.handle, PARAM_ALPHA, alpha)
        if periodic is not None and any(periodic):   # three booleans (x, y, z): FSP_PARAM_PERIODIC
            try:
                plan_set_param(self.handle, PARAM_PERIODIC, sum(1 << d for d in range(3) if periodic[d]))
            except FspError:
                destroy(self.handle)
                self.handle = None
                raise

    def precompute_green(self):
        precompute_green(self.handle)
        return self

    def set_spacing(self, h):
        """New spacings for the same mesh; precompute_green must be called again."""
        plan_set_spacing(self.handle, h)
        self.h = tuple(float(v) for v in np.broadcast_to(np.asarray(h, dtype=np.float64), (3,)))
        return self

    def solve(self, rho, phi=None):
        """rho: contiguous fp64 CUDA tensor of shape N.  Returns phi (allocated if not given)."""
        import torch
        assert rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous() and tuple(rho.shape) == self.N
        if phi is None:
            phi = torch.empty_like(rho)
        assert phi.is_cuda and phi.dtype == torch.float64 and phi.is_contiguous() and tuple(phi.shape) == self.N
        solve(self.handle, rho, phi)
        return phi

    def solve_field(self, rho, phi=None, E=None, want_phi: bool = True):
        """phi and E = -grad phi.  Returns (phi or None, E) with E of shape (3,) + N."""
        import torch
        assert rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous() and tuple(rho.shape) == self.N
        if phi is None and want_phi:
            phi = torch.empty_like(rho)
        if E is None:
            E = torch.empty((3,) + self.N, dtype=torch.float64, device=rho.device)
        assert E.is_cuda and E.dtype == torch.float64 and E.is_contiguous() and tuple(E.shape) == (3,) + self.N
        solve_field(self.handle, rho, phi if want_phi else None, E)
        return (phi if want_phi else None), E

    def solve_field_host(self, rho_host, phi_host, E_host):
        solve_field_host(self.handle, rho_host, phi_host, E_host)
        return phi_host, E_host

    def solve_host(self, rho_host, phi_host):
        """Host buffers (numpy arrays or pinned torch CPU tensors), copies inside the call."""
        solve_host(self.handle, rho_host, phi_host)
        return phi_host

    def solve_host_batch(self, rho_hosts, phi_hosts):
        """n pipelined solves from host buffers (copy-in, solve and copy-out of neighbouring solves overlap)."""
        solve_host_batch(self.handle, rho_hosts, phi_hosts)
        return phi_hosts

    def vg_factors(self):
        return get_vg_factors(self.handle)

    def vg_lattice_is_safe(self) -> bool:
        return vg_lattice_is_safe(self.handle)

    def green_table(self) -> np.ndarray:
        return get_green_table(self.handle, self.N)

    def green_spectrum(self) -> np.ndarray:
        return get_green_spectrum(self.handle, self.N)

    @property
    def bytes(self) -> int:
        return plan_bytes(self.handle)

    @property
    def precompute_peak_bytes(self) -> int:
        return precompute_peak_bytes(self.handle)

    def model_bytes(self):
        return model_bytes_per_solve(self.handle)

    def set_profiling(self, on: bool):
        set_profiling(self.handle, on)

    def kernel_times(self):
        return get_kernel_times(self.handle)

    def destroy(self):
        if self.handle:
            destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# ---- slab decomposition (include/fsp.h "slab decomposition over several GPUs") ---------------------------------
def shard_planes(Nx: int, nranks: int, rank: int):
    k0, npl = _i(0), _i(0)
    _chk(lib().fsp_shard_planes(Nx, nranks, rank, ctypes.byref(k0), ctypes.byref(npl)), "fsp_shard_planes")
    return int(k0.value), int(npl.value)


def shard_block(Nx: int, Ny: int, Nz: int, nranks: int, src_rank: int, dst_rank: int, direction: int):
    """(nrun, run_len, src_off, src_stride, dst_off, dst_stride) in complex elements."""
    out = (ctypes.c_longlong * 6)()
    _chk(lib().fsp_shard_block(Nx, Ny, Nz, nranks, src_rank, dst_rank, direction, out), "fsp_shard_block")
    return tuple(int(v) for v in out)


class ShardedPlan:
    """Rank `rank` of `nranks` of one solve split into y-slabs (marshalling only; the caller provides the barriers
    between the three phases and tells every rank where the others' workspaces are)."""

    def __init__(self, N, h, algorithm: int, rank: int, nranks: int, stream: int = 0):
        self.N = tuple(int(v) for v in N)
        self.rank, self.nranks = rank, nranks
        hh = (ctypes.c_double * 3)(*[float(v) for v in np.broadcast_to(np.asarray(h, dtype=np.float64), (3,))])
        out = ctypes.c_void_p()
        _chk(lib().fsp_sharded_create(ctypes.byref(out), *self.N, hh, algorithm, ctypes.c_void_p(stream), rank, nranks),
             "fsp_sharded_create")
        self.handle = out.value
        self.slab = (self.N[0], self.N[1] // nranks, self.N[2])

    def precompute_green(self):
        _chk(lib().fsp_sharded_precompute_green(self.handle), "fsp_sharded_precompute_green")
        return self

    def buffers(self):
        """(B1x address, B1y address, B1x bytes, B1y bytes) of this rank's transpose targets."""
        a, b, na, nb = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_size_t(), ctypes.c_size_t()
        _chk(lib().fsp_sharded_buffers(self.handle, ctypes.byref(a), ctypes.byref(b), ctypes.byref(na), ctypes.byref(nb)),
             "fsp_sharded_buffers")
        return a.value, b.value, na.value, nb.value

    def set_peers(self, b1x_addrs, b1y_addrs):
        n = self.nranks
        xa = (ctypes.c_void_p * n)(*b1x_addrs)
        ya = (ctypes.c_void_p * n)(*b1y_addrs)
        _chk(lib().fsp_sharded_set_peers(self.handle, xa, ya), "fsp_sharded_set_peers")

    def phase(self, which: int, rho_slab=None, phi_slab=None):
        _chk(lib().fsp_sharded_solve_phase(self.handle, which, _ptr(rho_slab) if rho_slab is not None else None,
                                           _ptr(phi_slab) if phi_slab is not None else None), "fsp_sharded_solve_phase")

    @property
    def bytes(self) -> int:
        return int(lib().fsp_sharded_bytes(self.handle))

    def destroy(self):
        if self.handle:
            _chk(lib().fsp_sharded_destroy(self.handle), "fsp_sharded_destroy")
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


def ipc_get_handle(dev_ptr: int) -> bytes:
    buf = ctypes.create_string_buffer(64)
    _chk(lib().fsp_ipc_get_handle(dev_ptr, ctypes.cast(buf, ctypes.c_void_p)), "fsp_ipc_get_handle")
    return buf.raw


def ipc_open_handle(handle: bytes) -> int:
    buf = ctypes.create_string_buffer(handle, 64)
    out = ctypes.c_void_p()
    _chk(lib().fsp_ipc_open_handle(ctypes.cast(buf, ctypes.c_void_p), ctypes.byref(out)), "fsp_ipc_open_handle")
    return out.value
