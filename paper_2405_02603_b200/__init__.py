"""B200-native free-space Poisson convolution (arxiv 2405.02603): Hockney-Eastwood and
Vico-Greengard spectra, pruned + fused fp64 FFT convolution in hand-written sm_100a CUDA.

``binding`` is the thin ctypes layer over the C ABI in ``include/fsp.h`` (``libfsp.so``);
``workloads`` holds the seeded synthetic inputs; ``build`` compiles the library in-tree.
"""
from . import binding, workloads  # noqa: F401
from .binding import HOCKNEY, VICO, VICO_2, VICO_SAFE, FspError, Plan  # noqa: F401
