"""CPU oracle for the free-space Poisson convolution (arxiv 2405.02603).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.  It shares no
code with ``paper_2405_02603_b200`` (the CUDA path) and neither imports the other.

The arithmetic lives in ``fsp_oracle.c`` (plain C, fp64, textbook radix-2 FFT / direct DFT); this
package only builds that file with gcc and marshals numpy arrays into it.
"""
from .oracle import (  # noqa: F401
    HOCKNEY,
    VICO,
    VICO_2,
    VICO_SAFE,
    G0_DEFAULT,
    ALPHA_DEFAULT,
    OraclePlan,
    build,
    dct1,
    direct_sum,
    direct_sum_mixed,
    solve_mixed,
    fft1d,
    fft3d,
    green_spectrum,
    green_table,
    green_table_vgm,
    green_table_vg_entries,
    vg_safe_factors,
    num_threads,
    set_num_threads,
    solve_with_spectrum,
    solve_field_with_spectrum,
    field_of_point_charges,
    vg_window,
)
