"""-m "not gpu": the C-ABI library loads and exports every symbol include/fsp.h declares, and the
host-side argument checks work without a GPU (no compute call is made here)."""
import ctypes
import os
import re

import pytest

from paper_2405_02603_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    return build.build_library()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "fsp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fsp_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(libpath):
    syms = _declared_symbols()
    assert len(syms) >= 16
    L = ctypes.CDLL(libpath)
    for s in syms:
        assert hasattr(L, s), f"{s} declared in include/fsp.h but not exported by libfsp.so"
    # and the binding knows every one of them
    assert set(syms) == set(binding.SIGNATURES)


def test_static_queries_and_error_strings(libpath):
    assert binding.version() >= 100
    assert [binding.kernel_name(i) for i in range(5)] == ["k_fwd_x_r2c", "k_fwd_y", "k_conv_z", "k_inv_y", "k_inv_x_c2r"]
    for code in (0, -1, -2, -3, -4, -5, -6):
        assert binding.strerror(code) and "unknown" not in binding.strerror(code)
    assert "unknown" in binding.strerror(-99)


@pytest.mark.parametrize("args", [
    (1, 16, 16, (0.1, 0.1, 0.1), 0),       # too small (any 2 <= N_d <= 1024 is accepted, R19)
    (16, 16, 0, (0.1, 0.1, 0.1), 0),
    (16, 1025, 16, (0.1, 0.1, 0.1), 0),    # too large
    (16, 2048, 16, (0.1, 0.1, 0.1), 0),    # too large
    (16, 16, 16, (0.1, -0.1, 0.1), 0),     # h <= 0
    (16, 16, 16, (0.1, 0.1, float("nan")), 0),
    (16, 16, 16, (0.1, 0.1, 0.1), 7),      # unknown algorithm
])
def test_invalid_arguments_are_rejected_on_the_host(libpath, args):
    with pytest.raises(binding.FspError) as ei:
        binding.plan_create(*args)
    assert ei.value.code == -1


def test_null_plan_is_rejected(libpath):
    L = binding.lib()
    assert L.fsp_precompute_green(None) == -1
    assert L.fsp_solve(None, None, None) == -1
    assert L.fsp_destroy(None) == -1
    assert L.fsp_plan_bytes(None) == 0
    assert L.fsp_plan_create(None, 16, 16, 16, None, 0, None) == -1


def test_no_silent_cpu_fallback(libpath):
    """Without a CUDA device plan creation must fail loudly (FSP_ERR_NO_DEVICE), never compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.FspError) as ei:
        binding.plan_create(16, 16, 16, (0.1, 0.1, 0.1), 0)
    assert ei.value.code == -5


def test_product_does_not_import_oracle():
    """The product path may not import, call or link anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2405_02603_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "fsp_oracle" not in txt, f


def test_sass_reuse_statistics_on_a_snippet():
    """paper_2405_02603_b200.sass_reuse: a source counts as free only if the PREVIOUS instruction carried .reuse on the
    same register in the same operand slot."""
    from paper_2405_02603_b200 import sass_reuse
    sass = """
        /*0000*/                   DFMA R10, R2.reuse, R4, R6 ;
        /*0010*/                   DFMA R12, -R2.reuse, R4, R6 ;
        /*0020*/                   DFMA R14, R2, R8.reuse, R12.reuse ;
        /*0030*/                   DFMA R16, R20, -R8, R12 ;
        /*0040*/                   DFMA R18, R20, c[0x3][0x10], R12 ;
        /*0050*/                   DADD R22, R18, -R16 ;
        /*0060*/                   LDS.128 R24, [R9+UR4+0x10] ;
        /*0070*/                   DMUL R26, R24, R24 ;
    """.splitlines()
    st = sass_reuse.reuse_statistics(sass)
    assert st[("DFMA", 3, 3)] == 1          # the first one
    assert st[("DFMA", 3, 2)] == 2          # R2 repeated; then R2 repeated again (R8, R12 new)
    assert st[("DFMA", 3, 1)] == 1          # R8 and R12 repeated, R20 new
    assert st[("DFMA", 2, 2)] == 1          # constant-bank operand: two register sources, neither flagged before
    assert st[("DADD", 2, 2)] == 1 and st[("DMUL", 2, 2)] == 1
