"""-m gpu, collected last: fsp_green_spectrum_static (include/fsp.h) -- the table -> spectrum step of the Green
precompute with its scratch in a file-scope `static __device__` array, for callers that cannot call cudaMalloc.

Checked against the existing path: a plan's own fsp_precompute_green / fsp_get_green_spectrum on the same table, at the
tolerance of the table parity tests, on two calls in a row (the second on a different, smaller mesh: the array keeps the
first call's contents, none of which may leak into the second result), plus the capacity and argument errors.
Runs alone in a fresh process as well as after the other GPU tests: it uses nothing but its own plans."""
import numpy as np
import pytest
import torch

from paper_2405_02603_b200 import binding

pytestmark = pytest.mark.gpu

REL_TOL = 1e-12   # relative L2, the bar of the spectrum parity tests (test_gpu_parity.py)


def _existing_path(N, h, alg):
    with binding.Plan(N, h, alg) as p:
        p.precompute_green()
        return p.green_table(), p.green_spectrum()


def _static_path(T):
    N = tuple(n - 1 for n in T.shape)
    Td = torch.from_numpy(T).cuda()
    Gd = torch.full_like(Td, float("nan"))
    binding.green_spectrum_static(Td, Gd, N, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return Gd.cpu().numpy()


def _rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def test_static_spectrum_matches_the_plan_twice_in_a_row():
    cases = [((64, 64, 64), (1.0 / 64,) * 3, binding.HOCKNEY),        # the full capacity: 65^3 entries
             ((32, 16, 48), (0.05, 0.1, 0.02), binding.VICO_2),       # smaller: stale scratch beyond it, a 3 * 2^k axis
             ((64, 64, 64), (1.0 / 64,) * 3, binding.HOCKNEY)]        # and the first one again
    for N, h, alg in cases:
        T, G_ref = _existing_path(N, h, alg)
        G = _static_path(T)
        assert np.isfinite(G).all()
        assert _rel_l2(G, G_ref) < REL_TOL, (N, _rel_l2(G, G_ref))
        # the DC entry is the weighted sum of the table (closed form of the cosine sum at k = 0)
        w = [np.r_[1.0, np.full(n - 1, 2.0), 1.0] for n in N]
        dc = np.einsum("i,j,k,ijk->", w[0], w[1], w[2], T)
        assert abs(G[0, 0, 0] - dc) <= 1e-12 * abs(dc)


def test_static_spectrum_same_result_on_immediate_repeat():
    T, G_ref = _existing_path((32, 32, 32), (0.1, 0.1, 0.1), binding.HOCKNEY)
    G1 = _static_path(T)
    G2 = _static_path(T)
    assert np.array_equal(G1, G2)
    assert _rel_l2(G1, G_ref) < REL_TOL
    # no device memory is taken by a call (after the first one, which may load the kernels' module)
    # (device-wide free memory as the driver reports it: the library does not go through torch's allocator, and
    # garbage left by earlier tests is collected first so that nothing is released in between)
    import gc
    Td = torch.from_numpy(T).cuda()
    Gd = torch.empty_like(Td)
    gc.collect()
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    binding.green_spectrum_static(Td, Gd, (32, 32, 32), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before
    assert np.array_equal(Gd.cpu().numpy(), G1)


def test_static_spectrum_rejects_what_does_not_fit():
    L = binding.lib()
    d = torch.zeros(8, dtype=torch.float64, device="cuda")
    ptr = d.data_ptr()
    assert 65 ** 3 == binding.STATIC_MAX_DOUBLES
    # one entry too many along z: 65 * 65 * 66 > capacity; nothing is launched, the buffers are not touched
    assert L.fsp_green_spectrum_static(ptr, ptr + 8, 64, 64, 65, None) == binding.ERR_STATIC_CAPACITY
    assert L.fsp_green_spectrum_static(ptr, ptr + 8, 128, 128, 128, None) == binding.ERR_STATIC_CAPACITY
    assert "static" in binding.strerror(binding.ERR_STATIC_CAPACITY)
    assert L.fsp_green_spectrum_static(None, ptr, 8, 8, 8, None) == -1
    assert L.fsp_green_spectrum_static(ptr, ptr, 8, 8, 8, None) == -1          # in place
    assert L.fsp_green_spectrum_static(ptr, ptr + 8, 0, 8, 8, None) == -1
    assert L.fsp_green_spectrum_static(ptr, ptr + 8, 2, 2, 1024, None) == -1   # N_d > 512
    torch.cuda.synchronize()
    assert float(d.abs().sum()) == 0.0
