"""-m gpu: periodic directions (SURVEY 8(f) N4, reading R20; PAPER.md:67 step 1, :72).  FSP_PARAM_PERIODIC
against the oracle's orc_solve_mixed, which follows the paper's step 1 literally (only the open directions are doubled,
N_d-point transforms along the periodic ones) -- the product instead runs its unchanged doubled-grid kernels with the
table folded to the nearest image, so the two share neither the grid nor the transform lengths."""
import numpy as np
import pytest

import oracle
from paper_2405_02603_b200 import binding
from tests.analytic import rel_l2, rel_max

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

L2_TOL, MAX_TOL = 1e-12, 1e-10


def _solve(N, h, periodic, rho):
    with binding.Plan(N, h, binding.HOCKNEY, periodic=periodic) as p:
        p.precompute_green()
        phi = p.solve(torch.from_numpy(rho).cuda())
        torch.cuda.synchronize()
        return phi.cpu().numpy(), p.green_table()


@pytest.mark.parametrize("periodic", [(1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 0, 1), (1, 1, 1)])
@pytest.mark.parametrize("N,h", [((16, 32, 8), (0.1, 0.05, 0.2)), ((24, 16, 40), (0.07, 0.11, 0.03))])
def test_periodic_directions_against_the_oracle(N, h, periodic):
    rng = np.random.default_rng(sum(N) + 8 * sum(periodic))
    rho = rng.standard_normal(N)
    got, T = _solve(N, h, periodic, rho)
    To = oracle.green_table(oracle.HOCKNEY, N, h)
    ref = oracle.solve_mixed(To, h, rho, periodic)
    assert np.isfinite(got).all()
    assert rel_l2(got, ref) <= L2_TOL, rel_l2(got, ref)
    assert rel_max(got, ref) <= MAX_TOL, rel_max(got, ref)
    # the table the plan reports is the folded one
    fold = [np.minimum(np.arange(n + 1), n - np.arange(n + 1)) if periodic[d] else np.arange(n + 1) for d, n in enumerate(N)]
    assert np.abs(T - To[np.ix_(*fold)]).max() <= 1e-13 * np.abs(To).max()


def test_periodic_tile_and_warp_kernels_against_the_plain_sum():
    """Meshes on which the TMA tile kernels (Nx, Ny >= 128) and k_conv_z_f (Nz = 256) run, sampled outputs against the
    nearest-image sum written out (orc_direct_sum_mixed)."""
    for N, h, periodic in (((128, 128, 32), (0.01, 0.02, 0.05), (1, 1, 0)), ((16, 16, 256), (0.1, 0.1, 0.01), (0, 0, 1))):
        rng = np.random.default_rng(N[2])
        rho = rng.standard_normal(N)
        got, _ = _solve(N, h, periodic, rho)
        To = oracle.green_table(oracle.HOCKNEY, N, h)
        idx = rng.choice(rho.size, 400, replace=False)
        ref = oracle.direct_sum_mixed(To, h, rho, periodic, idx)
        scale = np.abs(ref).max()
        assert np.abs(got.ravel()[idx] - ref).max() <= MAX_TOL * scale
        assert np.linalg.norm(got.ravel()[idx] - ref) <= L2_TOL * np.linalg.norm(ref)


def test_periodic_translation_invariance_and_field():
    """Shifting rho cyclically along a periodic direction shifts phi (exactly the same sums in another order: to
    rounding); E = -grad phi of fsp_solve_field is the derivative of the N_d-periodic interpolant there."""
    N, h, periodic = (32, 16, 16), (0.05, 0.1, 0.1), (1, 0, 0)
    rng = np.random.default_rng(2)
    rho = rng.standard_normal(N)
    a, _ = _solve(N, h, periodic, rho)
    b, _ = _solve(N, h, periodic, np.roll(rho, 5, axis=0))
    assert rel_max(b, np.roll(a, 5, axis=0)) <= 1e-12
    with binding.Plan(N, h, binding.HOCKNEY, periodic=periodic) as p:
        p.precompute_green()
        phi, E = p.solve_field(torch.from_numpy(rho).cuda())
        torch.cuda.synchronize()
        phi, E = phi.cpu().numpy(), E.cpu().numpy()
    assert rel_max(phi, a) <= 1e-13
    # spectral derivative of the periodic phi along x with numpy (the N_x-point transform, Nyquist mode dropped)
    k = 2 * np.pi * np.fft.fftfreq(N[0], d=h[0])
    k[N[0] // 2] = 0.0
    Ex = -np.fft.ifft(1j * k[:, None, None] * np.fft.fft(phi, axis=0), axis=0).real
    assert rel_l2(E[0], Ex) <= 1e-11


def test_periodic_is_rejected_where_it_is_not_defined():
    with pytest.raises(binding.FspError):
        binding.Plan((16, 16, 16), (0.1,) * 3, binding.VICO_2, periodic=(1, 0, 0))   # truncated kernel: open only
    with pytest.raises(binding.FspError):
        binding.Plan((18, 16, 16), (0.1,) * 3, binding.HOCKNEY, periodic=(1, 0, 0))  # embedded mesh: period would change
    with binding.Plan((16, 16, 16), (0.1,) * 3, binding.HOCKNEY) as p:
        with pytest.raises(binding.FspError):
            binding.plan_set_param(p.handle, binding.PARAM_PERIODIC, 8)
        with pytest.raises(binding.FspError):
            binding.plan_set_param(p.handle, binding.PARAM_PERIODIC, 1.5)
        binding.plan_set_param(p.handle, binding.PARAM_PERIODIC, 0)


@pytest.mark.parametrize("N,h", [((16, 8, 512), (0.1, 0.2, 0.01)), ((8, 16, 256), (0.1, 0.1, 0.02)), ((8, 8, 1024), (0.1, 0.1, 0.01)),
                                 ((8, 24, 128), (0.1, 0.1, 0.02)), ((12, 8, 64), (0.1, 0.1, 0.05)), ((20, 12, 16), (0.1, 0.1, 0.1)), ((8, 12, 8), (0.1, 0.1, 0.1))])
def test_periodic_z_on_nz_point_transforms(N, h):
    """k_conv_z_periodic (periodic z, Nz a power of two: Nz-point transforms instead of the padded 2 Nz; both spectrum
    row layouts, ragged last lane group at the small sizes) against the
    oracle's literal step 1, full field, and against the doubled-grid kernel (FSP_PARAM_PERIODIC_FAST_Z = 0)."""
    rng = np.random.default_rng(N[2])
    rho = rng.standard_normal(N)
    To = oracle.green_table(oracle.HOCKNEY, N, h)
    for periodic in ((0, 0, 1), (1, 0, 1)):
        ref = oracle.solve_mixed(To, h, rho, periodic)
        got = {}
        for fast in (1, 0):
            with binding.Plan(N, h, binding.HOCKNEY, periodic=periodic) as p:
                binding.plan_set_param(p.handle, binding.PARAM_PERIODIC_FAST_Z, fast)
                p.precompute_green()
                phi = p.solve(torch.from_numpy(rho).cuda())
                torch.cuda.synchronize()
                got[fast] = phi.cpu().numpy()
            assert rel_l2(got[fast], ref) <= L2_TOL, (fast, rel_l2(got[fast], ref))
            assert rel_max(got[fast], ref) <= MAX_TOL, (fast, rel_max(got[fast], ref))
        # two different kernels ran: visible in the rounding where the doubled-grid kernel transforms the padded pencil in
        # one piece (k_conv_z_f, Nz = 256, 512); the branch-pair kernels of the other sizes compute their even branch
        # exactly as k_conv_z_periodic does and add an odd branch that is zero to rounding, so the bits may agree there
        if N[2] in (256, 512):
            assert not np.array_equal(got[0], got[1])
