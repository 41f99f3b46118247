"""-m gpu: the parity gaps the round-1 review named, closed.

(a) FULL-FIELD comparisons with the oracle (O2) on meshes on which every persistent kernel
    runs its loop body at least twice per CTA (TMA buffer refill and mbarrier phase flip of the tile kernels, the
    second and later pair steps of k_conv_z_p): the sampled full-size checks cannot exclude a fault confined to a
    few tiles, and the thin slabs of test_gpu_parity.py give every CTA at most one tile.
(b) SURVEY 8(d) parity protocol at size: full-field O2 for BASELINE config 3 (256^3, Gaussian + noise) and
    config 4 (128 x 128 x 512 beam), HE and VG, with the ORACLE's tables.
(c) Vico-Greengard tables at size against the oracle's: VICO_2 / VICO_SAFE at 256^3 and on the beam mesh in
    full, VICO_2 at 512^3 on sampled entries against the explicit triple cosine sum; plain
    VICO at 256^3 (BASELINE config 3: 1024^3 precompute lattice) against VICO_2 (PAPER.md:102's own invariant).
(d) the accuracies bench.py only prints, asserted: HE 2.195e-4 at 256^3, VG at round-off
    at 256^3 and 512^3.
Tolerances are BASELINE.json's: relative L2 <= 1e-12, max-norm relative <= 1e-10; tables 1e-13 of their maximum.
"""
import functools

import numpy as np
import pytest

import oracle
from paper_2405_02603_b200 import binding, workloads as W
from tests.analytic import gaussian_potential_iso, rel_l2, rel_max

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

L2_TOL, MAX_TOL, TABLE_TOL = 1e-12, 1e-10, 1e-13
ALGS = {"HE": (binding.HOCKNEY, oracle.HOCKNEY), "VG": (binding.VICO, oracle.VICO), "VG2": (binding.VICO_2, oracle.VICO_2),
        "VGS": (binding.VICO_SAFE, oracle.VICO_SAFE)}


def gpu_solve(plan, rho_np):
    rho = torch.from_numpy(rho_np).cuda()
    phi = plan.solve(rho)
    torch.cuda.synchronize()
    return phi.cpu().numpy()


def check(got, ref):
    assert np.isfinite(got).all()
    assert rel_l2(got, ref) <= L2_TOL, f"rel L2 {rel_l2(got, ref):.3e}"
    assert rel_max(got, ref) <= MAX_TOL, f"max rel {rel_max(got, ref):.3e}"


@functools.lru_cache(maxsize=2)
def oracle_table(alg, N, h):
    return oracle.green_table(ALGS[alg][1], N, h)


# ---- (a) persistent loops iterate >= 2 times per CTA --------------------------------------------------------
# tiles / pair steps per launch against the resident CTAs (148 SMs x CTAs per SM):
#   (32, 32, 512): K3 pair kernel 33*64/2 = 1056 pair steps on 148 x 4 pairs; x/y first-generation
#   (64, 32, 256): K3 pair kernel (Nz = 256) 65*64/2 = 2080 pair steps on 148 x 6 pairs
#   (32, 512, 64): K2/K4 tile kernels <512>: 33*8 = 264 tiles on 148 CTAs
#   (32, 128, 256): K2/K4 tile kernels <128>: 33*32 = 1056 tiles on 592 CTAs; K3 pair kernel <256>
#   (512, 64, 64): K1/K5 tile kernels <256>: 64*64/16 = 256 tiles on 148 CTAs
#   (256, 64, 128): K1/K5 tile kernels <128>: 512 tiles on 296 CTAs; K2/K4 first-generation
#   (128, 256, 128): K1/K5 <64>, K2/K4 <256> (129*16 = 2064 tiles on 296 CTAs)
LOOP_MESHES = [(32, 32, 512), (64, 32, 256), (32, 512, 64), (32, 128, 256), (512, 64, 64), (256, 64, 128), (128, 256, 128)]


@pytest.mark.parametrize("alg", ["HE", "VG2"])
@pytest.mark.parametrize("N", LOOP_MESHES)
def test_full_field_where_every_persistent_loop_iterates(N, alg):
    w = W.random_density(N, seed=sum(N) + 1)
    with binding.Plan(w.N, w.h, ALGS[alg][0]) as p:
        got = gpu_solve(p.precompute_green(), w.rho)
    ref = oracle.OraclePlan(w.N, w.h, ALGS[alg][1]).precompute_green().solve(w.rho)
    check(got, ref)


@pytest.mark.parametrize("N", [(32, 32, 512), (512, 64, 64), (32, 256, 128)])
def test_full_field_of_the_field_output_where_loops_iterate(N):
    """fsp_solve_field (the DER variants of the same persistent kernels), all three components, full field."""
    w = W.random_density(N, seed=sum(N) + 2)
    with binding.Plan(w.N, w.h, binding.HOCKNEY) as p:
        p.precompute_green()
        phi, E = p.solve_field(torch.from_numpy(w.rho).cuda())
        torch.cuda.synchronize()
        phi, E = phi.cpu().numpy(), E.cpu().numpy()
    phi_o, E_o = oracle.OraclePlan(w.N, w.h, oracle.HOCKNEY).precompute_green().solve_field(w.rho)
    check(phi, phi_o)
    for d in range(3):
        check(E[d], E_o[d])


@pytest.mark.parametrize("N,variant", [((32, 32, 512), 1), ((32, 32, 512), 2), ((64, 32, 256), 1), ((16, 64, 512), 0),
                                       ((16, 24, 96), 1), ((16, 24, 96), 2), ((40, 12, 192), 0)])
# (.., 96): default = the prime-factor warp kernel k_conv_z_pf; 1 = the branch kernel k_conv_z_g; 2 = k_conv_z_g2
def test_z_pass_kernel_variants_full_field(N, variant):
    """FSP_PARAM_K3_VARIANT: the branch-pair kernels of the z pass (k_conv_z_p, k_conv_z_s) stay selectable for A/B
    measurements; each against the oracle, phi and the field (the DER variants), where the persistent loops iterate."""
    w = W.random_density(N, seed=sum(N) + 3)
    with binding.Plan(w.N, w.h, binding.VICO_2) as p:
        binding.plan_set_param(p.handle, binding.PARAM_K3_VARIANT, variant)
        with pytest.raises(binding.FspError):
            binding.plan_set_param(p.handle, binding.PARAM_K3_VARIANT, 3)
        p.precompute_green()
        phi, E = p.solve_field(torch.from_numpy(w.rho).cuda())
        phi2 = p.solve(torch.from_numpy(w.rho).cuda())
        torch.cuda.synchronize()
        assert torch.equal(phi, phi2)
        phi, E = phi.cpu().numpy(), E.cpu().numpy()
    phi_o, E_o = oracle.OraclePlan(w.N, w.h, oracle.VICO_2).precompute_green().solve_field(w.rho)
    check(phi, phi_o)
    for d in range(3):
        check(E[d], E_o[d])


def test_forward_y_kernel_variants_are_both_correct():
    """FSP_PARAM_K2_VARIANT at Ny = 512: the padded-column kernel (default) and the two-branch tile kernel, full field,
    264 tiles on 148 CTAs (the persistent loop iterates)."""
    w = W.random_density((32, 512, 64), seed=77)
    ref = oracle.OraclePlan(w.N, w.h, oracle.HOCKNEY).precompute_green().solve(w.rho)
    for variant in (0, 1):
        with binding.Plan(w.N, w.h, binding.HOCKNEY) as p:
            binding.plan_set_param(p.handle, binding.PARAM_K2_VARIANT, variant)
            check(gpu_solve(p.precompute_green(), w.rho), ref)


# ---- (b) BASELINE configs 3 and 4, full field against O2 with the oracle's own table -------------------------
@pytest.mark.parametrize("alg", ["HE", "VG2"])
def test_config3_256_full_field_against_the_oracle(alg):
    """256^3, Gaussian + 1e-6 noise: the oracle's un-pruned 512^3 complex FFT convolution (2 x 2.1 GB on the host)."""
    w = W.config3()
    with binding.Plan(w.N, w.h, ALGS[alg][0]) as p:
        got = gpu_solve(p.precompute_green(), w.rho)
    T = oracle_table(alg, w.N, w.h)
    ref = oracle.solve_with_spectrum(oracle.green_spectrum(T), w.h, w.rho)
    check(got, ref)


@pytest.mark.parametrize("alg", ["HE", "VG2", "VGS"])
def test_config4_beam_full_field_against_the_oracle(alg):
    """128 x 128 x 512 beam-like Gaussian; VG2 = the paper's literal 4x lattice (aliased on this box, R12: parity is
    the criterion), VGS = the anisotropy-safe lattice (513 x 513 x 1025)."""
    w = W.config4()
    with binding.Plan(w.N, w.h, ALGS[alg][0]) as p:
        got = gpu_solve(p.precompute_green(), w.rho)
    T = oracle_table(alg, w.N, w.h)
    ref = oracle.solve_with_spectrum(oracle.green_spectrum(T), w.h, w.rho)
    check(got, ref)


def _host_memory_available_gib():
    try:
        import psutil
        return psutil.virtual_memory().available / 2 ** 30
    except Exception:   # noqa: BLE001
        return 0.0


@pytest.mark.skipif(_host_memory_available_gib() < 60.0, reason="the oracle's 1024^3 complex arrays need about 40 GiB of host memory")
@pytest.mark.parametrize("alg", ["HE", "VG2"])
def test_config5_512_full_field_against_the_oracle(alg):
    """BASELINE config 5, the bench workload itself (512^3, Gaussian sigma = 0.05; HE and the memory-reduced VG), FULL
    field against the oracle's un-pruned 1024^3 complex FFT convolution with the ORACLE's table (two arrays of 17 GB on
    the host, under a minute on 16 cores): the sampled check of
    test_gpu_parity.py::test_full_size_sampled_against_plain_definition cannot exclude a fault confined to a few tiles
    of the launch configuration the bench times; this can."""
    w = W.config5()
    with binding.Plan(w.N, w.h, ALGS[alg][0]) as p:
        got = gpu_solve(p.precompute_green(), w.rho)
    G = oracle.green_spectrum(oracle.green_table(ALGS[alg][1], w.N, w.h))
    ref = oracle.solve_with_spectrum(G, w.h, w.rho)
    del G
    check(got, ref)


# ---- (c) Vico-Greengard tables at size -----------------------------------------------------------------------
@pytest.mark.parametrize("name,alg", [("256", "VG2"), ("beam", "VG2"), ("beam", "VGS"), ("512", "VG2")])
def test_vg_table_at_size_against_the_oracle_table(name, alg):
    """The DCT paths that only run at size (lattices 513^3, 257 x 257 x 1025, 513 x 513 x 1025, and the 1025^3 lattice of
    BASELINE config 5 with its chunked fused z pass) against the oracle's transform route, every entry."""
    if name == "512" and _host_memory_available_gib() < 40.0:
        pytest.skip("the oracle's 1025^3 lattice and its intermediates need about 25 GiB of host memory")
    w = {"256": W.config3, "beam": W.config4, "512": W.config5}[name]()
    with binding.Plan(w.N, w.h, ALGS[alg][0]) as p:
        p.precompute_green()
        T = p.green_table()
        if alg == "VGS":
            assert p.vg_factors() == oracle.vg_safe_factors(w.N, w.h) == (8, 8, 4)
    To = oracle_table(alg, w.N, w.h)
    assert np.abs(T - To).max() <= TABLE_TOL * np.abs(To).max()


def test_vg2_table_at_512_on_sampled_entries_against_the_explicit_cosine_sum():
    """512^3 (BASELINE config 5): the 1025^3 lattice is out of reach of a host transform within a test, so 16 entries
    of the GPU's table are recomputed by the explicit triple cosine sum (1.1e9 terms each; oracle function pinned
    against scipy's DCT-I, the oracle's transform route and numpy's ifftn of Eq. 3 on small meshes)."""
    w = W.config5()
    with binding.Plan(w.N, w.h, binding.VICO_2) as p:
        p.precompute_green()
        T = p.green_table()
    rng = np.random.default_rng(29)
    ent = np.concatenate([np.array([(0, 0, 0), (512, 512, 512), (1, 0, 0), (0, 0, 1), (512, 0, 3), (255, 256, 257)]),
                          rng.integers(0, 513, size=(10, 3))])
    ref = oracle.green_table_vg_entries(w.N, w.h, (4, 4, 4), ent)
    got = T[ent[:, 0], ent[:, 1], ent[:, 2]]
    assert np.abs(got - ref).max() <= TABLE_TOL * np.abs(T).max()
    assert np.abs(ref[0] / T.max() - 1.0) < 1e-12      # the origin entry is the table's maximum: the scale is pinned


def test_plain_vico_at_config3_size():
    """BASELINE config 3 names "VG (oversampled precompute)": FSP_VICO at 256^3, i.e. the (4N)^3 = 1024^3 lattice of
    PAPER.md:94-98.  Its table equals the FSP_VICO_2 table to round-off (the modified precompute
    computes the same Green's function) and the oracle's; the solve matches Def. O1 on sampled outputs."""
    w = W.config3()
    with binding.Plan(w.N, w.h, binding.VICO) as p:
        p.precompute_green()
        T = p.green_table()
        got = gpu_solve(p, w.rho)
        assert 0 < p.precompute_peak_bytes <= 10 * 2 ** 30   # half-spectrum C2R route: 8.6 GB, not the 17 GB full grid
    with binding.Plan(w.N, w.h, binding.VICO_2) as p2:
        T2 = p2.precompute_green().green_table()
    assert np.abs(T - T2).max() <= TABLE_TOL * np.abs(T2).max()
    To = oracle_table("VG2", w.N, w.h)
    assert np.abs(T - To).max() <= TABLE_TOL * np.abs(To).max()
    idx = np.random.default_rng(31).integers(0, 256 ** 3, size=200)
    ref = oracle.direct_sum(To, w.h, w.rho, idx)
    g = got.reshape(-1)[idx]
    assert np.linalg.norm(g - ref) / np.linalg.norm(ref) <= L2_TOL
    assert np.abs(g - ref).max() / np.abs(got).max() <= MAX_TOL


# ---- (d) accuracies against the closed form, asserted -------------------------------------
def test_accuracy_at_size_against_the_closed_form():
    """Normalised Gaussian sigma = 0.05 in the unit cube: HE is second order with 2.195e-4 at 256^3 (BASELINE.md
    section 2, the survey's numpy value) and a quarter of that at 512^3; VG is at round-off (spectral)."""
    for n, he_ref in ((256, 2.195e-4), (512, 2.195e-4 / 4.0)):
        w = W.config1(n)
        ex = gaussian_potential_iso(w)
        with binding.Plan(w.N, w.h, binding.HOCKNEY) as p:
            he = rel_l2(gpu_solve(p.precompute_green(), w.rho), ex)
        assert he == pytest.approx(he_ref, rel=5e-3 if n == 256 else 2e-2)
        with binding.Plan(w.N, w.h, binding.VICO_2) as p:
            vg = rel_l2(gpu_solve(p.precompute_green(), w.rho), ex)
        assert vg < 1e-13, vg
