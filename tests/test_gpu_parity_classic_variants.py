"""GPU parity of the CLASSIC-CUDA fast variants (-m gpu; collected right after tests/test_gpu_parity.py, before the
opt-in TMA / tcgen05 file): `slice_impl` 3 (warp per point from global memory) and 4 (warp per point from a tile staged
by cp.async), `match_impl` 2 (the warp-level tensor-core matcher: cp.async + ldmatrix + mma.sync).  None of them uses a
tensor map, an mbarrier, TMEM or tcgen05 -- nothing a device fault of this repository's history could come from -- so they
run by default, held to the same bars as the reference kernels: slices relative L2 <= 1e-5 against the oracle, distances
<= 1e-4, argmin exact outside near-ties.  These are the kernels `bench.py` uses when the TMA / tcgen05 variants have not
been cleared (it checks them in-process with spf_selftest first).
"""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from spf_inputs import CONFIGS, make_model, make_detector, make_mask, random_quaternions, poisson_images, surrogate_slices, sample_pairs, photon_scale

import test_gpu_parity as base
from test_gpu_parity import spf, tiny, _dev, _rel_l2, SLICE_TOL, MATCH_SIZES  # noqa: F401  (fixtures)

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(1500)]

CLASSIC_SLICERS = [3, 4]


@pytest.mark.parametrize("impl", CLASSIC_SLICERS)
@pytest.mark.parametrize("force_complex,layout", [(0, True), (1, True), (0, False), (1, False)])
def test_classic_slice_tiny_full(spf, tiny, impl, force_complex, layout):
    base.slice_tiny_full(spf, tiny, impl, force_complex, layout)


@pytest.mark.parametrize("impl", CLASSIC_SLICERS)
@pytest.mark.parametrize("N,eps", [(16, 1e-6), (21, 1e-9)])
def test_classic_slice_general_model(spf, impl, N, eps):
    """Non-even model (complex fine grid), even and odd N, w = 8 and w = 10 (16-cell window from global memory)."""
    rng = np.random.default_rng(4)
    A = rng.standard_normal((N, N, N)).astype(np.float32)
    pix = make_detector(1, 16)
    refs = random_quaternions(9, seed=31)
    c_ref = orc.slice_points(A, refs, pix)
    ctx = spf.SpfContext(N, eps=eps)
    ctx.spf_set_option("slice_impl", impl)
    ctx.spf_set_detector_layout(1, 16, 16)
    ctx.spf_prepare_model(_dev(A))
    c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX).cpu().numpy()
    ctx.spf_check_fault()
    assert _rel_l2(c, c_ref) <= max(SLICE_TOL, 10 * eps)


@pytest.mark.parametrize("impl", CLASSIC_SLICERS)
def test_classic_slice_small_config_sampled_and_equal_to_each_other(spf, impl):
    """Small (configs[1]), real and complex grid, 4,096 oracle samples; variants 3 and 4 walk the same window with the same
    weights in the same order, so their outputs are identical bit for bit."""
    cfg = CONFIGS["small"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_set_detector_layout(cfg.panels, cfg.panel_edge, cfg.panel_edge)
    ctx.spf_prepare_model(_dev(model))
    sm, sj = sample_pairs(cfg.M, cfg.P, 4096)
    ref = orc.slice_points(model, refs, pix, sm, sj)
    for force_complex in (0, 1):
        ctx.spf_set_option("force_complex_grid", force_complex)
        ctx.spf_set_option("slice_impl", impl)
        c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX)
        ctx.spf_check_fault()
        got = c[torch.from_numpy(sm).cuda(), torch.from_numpy(sj).cuda()].cpu().numpy()
        assert _rel_l2(got, ref) <= SLICE_TOL
        ctx.spf_set_option("slice_impl", 3 if impl == 4 else 4)
        assert torch.equal(ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX), c)


@pytest.mark.parametrize("n_img,M,P,masked", MATCH_SIZES)
def test_mma_match_vs_oracle_ragged_sizes(spf, n_img, M, P, masked):
    base.match_vs_oracle_ragged_sizes(spf, "mma", n_img, M, P, masked)


def test_mma_match_planted_ties_and_general_values(spf):
    """Exact duplicates (lowest index wins), noise-free images (two image planes, 3 products), counts above 2,048 at
    d ~ 3e-4 of the norms (conditioned expansion + refinement: the plain 1e-4 d bar), power-of-two scaling, permutation."""
    base.match_planted_ties_and_general_values(spf, "mma")


def test_mma_match_paper_scale_sampled(spf):
    """10,000 Poisson images x 10,000 surrogate slices x 65,536 pixels (5 % masked) through the mma.sync matcher; 24 sampled
    image rows brute-forced by the oracle."""
    cfg = CONFIGS["paper_scale"]
    pix = make_detector(cfg.panels, cfg.panel_edge)
    mask = make_mask(cfg.panels, cfg.panel_edge, cfg.masked_frac)
    ctx = spf.SpfContext(8)
    base.set_match_variant(ctx, "mma")
    S = surrogate_slices(cfg.M, pix, device="cuda")
    S *= photon_scale(S, mask, cfg.photons)
    g = torch.Generator(device="cuda"); g.manual_seed(3)
    truth = torch.randint(0, cfg.M, (cfg.n_img,), generator=g, device="cuda")
    images = torch.empty((cfg.n_img, cfg.P), dtype=torch.float32, device="cuda")
    for s in range(0, cfg.n_img, 1000):
        images[s:s + 1000] = poisson_images(S[truth[s:s + 1000]], seed=4 + s)
    bi, bd = ctx.spf_match(images, S, _dev(mask))
    ctx.spf_check_fault()
    assert ctx.spf_last_match_products() == 2
    rows = np.random.default_rng(6).choice(cfg.n_img, 24, replace=False)
    sel = torch.from_numpy(rows).cuda()
    ties = base._check_match(bi[sel], bd[sel], images[sel].cpu().numpy(), S.cpu().numpy(), mask, "paper-scale mma")
    print("paper-scale, mma.sync matcher: 24 sampled rows agree with the oracle (%d near-ties)" % ties)


def test_selftest_switches_the_classic_variants_on_in_process(spf, tiny):
    """spf_selftest (the C library's own check) on the device: the classic variants agree with the reference kernels and
    become the context's choice -- what bench.py relies on."""
    cfg, model, pix, refs, c_ref = tiny
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_prepare_model(_dev(model))
    for v in ("slice_gcoop", "slice_coop_ld", "match_mma"):
        r = ctx.spf_selftest(v)
        print(v, r["detail"])
        assert r["passed"], r
    assert ctx.spf_get_option("match_impl") == 2 and ctx.spf_get_option("slice_impl") in (1, 3, 4)
    c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX).cpu().numpy()     # whatever is now switched on still matches the oracle
    assert _rel_l2(c, c_ref) <= SLICE_TOL


def test_microbench_reports_device_figures(spf):
    """spf_microbench: the SM-side denominators bench.py measures before its timed region.  Loose sanity bounds only (the
    figures themselves are the measurement): every one is finite and above what any working B200 delivers."""
    ctx = spf.SpfContext(8)
    got = {k: ctx.spf_microbench(k) for k in ("lds32", "lds128", "l2", "hbm_copy")}
    print("spf_microbench GB/s:", {k: round(v, 1) for k, v in got.items()})
    assert got["lds32"] > 2000 and got["lds128"] > 2000 and got["l2"] > 1000 and got["hbm_copy"] > 1000
    assert all(np.isfinite(v) and v < 1e6 for v in got.values())
