"""GPU parity of the faster kernel variants (-m gpu; collected after tests/test_gpu_parity.py).

`slice_impl = 3` (warp-per-point gather from global memory), `2` (the same gather from a TMA-staged
shared-memory tile) and
`match_impl = 0` (the tcgen05 GEMM, on single CTAs and on `cta_group::2` pairs) are held to the same bars as the default variants: slices relative L2 <= 1e-5 against the oracle,
distances <= 1e-4, argmin exact outside near-ties.  Before a variant is launched in this process its
device self-check (paper_2109_05339_b200/selfcheck.py) must have passed in a child process; if it did
not, the test fails there, with the child's report, without launching the variant here.

OPT-IN: these kernels have not yet passed on hardware, and an earlier GPU session of
this repository raised SM exceptions that were never traced to a kernel.  Until the first-contact protocol
(profiles/r02_first_contact.md) has cleared a variant, this file runs only with SPF_NATIVE=1 in the
environment; otherwise every test here is SKIPPED, loudly, and the default `pytest -m gpu` launches the
library's default kernels only.
"""
import os

import numpy as np
import pytest
import torch

from oracle import oracle as orc
from spf_inputs import CONFIGS, make_model, make_detector, random_quaternions, sample_pairs

import test_gpu_parity as base
from test_gpu_parity import spf, tiny, _dev, _rel_l2, SLICE_TOL, MATCH_SIZES  # noqa: F401  (fixtures)

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(1500)]


@pytest.fixture(scope="module")
def verified(spf):
    if os.environ.get("SPF_NATIVE", "0") != "1":
        pytest.skip("TMA / tcgen05 kernel variants are opt-in until cleared on hardware: set SPF_NATIVE=1 (DESIGN.md section 0)")
    from paper_2109_05339_b200 import selfcheck
    report = {}
    selfcheck.verified_variants(0, report=report)
    return report


def _require(verified, variant):
    r = verified[variant]
    if not r["ok"]:
        pytest.fail("device self-check of %s did not pass (status %s): %s" % (variant, r["status"], r["detail"]))


@pytest.mark.parametrize("variant", ["slice_gcoop", "slice_coop_ld", "slice_coop", "match_cg1", "match_cg2"])
def test_variant_selfcheck(verified, variant):
    _require(verified, variant)


# --------------------------------------------------------------------------------- staged slicing

STAGED = [("slice_gcoop", 3), ("slice_coop_ld", 4), ("slice_coop", 2)]


@pytest.mark.parametrize("variant,impl", STAGED)
@pytest.mark.parametrize("force_complex,layout", [(0, True), (1, True), (0, False), (1, False)])
def test_staged_slice_tiny_full(spf, tiny, verified, force_complex, layout, variant, impl):
    _require(verified, variant)
    base.slice_tiny_full(spf, tiny, impl, force_complex, layout)


def test_staged_slice_equals_the_layout_free_result(spf, tiny, verified):
    """Patch shape only changes which tile is staged, never the value: bit-identical outputs (the warp-per-point
    form adds its partial sums in a fixed lane order, so it is layout-free)."""
    _require(verified, "slice_coop")
    cfg, model, pix, refs, _ = tiny
    outs = []
    for layout in ((1, 32, 32), (4, 16, 16), (0, 0, 0)):
        ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
        ctx.spf_set_option("slice_impl", 2)
        ctx.spf_set_detector_layout(*layout)
        ctx.spf_prepare_model(_dev(model))
        outs.append(ctx.spf_slice(_dev(refs[:8]), _dev(pix), spf.SPF_OUT_COMPLEX).cpu().numpy())
        ctx.spf_check_fault()
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


@pytest.mark.parametrize("variant,impl", STAGED)
@pytest.mark.parametrize("N,eps", [(16, 1e-6), (21, 1e-9)])
def test_staged_slice_general_model(spf, verified, N, eps, variant, impl):
    """Non-even model (complex fine grid), even and odd N, w = 8 and w = 10 (w = 10 gathers from global memory with the 16-cell window)."""
    _require(verified, variant)
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


@pytest.mark.parametrize("variant,impl", STAGED)
def test_staged_slice_small_config_sampled(spf, verified, variant, impl):
    """Small (configs[1]) through the staged kernels, real and complex grid, 4,096 oracle samples."""
    _require(verified, variant)
    cfg = CONFIGS["small"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_set_option("slice_impl", impl)
    ctx.spf_set_detector_layout(cfg.panels, cfg.panel_edge, cfg.panel_edge)
    ctx.spf_prepare_model(_dev(model))
    sm, sj = sample_pairs(cfg.M, cfg.P, 4096)
    ref = orc.slice_points(model, refs, pix, sm, sj)
    for force_complex in (0, 1):
        ctx.spf_set_option("force_complex_grid", force_complex)
        c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX)
        got = c[torch.from_numpy(sm).cuda(), torch.from_numpy(sj).cuda()].cpu().numpy()
        ctx.spf_check_fault()
        assert _rel_l2(got, ref) <= SLICE_TOL


# --------------------------------------------------------------------------------- tcgen05 matching

TC = [("match_cg1", "cg1"), ("match_cg2", "cg2")]


@pytest.mark.parametrize("check,variant", TC)
@pytest.mark.parametrize("n_img,M,P,masked", MATCH_SIZES)
def test_tcgen05_match_vs_oracle_ragged_sizes(spf, verified, n_img, M, P, masked, check, variant):
    _require(verified, check)
    base.match_vs_oracle_ragged_sizes(spf, variant, n_img, M, P, masked)


@pytest.mark.parametrize("check,variant", TC)
def test_tcgen05_match_planted_ties_and_general_values(spf, verified, check, variant):
    """Exact duplicates (lowest index wins), noise-free images (two-plane image path, |d| <= 1e-6 (|I|^2 + |S|^2)),
    counts above 2,048, power-of-two scaling, permutation of the reference set."""
    _require(verified, check)
    base.match_planted_ties_and_general_values(spf, variant)


def test_tcgen05_end_to_end_tiny(spf, tiny, verified):
    """Tiny end to end with the tensor-core matcher: oracle slices + oracle matching on one side, GPU slices +
    tcgen05 matching on the other."""
    _require(verified, "match_cg1")
    from spf_inputs import planted_truth_quaternions, photon_scale, poisson_images
    cfg, model, pix, refs, c_ref = tiny
    truth, _ = planted_truth_quaternions(cfg.n_img, refs)
    alpha = photon_scale(c_ref.real, None, cfg.photons)
    images = poisson_images(alpha * orc.slice_points(model, truth, pix).real)
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_prepare_model(_dev(model))
    slices = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_INTENSITY, scale=alpha)
    oi, od, osd, _ = orc.match(images, alpha * c_ref.real)
    near = (osd - od) <= base.DIST_TOL * od
    for variant in ("cg1",) + (("cg2",) if verified["match_cg2"]["ok"] else ()):
        base.set_match_variant(ctx, variant)
        bi, bd = ctx.spf_match(_dev(images), slices)
        ctx.spf_check_fault()
        bi, bd = bi.cpu().numpy(), bd.cpu().numpy()
        assert np.all((bi == oi) | near) and np.all(np.abs(bd - od) <= base.DIST_TOL * od), variant


def test_tcgen05_variants_and_cuda_core_matcher_agree_on_counts(spf, verified):
    """Photon-count images are exact in one fp16 plane (2 products per K step) and both tcgen05 variants add
    the same products in the same K order into fp32 accumulators: distances agree to fp32 round-off, and with
    the CUDA-core difference form to the parity tolerance."""
    _require(verified, "match_cg1")
    rng = np.random.default_rng(23)
    M, P, n_img = 700, 3000, 260
    S = (rng.random((M, P)) * 2).astype(np.float32)
    I = rng.poisson(S[rng.integers(0, M, n_img)]).astype(np.float32)
    ctx = spf.SpfContext(8)
    res = {}
    for variant in ("simt", "cg1") + (("cg2",) if verified["match_cg2"]["ok"] else ()):
        base.set_match_variant(ctx, variant)
        bi, bd = ctx.spf_match(_dev(I), _dev(S))
        ctx.spf_check_fault()
        assert ctx.spf_last_match_products() == (0 if variant == "simt" else 2)
        res[variant] = (bi.cpu().numpy(), bd.cpu().numpy())
        base._check_match(torch.from_numpy(res[variant][0]), torch.from_numpy(res[variant][1]), I, S, None, variant)
    assert np.allclose(res["simt"][1], res["cg1"][1], rtol=1e-4)
    if "cg2" in res:
        assert np.allclose(res["cg1"][1], res["cg2"][1], rtol=2e-6)


def test_tcgen05_accumulator_rounding_at_k_65536(spf, verified):
    """Does sm_100a's tensor-core accumulator round to nearest or truncate?  (decides the default of
    `match_chunk_kblocks`.)  Paper-scale statistics, K = 65,536 pixels, 128 images x 256 slices, the contraction's own
    a_i + b_m - 2 G (match_refine = 0): once with all of K accumulated in TMEM (chunk 0), once with the library's chunks
    of 32 K blocks.  The CPU replay predicts 1.9e-4 (truncating) or <= 5e-6 (nearest) for chunk 0 and <= 1e-5 for chunks
    of 32 under either rounding.  Only the library's setting is held to the bar; the other number is the measurement."""
    _require(verified, "match_cg1")
    from spf_inputs import make_mask, poisson_images, surrogate_slices
    cfg = CONFIGS["paper_scale"]
    pix = make_detector(cfg.panels, cfg.panel_edge)
    mask = make_mask(cfg.panels, cfg.panel_edge, cfg.masked_frac)
    S = surrogate_slices(256, pix)
    S *= np.float32(cfg.photons / float(S.sum(axis=1).mean()))
    I = poisson_images(S[np.arange(128) * 2 % 256])
    oi, od, _, _ = orc.match(I, S, mask)
    ctx = spf.SpfContext(8)
    base.set_match_variant(ctx, "cg2" if verified["match_cg2"]["ok"] else "cg1")
    ctx.spf_set_option("match_refine", 0)
    worst = {}
    for chunk in (0, 32):
        ctx.spf_set_option("match_chunk_kblocks", chunk)
        bi, bd = ctx.spf_match(_dev(I), _dev(S), _dev(mask))
        ctx.spf_check_fault()
        assert np.array_equal(bi.cpu().numpy(), oi)
        worst[chunk] = float(np.max(np.abs(bd.cpu().numpy() - od) / od))
    print("K = 65,536 accumulation, worst relative distance error: whole K in TMEM %.2e, chunks of 32 K blocks %.2e"
          % (worst[0], worst[32]))
    assert worst[32] <= 2e-5
