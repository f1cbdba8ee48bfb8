"""GPU parity tests (-m gpu): every step of the CUDA path against the oracle, through the C ABI.

Order matters (the driver runs with -x): this file exercises the library's DEFAULT kernel variants
(global-memory gather, CUDA-core difference-form matcher) first, then the full-size configuration (with
whatever `spf_autotune` verified on this device when SPF_NATIVE=1, else the defaults again);
tests/test_gpu_variants.py (collected after this file, opt-in through SPF_NATIVE=1) then holds the faster
variants -- TMA-staged slicing, the tcgen05 matcher on single CTAs and on CTA pairs -- to the same parity bar.  Every test ends with
`spf_check_fault`, so a pipeline whose watchdog gave up fails the test instead of passing on
garbage.

Tolerances (BASELINE.json:north_star): slices relative L2 <= 1e-5 at eps = 1e-6; distances relative
error <= 1e-4; argmin bit-exact except where the oracle's best two distances are within 1e-4 relative
(those are counted and reported, not failed).
"""
import os

import numpy as np
import pytest
import torch
from scipy import integrate

from oracle import oracle as orc
from spf_inputs import (CONFIGS, make_model, make_detector, make_mask, random_quaternions, planted_truth_quaternions,
                        photon_scale, poisson_images, surrogate_slices, sample_pairs)

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(1500)]

SLICE_TOL = 1e-5
DIST_TOL = 1e-4


def native_opt_in():
    """True when the caller asked for the TMA / tcgen05 variants (SPF_NATIVE=1); see tests/test_gpu_variants.py."""
    return os.environ.get("SPF_NATIVE", "0") == "1"


def choose_variants(ctx):
    """Library defaults, or -- opt-in -- whatever the device self-check verifies (what bench.py --native does)."""
    if native_opt_in():
        return ctx.spf_autotune()
    return {"slice_impl": 1, "match_impl": 1, "match_cta_group": 1, "native": "off (SPF_NATIVE != 1)"}


@pytest.fixture(scope="module")
def spf():
    import __graft_entry__ as ge
    ge.build()
    import paper_2109_05339_b200 as pkg
    return pkg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _rel_l2(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def _check_match(bi, bd, images, slices, mask=None, tag=""):
    """bi/bd from the GPU; oracle on the same fp32 arrays.  Returns the number of near-ties.
    One bar for every matcher and every case (BASELINE.json:north_star): |delta d| <= 1e-4 d, argmin exact unless
    the oracle's best two distances are within 1e-4 relative.  (The 1e-6 (|I|^2 + |S|^2) form of reading s14 is
    for the noise-free planted case only, where d = 0; it is asserted there directly.)"""
    oi, od, osd, _ = orc.match(images, slices, mask)
    bi, bd = np.asarray(bi.cpu()), np.asarray(bd.cpu())
    tol_abs = DIST_TOL * np.maximum(od, 1e-30)
    assert np.all(np.abs(bd - od) <= tol_abs + 1e-6 * (od == 0)), "%s distances differ: max rel %.3e" % (
        tag, float(np.max(np.abs(bd - od) / np.maximum(od, 1e-30))))
    near = (osd - od) <= tol_abs
    wrong = (bi != oi) & ~near
    assert not wrong.any(), "%s argmin differs at %s: gpu %s oracle %s" % (tag, np.flatnonzero(wrong), bi[wrong], oi[wrong])
    return int(near.sum())


# --------------------------------------------------------------------------------- a1 + a2: prepare

def _es_kernel_ft(xi, beta):
    f = lambda z: np.exp(beta * (np.sqrt(1 - z * z) - 1)) * np.cos(xi * z)
    return 2 * integrate.quad(f, 0, 1, epsabs=1e-14, epsrel=1e-13, limit=200)[0]


def test_deapodisation_factors_match_quadrature(spf):
    ctx = spf.SpfContext(21, eps=1e-6)
    info = ctx.info
    assert (info.n, info.n_fine, info.w) == (21, 42, 8) and abs(info.beta - 18.4) < 1e-12
    p = ctx.spf_debug_deapodisation()
    for i in (0, 3, 10, 17, 20):
        n = i - 10
        ref = 2.0 / (info.w * _es_kernel_ft(np.pi * info.w * n / info.n_fine, info.beta))
        assert abs(p[i] - ref) <= 1e-10 * abs(ref)
    assert np.allclose(p, p[::-1], rtol=1e-13)


@pytest.mark.parametrize("N", [21, 16])
def test_fine_grid_is_the_nudft_of_the_deapodised_model(spf, N):
    """b_l = sum_n A[n] p(n1)p(n2)p(n3) exp(-i n . l h): the oracle's NUDFT of A*p at the fine-grid points."""
    rng = np.random.default_rng(3)
    A = make_model(21, 12, 5.0) if N == 21 else rng.standard_normal((N, N, N)).astype(np.float32)
    ctx = spf.SpfContext(N, eps=1e-6)
    ctx.spf_prepare_model(_dev(A))
    assert ctx.info.grid_is_real == (1 if N == 21 else 0)
    nf = ctx.info.n_fine
    b = ctx.spf_debug_fine_grid().cpu().numpy()
    p = ctx.spf_debug_deapodisation()
    Ap = (A.astype(np.float64) * p[:, None, None] * p[None, :, None] * p[None, None, :]).astype(np.float32)
    l = rng.integers(0, nf, size=(300, 3))
    ref = orc.nudft(Ap, 2 * np.pi * l / nf)
    got = b[l[:, 0], l[:, 1], l[:, 2]]
    assert _rel_l2(got, ref) <= 2e-6


# --------------------------------------------------------------------------------- a3-a5: slicing

@pytest.fixture(scope="module")
def tiny():
    cfg = CONFIGS["tiny"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    return cfg, model, pix, refs, orc.slice_points(model, refs, pix)


def slice_tiny_full(spf, tiny, impl, force_complex, layout):
    cfg, model, pix, refs, c_ref = tiny
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    if layout:
        ctx.spf_set_detector_layout(1, 32, 32)
    ctx.spf_set_option("slice_impl", impl)
    ctx.spf_set_option("force_complex_grid", force_complex)
    ctx.spf_prepare_model(_dev(model))
    c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX).cpu().numpy()
    ctx.spf_check_fault()
    assert _rel_l2(c, c_ref) <= SLICE_TOL
    worst = max(_rel_l2(c[m], c_ref[m]) for m in range(cfg.M))
    assert worst <= 3 * SLICE_TOL, "worst single slice %.3e" % worst
    s = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_INTENSITY, scale=2.5).cpu().numpy()
    ctx.spf_check_fault()
    assert np.array_equal(s, (np.float32(2.5) * c.real.astype(np.float32)))


@pytest.mark.parametrize("force_complex,layout", [(0, True), (1, False)])
def test_slice_tiny_full(spf, tiny, force_complex, layout):
    slice_tiny_full(spf, tiny, 1, force_complex, layout)


def test_slice_is_independent_of_the_patch_layout(spf, tiny):
    cfg, model, pix, refs, _ = tiny
    outs = []
    for layout in ((1, 32, 32), (4, 16, 16), (0, 0, 0)):
        ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
        ctx.spf_set_detector_layout(*layout)
        ctx.spf_prepare_model(_dev(model))
        outs.append(ctx.spf_slice(_dev(refs[:8]), _dev(pix), spf.SPF_OUT_COMPLEX).cpu().numpy())
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


@pytest.mark.parametrize("N,eps", [(16, 1e-6), (21, 1e-9), (12, 1e-4)])
def test_slice_general_model_widths_and_even_n(spf, N, eps):
    """Non-even real model (complex fine grid), even N, w = 8 / 10 / 6 (runtime-width kernel)."""
    rng = np.random.default_rng(4)
    A = rng.standard_normal((N, N, N)).astype(np.float32)
    pix = make_detector(1, 16)
    refs = random_quaternions(9, seed=31)
    c_ref = orc.slice_points(A, refs, pix)
    ctx = spf.SpfContext(N, eps=eps)
    ctx.spf_prepare_model(_dev(A))
    assert ctx.info.grid_is_real == 0
    c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX).cpu().numpy()
    ctx.spf_check_fault()
    assert _rel_l2(c, c_ref) <= max(SLICE_TOL, 10 * eps)


def test_slice_edge_cases(spf, tiny):
    cfg, model, pix, refs, c_ref = tiny
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    with pytest.raises(spf.SpfError) as e:
        ctx.spf_slice(_dev(refs), _dev(pix))
    assert e.value.status == -4   # SPF_ESTATE
    ctx.spf_prepare_model(_dev(model))
    # empty inputs are no-ops
    assert ctx.spf_slice(_dev(refs[:0]), _dev(pix)).shape == (0, 1024)
    assert ctx.spf_slice(_dev(refs), _dev(pix[:0])).shape == (64, 0)
    # ragged P (not a multiple of the patch), unnormalised quaternion, q outside [-pi, pi] (2 pi-periodic)
    q3 = (3.0 * refs[:3]).astype(np.float32)
    c = ctx.spf_slice(_dev(q3), _dev(pix[:777]), spf.SPF_OUT_COMPLEX).cpu().numpy()
    assert _rel_l2(c, c_ref[:3, :777]) <= SLICE_TOL
    far = (pix[:200].astype(np.float64) + 2 * np.pi * np.array([1, -1, 2])).astype(np.float32)
    ident = np.array([[1, 0, 0, 0]], np.float32)
    c = ctx.spf_slice(_dev(ident), _dev(far), spf.SPF_OUT_COMPLEX).cpu().numpy()
    ref = orc.slice_points(model, ident, far)
    assert _rel_l2(c, ref) <= SLICE_TOL
    # points at the very edge of the period
    edge = np.array([[np.pi, -np.pi, 0.0], [-np.pi, np.pi, np.pi], [3.14159, 3.14159, -3.14159]], np.float32)
    c = ctx.spf_slice(_dev(ident), _dev(edge), spf.SPF_OUT_COMPLEX).cpu().numpy()
    # At the Nyquist edge the transform of this model is ~1e-5 while the slices' rms magnitude is ~36: a NUFFT's error
    # is relative to the scale of c (reading s15), not to each value, so the bar here is absolute, SLICE_TOL x rms |c|.
    # (A point-wise relative bar was what round 1 had; the emulator run of this very test showed it cannot hold.)
    assert np.max(np.abs(c - orc.slice_points(model, ident, edge))) <= SLICE_TOL * np.sqrt(np.mean(np.abs(c_ref) ** 2))
    ctx.spf_check_fault()
    with pytest.raises(spf.SpfError):
        spf.SpfContext(21, eps=0.0)


def test_slice_small_config_sampled(spf):
    """Small (BASELINE.json:configs[1]): all 1,024 x 16,384 points on the GPU, 4,096 sampled pairs from the oracle."""
    cfg = CONFIGS["small"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_set_detector_layout(cfg.panels, cfg.panel_edge, cfg.panel_edge)
    ctx.spf_prepare_model(_dev(model))
    assert ctx.info.grid_is_real == 1
    sm, sj = sample_pairs(cfg.M, cfg.P, 4096)
    ref = orc.slice_points(model, refs, pix, sm, sj)
    for force_complex in (0, 1):
        ctx.spf_set_option("force_complex_grid", force_complex)
        c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX)
        got = c[torch.from_numpy(sm).cuda(), torch.from_numpy(sj).cuda()].cpu().numpy()
        ctx.spf_check_fault()
        assert _rel_l2(got, ref) <= SLICE_TOL


# --------------------------------------------------------------------------------- a6-a8: matching

MATCH_SIZES = [(16, 64, 1024, False), (5, 300, 1000, True), (130, 257, 192, False), (300, 513, 2048, True)]


@pytest.mark.parametrize("n_img,M,P,masked", MATCH_SIZES)
def test_match_vs_oracle_ragged_sizes(spf, n_img, M, P, masked):
    match_vs_oracle_ragged_sizes(spf, "simt", n_img, M, P, masked)


def set_match_variant(ctx, variant):
    """"simt": the CUDA-core matcher (library default); "mma": the warp-level tensor-core matcher (mma.sync);
    "cg1" / "cg2": the tcgen05 GEMM on single CTAs / CTA pairs."""
    ctx.spf_set_option("match_impl", {"simt": 1, "mma": 2}.get(variant, 0))
    ctx.spf_set_option("match_cta_group", 2 if variant == "cg2" else 1)


def match_vs_oracle_ragged_sizes(spf, variant, n_img, M, P, masked):
    rng = np.random.default_rng(n_img * 7 + M)
    S = (rng.random((M, P)) * rng.random((M, 1)) * 3).astype(np.float32)
    I = rng.poisson(S[rng.integers(0, M, n_img)]).astype(np.float32)
    mask = (rng.random(P) > 0.2).astype(np.uint8) if masked else None
    ctx = spf.SpfContext(8)
    set_match_variant(ctx, variant)
    bi, bd = ctx.spf_match(_dev(I), _dev(S), None if mask is None else _dev(mask))
    ctx.spf_check_fault()
    assert ctx.spf_last_match_products() == (0 if variant == "simt" else 2)     # photon counts: one fp16 image plane
    _check_match(bi, bd, I, S, mask, variant)
    # the independent CUDA-core reference agrees with the oracle too (and gives the full matrix)
    ri, rd, dist = ctx.spf_match_reference(_dev(I), _dev(S), None if mask is None else _dev(mask))
    d_or = orc.distances(I, S, mask)
    assert np.allclose(dist.cpu().numpy(), d_or, rtol=1e-6)
    _check_match(ri, rd, I, S, mask, "ref")


def test_match_planted_ties_and_general_values(spf):
    match_planted_ties_and_general_values(spf, "simt")


def match_planted_ties_and_general_values(spf, variant):
    rng = np.random.default_rng(17)
    M, P = 200, 640
    S = rng.random((M, P)).astype(np.float32)
    S[150] = S[20]                      # exact duplicate: lowest index must win
    planted = np.array([20, 0, 199, 77])
    I = S[planted].copy()               # non-integer images: the two-plane image path of the tcgen05 kernel
    ctx = spf.SpfContext(8)
    set_match_variant(ctx, variant)
    bi, bd = ctx.spf_match(_dev(I), _dev(S))
    bi, bd = bi.cpu().numpy(), bd.cpu().numpy()
    assert list(bi) == list(planted)
    nrm = (I.astype(np.float64) ** 2).sum(1) + (S[planted].astype(np.float64) ** 2).sum(1)
    assert np.all(np.abs(bd) <= 1e-6 * nrm)      # reading s14: noise-free => |d| <= 1e-6 (|I|^2 + |S|^2)
    # large counts (> 2048: not exact in one fp16 term) and a wide dynamic range
    I2 = rng.poisson(3000.0 * S[rng.integers(0, M, 9)]).astype(np.float32)
    bi, bd = ctx.spf_match(_dev(I2), _dev((3000.0 * S).astype(np.float32)))
    # d ~ 3e-4 (|I|^2 + |S|^2) here: the plain expansion would cancel in fp32; the tensor-core matcher conditions
    # the expansion and recomputes the winner's distance in the difference form, so the bar is the same 1e-4 d
    _check_match(bi, bd, I2, (3000.0 * S).astype(np.float32), None, "large counts")
    # scaling: d(aI, aS) = a^2 d with a a power of two is exact through the rescale
    bi4, bd4 = ctx.spf_match(_dev(4 * I2), _dev((4 * (3000.0 * S).astype(np.float32))))
    assert np.array_equal(bi4.cpu().numpy(), bi.cpu().numpy())
    assert np.allclose(bd4.cpu().numpy(), 16 * bd.cpu().numpy(), rtol=1e-6)
    # permuting the reference set permutes the answer
    perm = rng.permutation(M)
    S3p = (3000.0 * S[perm]).astype(np.float32)
    bip, bdp = ctx.spf_match(_dev(I2), _dev(S3p))
    _check_match(bip, bdp, I2, S3p, None, "permuted")
    assert np.allclose(bdp.cpu().numpy(), bd.cpu().numpy(), rtol=1e-5)
    # empty image set is a no-op; M = 0 with images is an error
    assert ctx.spf_match(_dev(I[:0]), _dev(S))[0].shape == (0,)
    ctx.spf_check_fault()
    with pytest.raises(spf.SpfError):
        ctx.spf_match(_dev(I), _dev(S[:0]))


def test_end_to_end_tiny_poisson(spf, tiny):
    """Tiny, everything from the oracle on one side and everything from the GPU on the other."""
    cfg, model, pix, refs, c_ref = tiny
    truth, _ = planted_truth_quaternions(cfg.n_img, refs)
    alpha = photon_scale(c_ref.real, None, cfg.photons)
    images = poisson_images(alpha * orc.slice_points(model, truth, pix).real)
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_set_detector_layout(1, 32, 32)
    ctx.spf_prepare_model(_dev(model))
    slices = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_INTENSITY, scale=alpha)
    bi, bd = ctx.spf_match(_dev(images), slices)
    # oracle end to end: its own fp64 slices
    oi, od, osd, _ = orc.match(images, alpha * c_ref.real)
    bi, bd = bi.cpu().numpy(), bd.cpu().numpy()
    near = (osd - od) <= DIST_TOL * od
    assert np.all((bi == oi) | near)
    assert np.all(np.abs(bd - od) <= DIST_TOL * od)
    # host-buffer entry point gives the same answer
    ctx.spf_check_fault()
    hi, hd, hs = ctx.spf_orientation_match_host(model, refs, pix, images, scale=alpha, want_slices=True)
    assert np.array_equal(hi, bi) and np.array_equal(hd, bd) and np.array_equal(hs, slices.cpu().numpy())


def test_end_to_end_small_subset(spf):
    """Small model and detector, 48 orientations x 24 images: oracle slices everything itself (about 20 s)."""
    cfg = CONFIGS["small"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)[::4].copy()      # 4,096 pixels, still the whole detector footprint
    refs = random_quaternions(48, seed=2)
    truth, _ = planted_truth_quaternions(24, refs, planted_frac=0.25)
    c_ref = orc.slice_points(model, refs, pix)
    alpha = photon_scale(c_ref.real, None, cfg.photons)
    images = poisson_images(alpha * orc.slice_points(model, truth, pix).real)
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_prepare_model(_dev(model))
    c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX).cpu().numpy()
    assert _rel_l2(c, c_ref) <= SLICE_TOL
    slices = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_INTENSITY, scale=alpha)
    bi, bd = ctx.spf_match(_dev(images), slices)
    oi, od, osd, _ = orc.match(images, alpha * c_ref.real)
    bi, bd = bi.cpu().numpy(), bd.cpu().numpy()
    ctx.spf_check_fault()
    near = (osd - od) <= DIST_TOL * od
    assert np.all((bi == oi) | near) and np.all(np.abs(bd - od) <= DIST_TOL * od)


# --------------------------------------------------------------------------------- full size, bench configuration

def test_paper_scale_sampled(spf):
    """Paper-scale (configs[2]) in the launch configuration bench.py times: 10,000 x 65,536 slice points with
    4,096 sampled pairs from the oracle; matching of 10,000 images x 10,000 surrogate slices with 24 sampled
    image rows brute-forced by the oracle (5 % of the pixels masked)."""
    cfg = CONFIGS["paper_scale"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    mask = make_mask(cfg.panels, cfg.panel_edge, cfg.masked_frac)
    refs = random_quaternions(cfg.M, seed=2)
    ctx = spf.SpfContext(cfg.N, eps=cfg.eps)
    ctx.spf_set_detector_layout(cfg.panels, cfg.panel_edge, cfg.panel_edge)
    ctx.spf_prepare_model(_dev(model))
    variants = choose_variants(ctx)   # defaults, or (opt-in) the variants the device self-check passes; after prepare: the slicing checks use the model
    print("paper-scale runs with", variants)
    c = ctx.spf_slice(_dev(refs), _dev(pix), spf.SPF_OUT_COMPLEX)
    sm, sj = sample_pairs(cfg.M, cfg.P, 4096)
    got = c[torch.from_numpy(sm).cuda(), torch.from_numpy(sj).cuda()].cpu().numpy()
    ctx.spf_check_fault()
    del c
    ref = orc.slice_points(model, refs, pix, sm, sj)
    assert _rel_l2(got, ref) <= SLICE_TOL

    S = surrogate_slices(cfg.M, pix, device="cuda")
    alpha = photon_scale(S, mask, cfg.photons)
    S *= alpha
    g = torch.Generator(device="cuda"); g.manual_seed(3)
    truth = torch.randint(0, cfg.M, (cfg.n_img,), generator=g, device="cuda")
    images = torch.empty((cfg.n_img, cfg.P), dtype=torch.float32, device="cuda")
    for s in range(0, cfg.n_img, 1000):
        images[s:s + 1000] = poisson_images(S[truth[s:s + 1000]], seed=4 + s)
    bi, bd = ctx.spf_match(images, S, _dev(mask))
    ctx.spf_check_fault()
    rows = np.random.default_rng(6).choice(cfg.n_img, 24, replace=False)
    S_h = S.cpu().numpy()
    I_h = images[torch.from_numpy(rows).cuda()].cpu().numpy()
    ties = _check_match(bi[torch.from_numpy(rows).cuda()], bd[torch.from_numpy(rows).cuda()], I_h, S_h, mask, "paper-scale")
    print("paper-scale: 24 sampled rows agree with the oracle (%d near-ties)" % ties)
