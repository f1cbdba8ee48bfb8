"""The kernels' OWN SOURCE executed on the CPU under the functional emulator of tests/emu/, against the oracle.

tests/emu/build_emu.py compiles paper_2109_05339_b200/csrc/*.cu with g++ after a mechanical rewrite (launch syntax,
dynamic shared memory, inline-PTX wrappers replaced by functional stand-ins) and links it with a fiber scheduler that
runs every CUDA thread of a block -- or of a CTA pair -- cooperatively: block barriers, warp shuffles and votes,
mbarrier phases and transaction counts, deferred TMA copies with the 128-byte swizzle, a software TMEM and
tcgen05.mma reading its operands through the kernels' own shared-memory descriptors.  The tests below call the
library's C ABI exactly as the GPU tests do (tests/test_gpu_parity.py, tests/test_gpu_variants.py), at sizes the
emulator finishes in seconds, and hold the results to the same bars: slices relative L2 <= 1e-5, distances <= 1e-4,
argmin exact outside near-ties.

What this is: evidence, obtainable without a GPU, that the kernels' index arithmetic, barrier protocols, pipelines,
descriptors and epilogues are self-consistent and compute the method -- for the library's
default kernels AND for the TMA / tcgen05 variants.  What it is not: GPU parity.  The emulator implements the
programming model as tests/emu/ptx_emu.cuh states it; whether sm_100a agrees is only shown by `-m gpu` on a B200.
Poisoned memory (NaN in fresh device allocations, in shared memory and in TMEM) turns a read of anything the
kernels did not write into a NaN result, and the emulator faults on misaligned TMA destinations, uninitialised
barriers, TMEM accesses outside the warp's lane quadrant or the allocation, and TMEM left allocated at exit.
"""
import os
import sys

import numpy as np
import pytest

from oracle import oracle as orc
from spf_inputs import (CONFIGS, make_model, make_detector, random_quaternions, planted_truth_quaternions, photon_scale,
                        poisson_images)

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))
import emu_binding as eb  # noqa: E402
from emu_binding import EmuContext, EmuError, SPF_OUT_COMPLEX, SPF_OUT_INTENSITY  # noqa: E402

SLICE_TOL = 1e-5
DIST_TOL = 1e-4
# Every (variant x case) combination runs by default (under three minutes); SPF_EMU_FULL=0 keeps one representative of
# every kernel and code path (for the AddressSanitizer build, which is several times slower).
FULL = os.environ.get("SPF_EMU_FULL", "1") == "1"
full_only = pytest.mark.skipif(not FULL, reason="SPF_EMU_FULL=0: one representative per code path")
SLICERS = [(1, "thread-per-point global gather (library default)"), (3, "warp-per-point from global memory"),
           (4, "warp-per-point from a cp.async-staged tile"), (2, "warp-per-point from a TMA-staged tile")]
MATCHERS = ["simt", "mma", "cg1", "cg2"]


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def tiny():
    cfg = CONFIGS["tiny"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    return cfg, model, pix, refs, orc.slice_points(model, refs, pix)


def _matcher(ctx, variant):
    ctx.set_option("match_impl", {"simt": 1, "mma": 2}.get(variant, 0))
    ctx.set_option("match_cta_group", 2 if variant == "cg2" else 1)


def _check_match(bi, bd, I, S, mask=None):
    oi, od, osd, _ = orc.match(I, S, mask)
    tol = DIST_TOL * np.maximum(od, 1e-30)
    assert np.all(np.isfinite(bd))
    assert np.all(np.abs(bd - od) <= tol + 1e-6 * (od == 0)), "max rel %.3e" % float(np.max(np.abs(bd - od) / np.maximum(od, 1e-30)))
    near = (osd - od) <= tol
    assert np.all((bi == oi) | near), (bi, oi)
    return float(np.max(np.abs(bd - od) / np.maximum(od, 1e-30)))


# --------------------------------------------------------------------------------- a1 + a2: spf_prepare_model

@pytest.mark.parametrize("N", [21, 16])
def test_emulated_prepare_is_the_nudft_of_the_deapodised_model(N):
    """k_check_even, k_deapod_pad, (DFT stub in place of cuFFT), k_relayout: b_l against the oracle's NUDFT of A p p p."""
    rng = np.random.default_rng(3)
    A = make_model(21, 12, 5.0) if N == 21 else rng.standard_normal((N, N, N)).astype(np.float32)
    ctx = EmuContext(N, eps=1e-6)
    ctx.prepare_model(A)
    assert ctx.info.grid_is_real == (1 if N == 21 else 0)
    nf = ctx.info.n_fine
    b = ctx.fine_grid()
    p = ctx.deapodisation()
    Ap = (A.astype(np.float64) * p[:, None, None] * p[None, :, None] * p[None, None, :]).astype(np.float32)
    l = rng.integers(0, nf, size=(200, 3))
    ref = orc.nudft(Ap, 2 * np.pi * l / nf)
    assert _rel(b[l[:, 0], l[:, 1], l[:, 2]], ref) <= 2e-6


# --------------------------------------------------------------------------------- a3-a5: spf_slice

@pytest.mark.parametrize("impl,what", SLICERS)
@pytest.mark.parametrize("force_complex,layout", [(0, True), (1, False)])
def test_emulated_slice_tiny_vs_oracle(tiny, impl, what, force_complex, layout):
    cfg, model, pix, refs, c_ref = tiny
    m = 12                                       # 12 orientations x 1,024 pixels: 96 blocks of 128 points
    ctx = EmuContext(cfg.N, eps=cfg.eps)
    if layout:
        ctx.set_detector_layout(1, 32, 32)
    ctx.set_option("slice_impl", impl)
    ctx.set_option("force_complex_grid", force_complex)
    ctx.prepare_model(model)
    eb.counters(); eb.smem_counters()
    c = ctx.slice(refs[:m], pix, SPF_OUT_COMPLEX)
    n, sm = eb.counters(), eb.smem_counters()
    # the cp.async-staged tile (impl 4) is written one shared-memory wavefront per quarter-warp (the emulator's bank model)
    assert (sm["cpasync_groups"] > 0) == (impl == 4) and sm["cpasync_wavefronts"] == sm["cpasync_groups"], sm
    assert np.isfinite(c.view(np.float32)).all()
    assert _rel(c, c_ref[:m]) <= SLICE_TOL
    assert (n["tma_copies"] > 0) == (impl == 2), n          # the staged variant really stages, the others never touch TMA
    s = ctx.slice(refs[:m], pix, SPF_OUT_INTENSITY, scale=2.5)
    assert np.array_equal(s, np.float32(2.5) * c.real.astype(np.float32))


def test_emulated_slicers_agree_bit_for_bit_where_they_should(tiny):
    """Variants 2, 3 and 4 walk the same window with the same weights in the same order: identical bits; and the result
    does not depend on how pixels are grouped into patches."""
    cfg, model, pix, refs, _ = tiny
    outs = {}
    for impl in (2, 3, 4):
        for layout in ((1, 32, 32), (4, 16, 16), (0, 0, 0)):
            ctx = EmuContext(cfg.N, eps=cfg.eps)
            ctx.set_detector_layout(*layout)
            ctx.set_option("slice_impl", impl)
            ctx.prepare_model(model)
            outs[(impl, layout)] = ctx.slice(refs[:4], pix, SPF_OUT_COMPLEX)
    first = outs[(2, (1, 32, 32))]
    for k, v in outs.items():
        assert np.array_equal(v, first), k


@pytest.mark.parametrize("impl", [1, 2, 3, 4])
@pytest.mark.parametrize("N,eps", [(16, 1e-6), (21, 1e-9), (12, 1e-4)])
def test_emulated_slice_general_model_widths_and_even_n(impl, N, eps):
    """Non-even model (complex grid), even N, w = 8 / 10 / 6 (run-time width: reference gather only)."""
    rng = np.random.default_rng(4)
    A = rng.standard_normal((N, N, N)).astype(np.float32)
    pix = make_detector(1, 16)
    refs = random_quaternions(5, seed=31)
    ctx = EmuContext(N, eps=eps)
    ctx.set_option("slice_impl", impl)
    ctx.set_detector_layout(1, 16, 16)
    ctx.prepare_model(A)
    assert ctx.info.grid_is_real == 0
    c = ctx.slice(refs, pix, SPF_OUT_COMPLEX)
    assert _rel(c, orc.slice_points(A, refs, pix)) <= max(SLICE_TOL, 10 * eps)


@pytest.mark.parametrize("impl", [1, 2, 3, 4])
def test_emulated_slice_edge_cases(tiny, impl):
    cfg, model, pix, refs, c_ref = tiny
    ctx = EmuContext(cfg.N, eps=cfg.eps)
    ctx.set_option("slice_impl", impl)
    with pytest.raises(EmuError) as e:
        ctx.slice(refs[:1], pix)
    assert e.value.status == -4                                     # SPF_ESTATE before spf_prepare_model
    ctx.prepare_model(model)
    assert ctx.slice(refs[:0], pix).shape == (0, 1024) and ctx.slice(refs[:2], pix[:0]).shape == (2, 0)
    # ragged P, unnormalised quaternions, q outside [-pi, pi], points at the very edge of the period
    c = ctx.slice((3.0 * refs[:3]).astype(np.float32), pix[:777], SPF_OUT_COMPLEX)
    assert _rel(c, c_ref[:3, :777]) <= SLICE_TOL
    ident = np.array([[1, 0, 0, 0]], np.float32)
    far = (pix[:200].astype(np.float64) + 2 * np.pi * np.array([1, -1, 2])).astype(np.float32)
    assert _rel(ctx.slice(ident, far, SPF_OUT_COMPLEX), orc.slice_points(model, ident, far)) <= SLICE_TOL
    edge = np.array([[np.pi, -np.pi, 0.0], [-np.pi, np.pi, np.pi], [3.14159, 3.14159, -3.14159]], np.float32)
    # |c| ~ 1e-5 at the Nyquist edge against an rms of ~36 over the slices: the bar is absolute (reading s15)
    err = np.max(np.abs(ctx.slice(ident, edge, SPF_OUT_COMPLEX) - orc.slice_points(model, ident, edge)))
    assert err <= SLICE_TOL * np.sqrt(np.mean(np.abs(c_ref) ** 2))


# --------------------------------------------------------------------------------- a6-a8: spf_match

@pytest.mark.parametrize("variant", MATCHERS)
@pytest.mark.parametrize("n_img,M,P,masked", [(16, 64, 1024, False), (5, 300, 1000, True), (130, 257, 192, False),
                                              pytest.param(300, 513, 320, True, marks=full_only)])
def test_emulated_match_vs_oracle_ragged_sizes(variant, n_img, M, P, masked):
    rng = np.random.default_rng(n_img * 7 + M)
    S = (rng.random((M, P)) * rng.random((M, 1)) * 3).astype(np.float32)
    I = rng.poisson(S[rng.integers(0, M, n_img)]).astype(np.float32)
    mask = (rng.random(P) > 0.2).astype(np.uint8) if masked else None
    ctx = EmuContext(8, sm_count=4)              # 4 SMs: 4 (2) persistent clusters, so clusters take several tiles
    _matcher(ctx, variant)
    eb.counters()
    bi, bd, prods = ctx.match(I, S, mask)
    n = eb.counters()
    assert prods == (0 if variant == "simt" else 2)              # photon counts: one fp16 image plane
    tc = variant in ("cg1", "cg2")                                # only the tcgen05 matcher issues tcgen05.mma and bulk tensor copies
    assert (n["mmas"] > 0) == tc and (n["tma_copies"] > 0) == tc
    _check_match(bi, bd, I, S, mask)
    if n_img * M <= 2000:                                        # the independent CUDA-core reference kernels (one block per
        ri, rd, dist = ctx.match_reference(I, S, mask)           # pair: only the small cases are affordable under emulation)
        assert np.allclose(dist, orc.distances(I, S, mask), rtol=1e-6)
        assert np.array_equal(ri, bi) or variant != "simt"


def test_emulated_mma_matcher_shared_memory_accesses_are_conflict_free():
    """k_match_mma's XOR swizzle (chunk ^ (row / 2) mod 4 over 64-byte rows): every ldmatrix phase (8 rows of 16 bytes)
    and every quarter-warp of cp.async.16 stores touches 8 distinct 16-byte bank groups, i.e. takes ONE shared-memory
    wavefront -- counted from the addresses the kernel's own source produces, for the one-plane and the two-plane
    (non-integer images) instantiation.  A model of the bank rule, not a hardware counter."""
    rng = np.random.default_rng(5)
    for integer_images in (True, False):
        S = (rng.random((140, 320)) * 3).astype(np.float32)
        I = rng.poisson(S[rng.integers(0, 140, 130)]).astype(np.float32)
        if not integer_images:
            I = I + rng.random(I.shape).astype(np.float32)
        ctx = EmuContext(8, sm_count=4)
        _matcher(ctx, "mma")
        eb.smem_counters()
        bi, bd, prods = ctx.match(I, S, None)
        n = eb.smem_counters()
        assert prods == (2 if integer_images else 3)
        assert n["ldsm_phases"] > 0 and n["ldsm_wavefronts"] == n["ldsm_phases"], n
        assert n["cpasync_groups"] > 0 and n["cpasync_wavefronts"] == n["cpasync_groups"], n
        _check_match(bi, bd, I, S, None)


@pytest.mark.parametrize("variant", ["mma", "cg1", "cg2"])
@pytest.mark.parametrize("chunk", [1, 3, 0])
def test_emulated_tcgen05_epilogue_without_refinement(variant, chunk):
    """The contraction's own a_i + b_m - 2 G (match_refine = 0), with the accumulator drained every 1 or 3 K blocks
    (both TMEM stages, many hand-overs between the MMA issuer and the epilogue warps) or once (chunk 0)."""
    rng = np.random.default_rng(11)
    n_img, M, P = 140, 300, 448
    S = (rng.random((M, P)) * 2).astype(np.float32)
    I = rng.poisson(S[rng.integers(0, M, n_img)]).astype(np.float32)
    ctx = EmuContext(8, sm_count=2)
    _matcher(ctx, variant)
    ctx.set_option("match_refine", 0)
    ctx.set_option("match_chunk_kblocks", chunk)
    bi, bd, prods = ctx.match(I, S)
    assert prods == 2
    worst = _check_match(bi, bd, I, S)
    assert worst < 2e-5


@pytest.mark.parametrize("variant", MATCHERS)
def test_emulated_match_planted_ties_and_general_values(variant):
    rng = np.random.default_rng(17)
    M, P = 200, 640
    S = rng.random((M, P)).astype(np.float32)
    S[150] = S[20]                                               # exact duplicate: the lowest index must win
    planted = np.array([20, 0, 199, 77])
    I = S[planted].copy()                                        # non-integer images: two fp16 image planes, 3 products
    ctx = EmuContext(8, sm_count=4)
    _matcher(ctx, variant)
    bi, bd, prods = ctx.match(I, S)
    assert list(bi) == list(planted) and prods == (0 if variant == "simt" else 3)
    nrm = (I.astype(np.float64) ** 2).sum(1) + (S[planted].astype(np.float64) ** 2).sum(1)
    assert np.all(np.abs(bd) <= 1e-6 * nrm)                      # reading s14, the noise-free case
    # counts above 2,048 (not exact in one fp16 term) at d ~ 3e-4 of the norms: same 1e-4 d bar (conditioning + refinement)
    S3 = (3000.0 * S).astype(np.float32)
    I2 = rng.poisson(3000.0 * S[rng.integers(0, M, 9)]).astype(np.float32)
    bi, bd, _ = ctx.match(I2, S3)
    _check_match(bi, bd, I2, S3)
    bi4, bd4, _ = ctx.match(4 * I2, 4 * S3)                      # power-of-two scaling passes through exactly
    assert np.array_equal(bi4, bi) and np.allclose(bd4, 16 * bd, rtol=1e-6)
    perm = rng.permutation(M)                                    # permuting the reference set permutes the answer
    bip, bdp, _ = ctx.match(I2, S3[perm])
    assert np.array_equal(perm[bip], bi) and np.allclose(bdp, bd, rtol=1e-5)
    with pytest.raises(EmuError):
        ctx.match(I, S[:0])


# --------------------------------------------------------------------------------- the whole path

@pytest.mark.parametrize("impl,variant", [(1, "simt"), pytest.param(3, "simt", marks=full_only), (4, "mma"),
                                          pytest.param(2, "cg1", marks=full_only), (2, "cg2")])
def test_emulated_end_to_end_tiny_poisson(tiny, impl, variant):
    """Tiny (BASELINE.json:configs[0]) end to end: everything from the oracle on one side, everything from the
    emulated kernels on the other -- the library defaults, and the TMA-staged slicer with each tcgen05 matcher."""
    cfg, model, pix, refs, c_ref = tiny
    truth, _ = planted_truth_quaternions(cfg.n_img, refs)
    alpha = photon_scale(c_ref.real, None, cfg.photons)
    images = poisson_images(alpha * orc.slice_points(model, truth, pix).real)
    ctx = EmuContext(cfg.N, eps=cfg.eps)
    ctx.set_detector_layout(1, 32, 32)
    ctx.set_option("slice_impl", impl)
    _matcher(ctx, variant)
    ctx.prepare_model(model)
    slices = ctx.slice(refs, pix, SPF_OUT_INTENSITY, scale=alpha)
    bi, bd, _ = ctx.match(images, slices)
    oi, od, osd, _ = orc.match(images, alpha * c_ref.real)        # the oracle's own fp64 slices
    near = (osd - od) <= DIST_TOL * od
    assert np.all((bi == oi) | near) and np.all(np.abs(bd - od) <= DIST_TOL * od)
    hi, hd, hs = ctx.orientation_match_host(model, refs, pix, images, scale=alpha)     # the host-buffer entry point
    assert np.array_equal(hi, bi) and np.array_equal(hd, bd) and np.array_equal(hs, slices)


def test_emulated_paper_scale_geometry_sampled(monkeypatch):
    """Paper-scale model, fine grid (320^3) and detector (4 panels of 128 x 128, 8 x 16 lattice patches), one orientation:
    512 blocks of each slicer on the real geometry -- every tile of the staged variant must fit and stage (no fallback) --
    with the FFT stub in fp32 (the arithmetic cuFFT uses), 1,024 sampled points from the oracle.  At w = 8 (reading
    s10b) the error is below 1e-6; w = 7 left 6e-6 here and up to 1.8e-5 on other samples."""
    monkeypatch.setenv("SPF_EMU_FFT32", "1")
    cfg = CONFIGS["paper_scale"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(1, seed=2)
    ctx = EmuContext(cfg.N, eps=cfg.eps)
    assert (ctx.info.n_fine, ctx.info.w) == (320, 8)
    ctx.set_detector_layout(cfg.panels, cfg.panel_edge, cfg.panel_edge)
    ctx.prepare_model(model)
    assert ctx.info.grid_is_real == 1
    rng = np.random.default_rng(6)
    sj = rng.integers(0, cfg.P, 1024)
    ref = orc.slice_points(model, refs, pix, np.zeros(1024, np.int64), sj)
    outs = {}
    for impl in (1, 2, 4):
        ctx.set_option("slice_impl", impl)
        eb.counters()
        outs[impl] = ctx.slice(refs, pix, SPF_OUT_COMPLEX)
        n = eb.counters()
        err = _rel(outs[impl][0, sj], ref)
        print("paper-scale geometry, slice_impl %d: relative L2 %.2e, %d bulk tensor copies" % (impl, err, n["tma_copies"]))
        assert err <= 2e-6
        if impl == 2:
            assert n["tma_copies"] >= 512 * 8                  # every one of the 512 blocks staged its box, >= 8 x-planes each
    assert _rel(outs[2], outs[1]) <= 2e-6 and np.array_equal(outs[4], outs[2])


def test_emulated_spf_selftest_checks_and_switches_variants_on(tiny):
    """spf_selftest (the C library's own variant check) executed under the emulator: every variant
    agrees with the reference kernels on the check's seeded cases, a passing matcher becomes the context's choice
    (pairs supersede single CTAs), and a C caller needs no other option to reach the TMA / tcgen05 kernels."""
    cfg, model, pix, refs, c_ref = tiny
    ctx = EmuContext(cfg.N, eps=cfg.eps, sm_count=4)
    ctx.set_option("selftest_small", 1)
    with pytest.raises(EmuError) as e:
        ctx.selftest("slice_coop")
    assert e.value.status == -4                       # slicers check the caller's own model: SPF_ESTATE before prepare
    ctx.prepare_model(model)
    for v in (("slice_gcoop", "slice_coop_ld", "slice_coop", "match_mma", "match_cg1", "match_cg2") if FULL else ("slice_coop_ld", "slice_coop", "match_cg2")):
        r = ctx.selftest(v)
        print(v, r)
        assert r["passed"], r
        assert r["worst_rel"] <= (3e-6 if v.startswith("slice") else 1e-4)
    with pytest.raises(EmuError):
        ctx.selftest("no_such_variant")
    # the matcher is now the tcgen05 pair kernel with no option set by the caller: MMAs are issued
    rng = np.random.default_rng(2)
    S = rng.random((70, 256)).astype(np.float32)
    I = rng.poisson(S[:9]).astype(np.float32)
    eb.counters()
    bi, bd, prods = ctx.match(I, S)
    assert prods == 2 and eb.counters()["mmas"] > 0
    _check_match(bi, bd, I, S)


@pytest.mark.parametrize("impl,variant", [(1, "simt"), pytest.param(4, "mma", marks=full_only),
                                          pytest.param(2, "cg1", marks=full_only), (2, "cg2")])
def test_emulated_streaming_slice_match_equals_the_two_step_path(tiny, impl, variant):
    """spf_slice_match: 64 orientations in ragged chunks of 24 -- the slice array never exists -- give
    the argmin and distances of spf_slice + spf_match, and agree with the oracle end to end."""
    cfg, model, pix, refs, c_ref = tiny
    truth, _ = planted_truth_quaternions(cfg.n_img, refs)
    alpha = photon_scale(c_ref.real, None, cfg.photons)
    images = poisson_images(alpha * orc.slice_points(model, truth, pix).real)
    mask = (np.random.default_rng(1).random(cfg.P) > 0.05).astype(np.uint8)
    ctx = EmuContext(cfg.N, eps=cfg.eps)
    ctx.set_detector_layout(1, 32, 32)
    ctx.set_option("slice_impl", impl)
    _matcher(ctx, variant)
    ctx.prepare_model(model)
    slices = ctx.slice(refs, pix, SPF_OUT_INTENSITY, scale=alpha)
    bi2, bd2, _ = ctx.match(images, slices, mask)
    bi, bd = ctx.slice_match(refs, pix, images, scale=alpha, mask=mask, chunk_M=24)
    assert np.array_equal(bi, bi2)
    assert np.allclose(bd, bd2, rtol=(0 if variant == "simt" else 1e-6), atol=0)
    oi, od, osd, _ = orc.match(images, alpha * c_ref.real, mask)
    near = (osd - od) <= DIST_TOL * od
    assert np.all((bi == oi) | near) and np.all(np.abs(bd - od) <= DIST_TOL * od)
    one, _ = ctx.slice_match(refs, pix, images, scale=alpha, mask=mask, chunk_M=1000)     # chunk_M > M: a single chunk
    assert np.array_equal(one, bi)
