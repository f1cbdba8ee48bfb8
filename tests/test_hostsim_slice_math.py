"""CPU check of the CUDA path's interpolation ARITHMETIC (steps a1-a5) against the oracle.

tests/hostsim/spf_hostsim.cpp compiles paper_2109_05339_b200/csrc/spf_slice_math.cuh -- the header
k_slice and spf_create include -- with g++.  This is NOT GPU parity (the kernels themselves, their
shared-memory staging, cuFFT's fp32 rounding and the launch logic are not exercised); it shows that the
formulas the kernels evaluate (deapodisation, fold/ceil/fraction split, polynomial weights, w^3 sum,
centred grid with periodic halo) reach the oracle within the north_star tolerance.  The fine grid is
built here with NumPy following spf_prepare.cu step by step, FFT in fp64 then stored as complex64.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from oracle import oracle as orc
from spf_inputs import CONFIGS, make_model, make_detector, random_quaternions, sample_pairs

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "hostsim")
SLICE_TOL = 1e-5


@pytest.fixture(scope="module")
def sim():
    src, lib = os.path.join(HERE, "spf_hostsim.cpp"), os.path.join(HERE, "libspf_hostsim.so")
    hdr = os.path.join(HERE, "..", "..", "paper_2109_05339_b200", "csrc", "spf_slice_math.cuh")
    if not os.path.exists(lib) or os.path.getmtime(lib) < max(os.path.getmtime(src), os.path.getmtime(hdr)):
        subprocess.run(["g++", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c++17", "-ffp-contract=off", src, "-o", lib], check=True)
    L = C.CDLL(lib)
    L.hostsim_deapod.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p]
    L.hostsim_fit.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
    L.hostsim_fit.restype = C.c_int
    L.hostsim_slice.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_long,
                                C.c_void_p, C.c_long, C.c_int, C.c_void_p]
    L.hostsim_cell.argtypes = [C.c_double, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    L.hostsim_slice_blocks.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_long,
                                       C.c_void_p, C.c_long, C.c_void_p, C.c_long, C.c_int, C.c_uint, C.c_void_p, C.c_void_p]
    L.hostsim_tile_geom.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint, C.c_void_p]
    L.hostsim_scatter_model.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p]
    L.hostsim_relayout.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
    L.hostsim_count_uneven.argtypes = [C.c_void_p, C.c_int]
    L.hostsim_count_uneven.restype = C.c_long
    L.hostsim_patch_table.argtypes = [C.c_int, C.c_int, C.c_int, C.c_long, C.c_void_p, C.c_long]
    L.hostsim_patch_table.restype = C.c_long
    return L


def _plan(N, eps):
    w = min(max(int(np.ceil(np.log10(1.0 / eps) - 1e-9)) + 2, 3), 10)      # spf_plan_kernel_width (reading s10b)
    nf = 2 * N + (2 * N) % 2
    while True:
        v = nf
        for p in (2, 3, 5, 7):
            while v % p == 0:
                v //= p
        if v == 1:
            break
        nf += 2
    halo = (w + 1) // 2 + 1
    return w, nf, halo


def _padded_grid(sim, A, w, nf, halo):
    """spf_prepare_model on the CPU: deapodise + scatter (k_deapod_pad) and the centred layout with periodic halo
    (k_relayout) through the header's own index maps, host-compiled; the forward FFT in between is NumPy's, in
    fp64, stored as complex64 (cuFFT's fp32 rounding is what this replay does not see)."""
    N = A.shape[0]
    p = np.empty(N)
    sim.hostsim_deapod(N, nf, w, p.ctypes.data)
    p32 = p.astype(np.float32)
    fine = np.zeros((nf, nf, nf), np.complex64)
    sim.hostsim_scatter_model(np.ascontiguousarray(A, np.float32).ctypes.data, p32.ctypes.data, N, nf, fine.ctypes.data)
    # independent restatement of the scatter (deapodised model at index n mod n_f): the two must agree exactly
    idx = (np.arange(N) - N // 2) % nf
    want = np.zeros((nf, nf, nf), np.complex64)
    want[np.ix_(idx, idx, idx)] = (A * (p32[:, None, None] * p32[None, :, None])) * p32[None, None, :]
    assert np.array_equal(fine, want)
    b = np.ascontiguousarray(np.fft.fftn(fine.astype(np.complex128)).astype(np.complex64))
    npad = nf + 2 * halo
    sz = (npad + 3) & ~3
    g = np.empty((npad, npad, sz), np.complex64)
    sim.hostsim_relayout(b.ctypes.data, nf, npad, sz, nf // 2 + halo, g.ctypes.data)
    l = (np.arange(npad) - (nf // 2 + halo)) % nf
    assert np.array_equal(g[:, :, :npad], b[np.ix_(l, l, l)]) and not g[:, :, npad:].any()
    return g, npad, sz


def _slice(sim, g, is_real, npad, sz, nf, halo, w, quats, pix, use_poly):
    grid = np.ascontiguousarray(g.real.astype(np.float32)) if is_real else np.ascontiguousarray(g).view(np.float32)
    quats, pix = np.ascontiguousarray(quats, np.float32), np.ascontiguousarray(pix, np.float32)
    out = np.empty((quats.shape[0], pix.shape[0]), np.complex64)
    sim.hostsim_slice(grid.ctypes.data, int(is_real), npad, sz, nf, halo, w, quats.ctypes.data, quats.shape[0],
                      pix.ctypes.data, pix.shape[0], int(use_poly), out.ctypes.data)
    return out


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_evenness_check_decides_when_the_fine_grid_is_real(sim):
    """k_check_even's rule (replayed): zero voxels break A[n] == A[-n] exactly when the transform of the model is
    real -- odd N: plain point symmetry about the centre voxel; even N: the unpaired index-0 planes must be zero."""
    rng = np.random.default_rng(2)
    count = lambda A: sim.hostsim_count_uneven(np.ascontiguousarray(A, np.float32).ctypes.data, A.shape[0])
    imag_frac = lambda A: (lambda F: float(np.abs(F.imag).max() / np.abs(F.real).max()))(
        np.fft.fftn(np.roll(A.astype(np.float64), [-(A.shape[0] // 2)] * 3, (0, 1, 2))))
    tiny = CONFIGS["tiny"]
    A = make_model(tiny.N, tiny.n_atoms, tiny.atom_radius)
    assert count(A) == 0 and imag_frac(A) < 1e-12
    B = A.copy(); B[3, 4, 5] += 1e-3
    assert count(B) == 2 and imag_frac(B) > 1e-6               # the voxel and its partner
    for N in (8, 12):
        R = rng.standard_normal((N, N, N)).astype(np.float32)
        idx = (N - np.arange(N)) % N                            # mirror about index N/2: i -> N - i (index 0 maps to itself)
        S = (0.5 * (R + R[np.ix_(idx, idx, idx)])).astype(np.float32)
        assert count(S) > 0                                     # index-0 planes are not zero: unpaired frequencies
        S[0] = 0; S[:, 0] = 0; S[:, :, 0] = 0
        assert count(S) == 0 and imag_frac(S) < 1e-6
        assert count(R) > 0


def test_polynomial_weights_reach_1e7(sim):
    """Only the w = 7 and w = 10 kernels use the polynomial weights (other widths evaluate expf/sqrtf);
    at small w the sqrt singularity at the support edge (amplitude exp(-beta)) defeats a degree-12 fit."""
    for w in (7, 10):
        coef = np.zeros((16, 13), np.float32)
        worst = C.c_double()
        deg = sim.hostsim_fit(w, coef.ctypes.data, C.byref(worst))
        assert 6 <= deg <= 12 and worst.value < 1e-7, (w, deg, worst.value)


@pytest.mark.parametrize("use_poly,is_real", [(1, 1), (0, 1), (1, 0)])
def test_tiny_full_vs_oracle(sim, use_poly, is_real):
    cfg = CONFIGS["tiny"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    assert (w, nf) == (8, 42)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    assert np.abs(g.imag).max() <= 1e-5 * np.abs(g.real).max()        # even model => real fine grid
    c = _slice(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, use_poly)
    ref = orc.slice_points(A, refs, pix)
    assert _rel(c.real if is_real else c, ref.real if is_real else ref) <= SLICE_TOL
    worst = max(_rel(c[m].real, ref[m].real) for m in range(cfg.M))
    assert worst <= 3 * SLICE_TOL


def test_small_sampled_vs_oracle(sim):
    """Small (configs[1]): 81^3 model, n_fine 162; 64 orientations x 16,384 pixels, 2,048 sampled pairs from the oracle."""
    cfg = CONFIGS["small"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(64, seed=2)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    c = _slice(sim, g, 1, npad, sz, nf, halo, w, refs, pix, 1)
    sm, sj = sample_pairs(64, cfg.P, 2048)
    ref = orc.slice_points(A, refs, pix, sm, sj)
    assert _rel(c[sm, sj].real, ref.real) <= SLICE_TOL


def test_general_complex_model_even_n_and_wide_kernel(sim):
    rng = np.random.default_rng(4)
    for N, eps in ((16, 1e-6), (21, 1e-9)):
        A = rng.standard_normal((N, N, N)).astype(np.float32)
        pix = make_detector(1, 16)
        refs = random_quaternions(5, seed=31)
        w, nf, halo = _plan(N, eps)
        g, npad, sz = _padded_grid(sim, A, w, nf, halo)
        c = _slice(sim, g, 0, npad, sz, nf, halo, w, refs, pix, 1 if w in (7, 10) else 0)
        assert _rel(c, orc.slice_points(A, refs, pix)) <= SLICE_TOL


def test_cell_index_stays_inside_the_padded_grid(sim):
    """Every coordinate -- in range, at the period edge, far outside, NaN, inf -- gives a first cell in
    [0, np - w], so the w taps never leave the padded grid (the clamp only acts on non-finite input)."""
    p, f = C.c_int(), C.c_float()
    for w, nf in ((7, 42), (7, 320), (10, 405), (2, 8)):
        halo = (w + 1) // 2 + 1
        npad = nf + 2 * halo
        xs = list(np.linspace(-np.pi, np.pi, 2001)) + [np.pi, -np.pi, np.nextafter(np.pi, 4), 7 * np.pi, -123.456, 1e300,
                                                        float("nan"), float("inf"), float("-inf")]
        lo, hi = npad, -1
        for x in xs:
            sim.hostsim_cell(float(x), nf, halo, w, C.byref(p), C.byref(f))
            assert 0 <= p.value <= npad - w, (w, nf, x, p.value)
            assert -0.5 * w - 1e-6 <= f.value <= 1.0
            if np.isfinite(x) and abs(x) <= np.pi:
                lo, hi = min(lo, p.value), max(hi, p.value)
        assert lo >= 1 and hi + w - 1 <= npad - 2      # finite in-range input never touches the clamp


def test_paper_scale_sampled_vs_oracle(sim):
    """Paper-scale model (configs[2]: 151^3, n_fine 320, w 8): 8 orientations x 65,536 pixels through the
    host-compiled arithmetic, 2,048 sampled pairs from the oracle.  The thinnest margin of the configs."""
    cfg = CONFIGS["paper_scale"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(8, seed=2)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    assert (w, nf) == (8, 320)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    c = _slice(sim, g, 1, npad, sz, nf, halo, w, refs, pix, 1)
    sm, sj = sample_pairs(8, cfg.P, 2048)
    ref = orc.slice_points(A, refs, pix, sm, sj)
    err = _rel(c[sm, sj].real, ref.real)
    print("paper-scale host-compiled slice arithmetic vs oracle: rel L2 %.3e" % err)
    assert err <= SLICE_TOL


# ------------------------------------------------------------------------------------------------
# staged kernel (slice_impl 2) and its global-memory twin (3): block-level replay of the tile staging and of the warp-per-point gather
# ------------------------------------------------------------------------------------------------
def _patch_table(sim, panels, rows, cols, P):
    """The table spf_slice itself builds (build_patch_table, spf_slice_math.cuh), through the host-compiled header."""
    n = sim.hostsim_patch_table(panels, rows, cols, P, None, 0)
    tab = np.empty(n, np.int32)
    assert sim.hostsim_patch_table(panels, rows, cols, P, tab.ctypes.data, n) == n
    return tab


def test_patch_table_covers_every_pixel_once(sim):
    """Lattice layout: 8 x 16 tiles of one panel, ragged panel edges padded with -1; no promise (or a promise that
    does not multiply out to P): runs of 128 consecutive pixels.  Every pixel index appears exactly once."""
    for panels, rows, cols, P in ((1, 32, 32, 1024), (4, 128, 128, 65536), (1, 40, 40, 1600), (3, 9, 17, 459),
                                  (0, 0, 0, 777), (2, 16, 16, 500), (0, 0, 0, 128), (1, 1, 1, 1)):
        tab = _patch_table(sim, panels, rows, cols, P)
        assert len(tab) % 128 == 0
        real = tab[tab >= 0]
        assert len(real) == P and np.array_equal(np.sort(real), np.arange(P))
        lattice = panels > 0 and panels * rows * cols == P
        if lattice:
            assert len(tab) == panels * -(-rows // 8) * -(-cols // 16) * 128
            first = tab[:128].reshape(8, 16)                   # first tile of panel 0: rows 0..7 x cols 0..15
            rr, cc = np.meshgrid(np.arange(8), np.arange(16), indexing="ij")
            want = np.where((rr < rows) & (cc < cols), rr * cols + cc, -1)
            assert np.array_equal(first, want)
        else:
            assert len(tab) == -(-P // 128) * 128 and np.array_equal(tab[:P], np.arange(P))


def _slice_blocks(sim, g, is_real, npad, sz, nf, halo, w, quats, pix, table, coop, cap=None):
    grid = np.ascontiguousarray(g.real.astype(np.float32)) if is_real else np.ascontiguousarray(g).view(np.float32)
    quats, pix = np.ascontiguousarray(quats, np.float32), np.ascontiguousarray(pix, np.float32)
    out = np.full((quats.shape[0], pix.shape[0]), np.nan + 0j, np.complex64)
    stats = np.zeros(3, np.int64)
    if cap is None:
        cap = 48 * 1024 * (1 if is_real else 2)    # launch_slice (spf_slice.cu)
    sim.hostsim_slice_blocks(grid.ctypes.data, int(is_real), npad, sz, nf, halo, w, quats.ctypes.data, quats.shape[0],
                             pix.ctypes.data, pix.shape[0], table.ctypes.data, len(table) // 128, int(coop), cap,
                             out.ctypes.data, stats.ctypes.data)
    return out, stats


@pytest.mark.parametrize("coop,is_real,layout", [(1, 1, True), (1, 0, True), (1, 1, False), (1, 0, False),
                                                 (2, 1, True), (2, 0, False)])
def test_staged_block_replay_tiny_full_vs_oracle(sim, coop, is_real, layout):
    """Tiny through the staged data path: every block's tile image holds NaN wherever no TMA copy writes,
    so a finite result within tolerance shows every read (zero-weight window padding included) stays
    inside the staged box, and that the tile indexing and the lane decomposition add up to the w^3 sum."""
    cfg = CONFIGS["tiny"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    table = _patch_table(sim, 1, 32, 32, cfg.P) if layout else _patch_table(sim, 0, 0, 0, cfg.P)
    c, stats = _slice_blocks(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, table, coop)
    assert np.isfinite(c.view(np.float32)).all()
    assert (stats[0] > 0 or coop == 2) and stats[0] + stats[1] == cfg.M * (len(table) // 128)
    if coop == 2:
        assert stats[0] == 0          # variant 3 stages nothing: the warp walks the padded grid itself
    ref = orc.slice_points(A, refs, pix)
    assert _rel(c.real if is_real else c, ref.real if is_real else ref) <= SLICE_TOL
    # and it is the same arithmetic as the one-thread-per-point gather from the whole grid, up to summation order
    direct = _slice(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, 1)
    assert _rel(c, direct) <= 2e-6


def test_staged_block_replay_ragged_patch_and_complex_general_model(sim):
    """Ragged last patch (P not a multiple of 128) and a non-even model on the complex grid, N even."""
    rng = np.random.default_rng(4)
    N = 16
    A = rng.standard_normal((N, N, N)).astype(np.float32)
    pix = make_detector(1, 16)[:200]
    refs = random_quaternions(5, seed=31)
    w, nf, halo = _plan(N, 1e-6)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    table = _patch_table(sim, 0, 0, 0, 200)
    ref = orc.slice_points(A, refs, pix)
    c, stats = _slice_blocks(sim, g, 0, npad, sz, nf, halo, w, refs, pix, table, 1)
    assert np.isfinite(c.view(np.float32)).all() and stats[0] > 0
    assert _rel(c, ref) <= SLICE_TOL


def test_warp_per_point_fallback_blocks_equal_the_staged_ones(sim):
    """A block of variant 2 whose box does not fit the tile walks the padded grid instead (the path variant 3 always
    takes): same lanes, same weights, same exchange order, so the results are bit-identical to the staged ones."""
    cfg = CONFIGS["tiny"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(8, seed=2)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    table = _patch_table(sim, 1, 32, 32, cfg.P)
    for is_real in (1, 0):
        staged, st1 = _slice_blocks(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, table, 1)
        forced, st2 = _slice_blocks(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, table, 1, cap=1024)
        direct, st3 = _slice_blocks(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, table, 2)
        assert st1[0] > 0 and st2[0] == 0 and st3[0] == 0
        assert np.array_equal(staged, forced) and np.array_equal(staged, direct)


def test_wide_warp_per_point_replay(sim):
    """w = 10 through variant 3's 16-cell window (2 rows x 16 cells per load, idle lanes beyond the 10th cell, 44-float
    weight sets): real and complex grid against the oracle, and against the one-thread-per-point sum."""
    rng = np.random.default_rng(9)
    N = 21
    w, nf, halo = _plan(N, 1e-9)
    pix = make_detector(1, 32)[:1000]               # ragged: the last patch is partly empty
    refs = random_quaternions(4, seed=31)
    table = _patch_table(sim, 0, 0, 0, 1000)
    for is_real in (1, 0):
        A = make_model(N, 12, 5.0) if is_real else rng.standard_normal((N, N, N)).astype(np.float32)
        g, npad, sz = _padded_grid(sim, A, w, nf, halo)
        c, stats = _slice_blocks(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, table, 2)
        assert np.isfinite(c.view(np.float32)).all() and stats[0] == 0
        ref = orc.slice_points(A, refs, pix)
        assert _rel(c.real if is_real else c, ref.real if is_real else ref) <= SLICE_TOL
        direct = _slice(sim, g, is_real, npad, sz, nf, halo, w, refs, pix, 1)
        assert _rel(c, direct) <= 2e-6


def test_staged_block_replay_paper_scale_sampled(sim):
    """Paper-scale model and detector (8 x 16 lattice patches of 4 x 128 x 128 pixels), 4 orientations through the
    warp-per-point path: every block must fit the 48 KB tile (no fallback), 2,048 sampled pairs from the oracle."""
    cfg = CONFIGS["paper_scale"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(4, seed=2)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    table = _patch_table(sim, cfg.panels, cfg.panel_edge, cfg.panel_edge, cfg.P)
    c, stats = _slice_blocks(sim, g, 1, npad, sz, nf, halo, w, refs, pix, table, 1)
    assert stats[1] == 0 and stats[2] <= 48 * 1024, stats
    assert np.isfinite(c.view(np.float32)).all()
    sm, sj = sample_pairs(4, cfg.P, 2048)
    ref = orc.slice_points(A, refs, pix, sm, sj)
    err = _rel(c[sm, sj].real, ref.real)
    print("paper-scale warp-per-point replay vs oracle: rel L2 %.3e; largest tile %d bytes" % (err, stats[2]))
    assert err <= SLICE_TOL


def test_tile_geometry_menu_and_bank_rule(sim):
    """tile_geom: an accepted box is on the tensor-map menu, covers the points' footprint plus the 8 x 8 window's
    spare row and cell (w = 7; none at w = 8), keeps x-planes 128-byte aligned, fits the capacity, and has a row pitch of 8 mod 16 cells --
    the four rows a warp reads at once then fall into four disjoint groups of 8 banks (real grid) or, per
    half-warp, two disjoint groups of 16 banks (complex grid).  w > 8 is never staged."""
    out = (C.c_int * 4)()
    for cell in (4, 8):
        cap = 48 * 1024 * (cell // 4)
        sim.hostsim_tile_geom(13, 20, 20, 10, cell, cap, out)
        assert out[3] == 0                      # the 8 x 8 window does not cover a 10-wide kernel
        for w, Lx in ((7, 7), (8, 8), (8, 13), (7, 22), (8, 22), (8, 30)):
            spare = 8 - w                       # the 8 x 8 window reads `spare` rows and cells past the w taps
            for Ly in range(w, 45):
                for Lz in range(w, 45):
                    sim.hostsim_tile_geom(Lx, Ly, Lz, w, cell, cap, out)
                    by, bz, S1, ok = out[0], out[1], out[2], out[3]
                    if not ok:
                        assert by > 40 or bz > 40 or Lz + spare > 40 or Lx * S1 * cell > cap
                        continue
                    assert by in range(8, 41, 4) and bz in range(8, 41, 4)
                    assert by >= Ly + spare and bz >= Lz + spare and S1 >= by * bz and (S1 * cell) % 128 == 0
                    assert Lx * S1 * cell <= cap
                    assert bz % 16 == 8
                    if cell == 4:
                        banks = sorted((h * bz + k) % 32 for h in range(4) for k in range(8))
                        assert banks == list(range(32))
                    else:
                        for half in (0, 2):
                            words = sorted(((h * bz + k) * 2 + e) % 32 for h in (half, half + 1) for k in range(8) for e in (0, 1))
                            assert words == list(range(32))


def test_bank_conflicts_thread_per_point_vs_warp_per_point():
    """Why slice_impl 2 gathers with a WARP per point, and why the round-1 one-thread-per-point staged form (variant 0)
    was deleted.  With one thread per point the 32 lanes of a warp read, at
    every tap, 32 words whose tile addresses follow the rotated pixel lattice -- generic orientations spread them
    over the 32 banks like random throws, and the load replays max-bank-multiplicity times.  Paper-scale
    geometry, seeded orientations: the mean replay factor is above 3, i.e. w^3 x 3.5 / 32 = 56 shared-memory
    wavefronts per point at w = 8, against 16 + 4 for the warp-per-point form whose lanes read 32 consecutive-bank words."""
    cfg = CONFIGS["paper_scale"]
    pix = make_detector(cfg.panels, cfg.panel_edge).astype(np.float64)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    off = nf // 2 + halo
    rng = np.random.default_rng(0)
    degs = []
    for q in random_quaternions(12, seed=9).astype(np.float64):
        qw, x, y, z = q / np.linalg.norm(q)
        R = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - qw * z), 2 * (x * z + qw * y)],
                      [2 * (x * y + qw * z), 1 - 2 * (x * x + z * z), 2 * (y * z - qw * x)],
                      [2 * (x * z - qw * y), 2 * (y * z + qw * x), 1 - 2 * (x * x + y * y)]])
        i0 = (np.ceil((pix @ R.T) * nf / (2 * np.pi) - w / 2).astype(int) + off).reshape(cfg.panels, cfg.panel_edge, cfg.panel_edge, 3)
        for _ in range(40):
            p, r0, c0 = rng.integers(cfg.panels), 8 * rng.integers(cfg.panel_edge // 8), 16 * rng.integers(cfg.panel_edge // 16)
            t = i0[p, r0:r0 + 8, c0:c0 + 16].reshape(-1, 3)
            lo = t.min(0)
            L = t.max(0) - lo + w
            by, bz = max(8, (L[1] + 3) // 4 * 4), max(8, (L[2] + 3) // 4 * 4)
            S1 = (by * bz + 31) // 32 * 32
            addr = (t[:, 0] - lo[0]) * S1 + (t[:, 1] - lo[1]) * bz + (t[:, 2] - lo[2])
            for wv in range(4):
                a = addr[32 * wv:32 * wv + 32]
                degs.append(max(len(set(a[a % 32 == b])) for b in set(a % 32)))
    mean = float(np.mean(degs))
    print("thread-per-point staged gather: mean bank-conflict degree %.2f over %d warps" % (mean, len(degs)))
    assert 3.0 < mean < 4.5
    assert w ** 3 * mean / 32 > 2 * (2 * w + 4)
