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
    return L


def _plan(N, eps):
    w = int(np.ceil(np.log10(1.0 / eps) - 1e-9)) + 1
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
    """spf_prepare_model in NumPy: deapodise (fp32, the kernel's operand order), scatter at n mod n_f,
    forward FFT, centred layout with periodic halo (padded index p <-> fine cell (p - off) mod n_f)."""
    N = A.shape[0]
    p = np.empty(N)
    sim.hostsim_deapod(N, nf, w, p.ctypes.data)
    p32 = p.astype(np.float32)
    v = (A * (p32[:, None, None] * p32[None, :, None])) * p32[None, None, :]
    fine = np.zeros((nf, nf, nf), np.complex64)
    idx = (np.arange(N) - N // 2) % nf
    fine[np.ix_(idx, idx, idx)] = v
    b = np.fft.fftn(fine.astype(np.complex128)).astype(np.complex64)
    npad = nf + 2 * halo
    sz = (npad + 3) & ~3
    l = (np.arange(npad) - (nf // 2 + halo)) % nf
    g = np.zeros((npad, npad, sz), np.complex64)
    g[:, :, :npad] = b[np.ix_(l, l, l)]
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
    assert (w, nf) == (7, 42)
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
    """Paper-scale model (configs[2]: 151^3, n_fine 320, w 7): 8 orientations x 65,536 pixels through the
    host-compiled arithmetic, 2,048 sampled pairs from the oracle.  The thinnest margin of the configs."""
    cfg = CONFIGS["paper_scale"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(8, seed=2)
    w, nf, halo = _plan(cfg.N, cfg.eps)
    assert (w, nf) == (7, 320)
    g, npad, sz = _padded_grid(sim, A, w, nf, halo)
    c = _slice(sim, g, 1, npad, sz, nf, halo, w, refs, pix, 1)
    sm, sj = sample_pairs(8, cfg.P, 2048)
    ref = orc.slice_points(A, refs, pix, sm, sj)
    err = _rel(c[sm, sj].real, ref.real)
    print("paper-scale host-compiled slice arithmetic vs oracle: rel L2 %.3e" % err)
    assert err <= SLICE_TOL
