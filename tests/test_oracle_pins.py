"""Pins for the oracle (-m "not gpu").  Each test checks oracle/ against something that is NOT the
oracle: a closed form, a library routine on a special case, an invariant, brute force.

The paper prints no worked numerical example (PAPER.md has no numbers for slicing or matching), so
there are no paper-value fixtures; what the paper and the mathematics fix is listed in
SURVEY.md section 8(c) "What pins each part" and is what is tested here.
"""
import numpy as np
import pytest
from scipy.spatial.distance import cdist

from oracle import oracle as orc
from spf_inputs import CONFIGS, make_model, make_detector, random_quaternions


def _gauss_blob(N, r0, s):
    n = np.arange(N) - N // 2
    g = [np.exp(-((n - r0[d]) ** 2) / (2 * s * s)) for d in range(3)]
    return (g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]).astype(np.float64)


def _gauss_blob_ft(x, r0, s):
    """Closed form of sum_n exp(-|n-r0|^2/2s^2) exp(-i n.x) by Poisson summation:
    prod_d sqrt(2 pi) s sum_k exp(-i r0_d (x_d + 2 pi k)) exp(-s^2 (x_d + 2 pi k)^2 / 2)."""
    out = np.ones(x.shape[0], np.complex128)
    for d in range(3):
        acc = 0
        for k in (-2, -1, 0, 1, 2):
            y = x[:, d] + 2 * np.pi * k
            acc = acc + np.exp(-1j * r0[d] * y) * np.exp(-0.5 * s * s * y * y)
        out *= np.sqrt(2 * np.pi) * s * acc
    return out


@pytest.fixture(scope="module")
def pts():
    rng = np.random.default_rng(11)
    return rng.uniform(-np.pi, np.pi, size=(40, 3))


def test_nudft_gaussian_closed_form_pins_sign_centring_axis_order(pts):
    # off-centre with three DIFFERENT offsets: a wrong sign flips the phase, a wrong centre shifts
    # it, a swapped axis mixes r0 components, a wrong normalisation scales it -- all fail here.
    N, s, r0 = 31, 2.0, np.array([2.0, -1.0, 3.5])
    A = _gauss_blob(N, r0, s)
    A32 = A.astype(np.float32)
    ref = _gauss_blob_ft(pts, r0, s)
    for direct in (False, True):
        c = orc.nudft(A32, pts, direct=direct)
        # fp32 storage of the model bounds the agreement (6e-8 relative per voxel); the blob sits
        # >= 5.7 s from the nearest face so the truncated tail is < 1e-7 of the peak voxel.
        assert np.abs(c - ref).max() <= 5e-7 * np.abs(ref).max()


def test_nudft_equals_fftn_on_the_fourier_grid():
    # x = 2 pi k / N  =>  c(x_k) = fftn(model rolled so that n = 0 sits at index 0)[k]
    rng = np.random.default_rng(5)
    for N in (8, 9):
        A = rng.standard_normal((N, N, N)).astype(np.float32)
        F = np.fft.fftn(np.roll(A.astype(np.float64), shift=-(N // 2), axis=(0, 1, 2)))
        ks = rng.integers(0, N, size=(30, 3))
        x = 2 * np.pi * ks / N
        ref = F[ks[:, 0], ks[:, 1], ks[:, 2]]
        for direct in (False, True):
            c = orc.nudft(A, x, direct=direct)
            assert np.abs(c - ref).max() <= 1e-11 * np.abs(F).max()


def test_nudft_factored_equals_direct_equals_numpy(pts):
    rng = np.random.default_rng(6)
    A = rng.standard_normal((7, 7, 7)).astype(np.float32)
    a = orc.nudft(A, pts, direct=False)
    b = orc.nudft(A, pts, direct=True)
    c = orc.nudft_numpy(A, pts)
    scale = np.abs(c).max()
    assert np.abs(a - b).max() <= 1e-12 * scale
    assert np.abs(a - c).max() <= 1e-12 * scale


def test_friedel_and_real_even(pts):
    rng = np.random.default_rng(7)
    A = rng.standard_normal((9, 9, 9)).astype(np.float32)
    c_pos, c_neg = orc.nudft(A, pts), orc.nudft(A, -pts)
    assert np.abs(c_neg - np.conj(c_pos)).max() <= 1e-12 * np.abs(c_pos).max()
    E = (0.5 * (A + A[::-1, ::-1, ::-1])).astype(np.float32)   # odd N: index flip is n -> -n
    c = orc.nudft(E, pts)
    assert np.abs(c.imag).max() <= 1e-12 * np.abs(c.real).max()


def test_linearity(pts):
    rng = np.random.default_rng(8)
    # dyadic coefficients and small-integer voxels: a*A1 + b*A2 is exact in fp32
    A1 = rng.integers(-8, 9, (6, 6, 6)).astype(np.float32)
    A2 = rng.integers(-8, 9, (6, 6, 6)).astype(np.float32)
    a, b = 0.5, -2.0
    lhs = orc.nudft((a * A1 + b * A2).astype(np.float32), pts)
    rhs = a * orc.nudft(A1, pts) + b * orc.nudft(A2, pts)
    assert np.abs(lhs - rhs).max() <= 1e-12 * np.abs(rhs).max()


# ---------------------------------------------------------------- rotation conventions (reading s2)

def _hamilton(p, q):
    pw, px, py, pz = p
    qw, qx, qy, qz = q
    return np.array([pw * qw - px * qx - py * qy - pz * qz,
                     pw * qx + px * qw + py * qz - pz * qy,
                     pw * qy - px * qz + py * qw + pz * qx,
                     pw * qz + px * qy - py * qx + pz * qw])


def test_rotation_identity_and_sign():
    assert np.allclose(orc.rotation_matrix([1, 0, 0, 0]), np.eye(3), atol=0)
    q = random_quaternions(5, seed=21)
    for k in range(5):
        assert np.array_equal(orc.rotation_matrix(q[k]), orc.rotation_matrix(-q[k]))
        R = orc.rotation_matrix(q[k])
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-14) and np.isclose(np.linalg.det(R), 1.0, atol=1e-14)
        assert np.allclose(R, orc.rotation_matrix_numpy(q[k]), atol=1e-15)


def test_rotation_is_active_hamilton():
    # +90 degrees about z: (1,0,0) -> (0,1,0)  (passive or JPL conventions give (0,-1,0))
    h = np.sqrt(0.5)
    R = orc.rotation_matrix(np.array([h, 0, 0, h], np.float32))
    assert np.allclose(R @ np.array([1.0, 0, 0]), [0, 1.0, 0], atol=1e-7)
    # +90 about x: (0,1,0) -> (0,0,1)
    R = orc.rotation_matrix(np.array([h, h, 0, 0], np.float32))
    assert np.allclose(R @ np.array([0, 1.0, 0]), [0, 0, 1.0], atol=1e-7)
    # not normalised input is normalised first
    assert np.allclose(orc.rotation_matrix(np.array([2.0, 0, 0, 2.0], np.float32)),
                       orc.rotation_matrix(np.array([h, 0, 0, h], np.float32)), atol=1e-7)


def test_rotation_composition():
    q = random_quaternions(6, seed=22).astype(np.float64)
    for a, b in ((0, 1), (2, 3), (4, 5)):
        prod = _hamilton(q[a], q[b])
        lhs = orc.rotation_matrix(prod.astype(np.float32))
        rhs = orc.rotation_matrix(q[a].astype(np.float32)) @ orc.rotation_matrix(q[b].astype(np.float32))
        assert np.allclose(lhs, rhs, atol=5e-7)   # fp32 rounding of the product quaternion


def test_slice_identity_quaternion_is_direct_evaluation_and_x_is_R_q():
    rng = np.random.default_rng(9)
    A = rng.standard_normal((7, 7, 7)).astype(np.float32)
    pix = rng.uniform(-1.5, 1.5, size=(12, 3)).astype(np.float32)
    ident = np.array([[1, 0, 0, 0]], np.float32)
    c = orc.slice_points(A, ident, pix)
    assert np.abs(c[0] - orc.nudft(A, pix.astype(np.float64))).max() <= 1e-12 * np.abs(c).max()
    # a general quaternion: the slice is the NUDFT at R q (not R^T q) -- checked with the numpy R
    qs = random_quaternions(3, seed=23)
    c = orc.slice_points(A, qs, pix)
    for m in range(3):
        x = pix.astype(np.float64) @ orc.rotation_matrix_numpy(qs[m]).T
        assert np.abs(c[m] - orc.nudft_numpy(A, x)).max() <= 1e-11 * np.abs(c).max()
        xT = pix.astype(np.float64) @ orc.rotation_matrix_numpy(qs[m])
        assert np.abs(c[m] - orc.nudft_numpy(A, xT)).max() > 1e-3 * np.abs(c).max()
    # selected pairs == the same entries of the full set
    sm = np.array([2, 0, 1, 2]); sj = np.array([5, 11, 0, 5])
    assert np.array_equal(orc.slice_points(A, qs, pix, sm, sj), c[sm, sj])


def test_rotation_invariance_of_isotropic_model():
    N, s = 25, 2.0
    A = _gauss_blob(N, np.zeros(3), s).astype(np.float32)
    pix = make_detector(1, 8)
    qs = random_quaternions(6, seed=24)
    c = orc.slice_points(A, qs, pix)
    # closed form depends on |x| only up to the periodic images (|x| <= 0.9 pi, s = 2: images 1e-6)
    assert np.abs(c - c[0:1]).max() <= 1e-5 * np.abs(c).max()
    ref = _gauss_blob_ft(pix.astype(np.float64), np.zeros(3), s)
    assert np.abs(c[0] - ref).max() <= 1e-5 * np.abs(ref).max()


def test_tiny_model_slices_are_real_and_friedel_symmetric():
    cfg = CONFIGS["tiny"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    assert A.dtype == np.float32 and A.shape == (21, 21, 21) and A[10, 10, 10] == 1.0
    assert np.array_equal(A, A[::-1, ::-1, ::-1])
    pix = make_detector(1, 8)
    both = np.concatenate([pix, -pix]).astype(np.float32)
    c = orc.slice_points(A, random_quaternions(2, seed=25), both)
    assert np.abs(c.imag).max() <= 1e-12 * np.abs(c).max()
    assert np.abs(c[:, :64] - c[:, 64:]).max() <= 1e-12 * np.abs(c).max()
    # C restatement vs numpy restatement on the real model
    cn = orc.slices_numpy(A, random_quaternions(2, seed=25), both[:10])
    assert np.abs(c[:, :10] - cn).max() <= 1e-12 * np.abs(c).max()


# ---------------------------------------------------------------- distances and argmin

def test_distances_equal_scipy_cdist_and_expanded_form():
    rng = np.random.default_rng(10)
    I = rng.poisson(0.3, (7, 50)).astype(np.float32)
    S = rng.random((9, 50)).astype(np.float32)
    d = orc.distances(I, S)
    ref = cdist(I.astype(np.float64), S.astype(np.float64), "sqeuclidean")
    assert np.abs(d - ref).max() <= 1e-12 * ref.max()
    I64, S64 = I.astype(np.float64), S.astype(np.float64)
    expanded = (I64 ** 2).sum(1)[:, None] + (S64 ** 2).sum(1)[None, :] - 2 * I64 @ S64.T
    assert np.abs(d - expanded).max() <= 1e-12 * ref.max()
    # fp64 slices entry point gives the same numbers
    assert np.array_equal(orc.distances(I, S.astype(np.float64)), d)
    # d(aI, aS) = a^2 d for a power of two (exact in fp32)
    assert np.allclose(orc.distances(4 * I, 4 * S), 16 * d, rtol=1e-14)


def test_distances_mask_drops_pixels():
    rng = np.random.default_rng(12)
    I = rng.poisson(1.0, (4, 40)).astype(np.float32)
    S = rng.random((5, 40)).astype(np.float32)
    mask = (rng.random(40) > 0.3).astype(np.uint8)
    keep = mask.astype(bool)
    ref = cdist(I[:, keep].astype(np.float64), S[:, keep].astype(np.float64), "sqeuclidean")
    assert np.abs(orc.distances(I, S, mask) - ref).max() <= 1e-12 * ref.max()
    assert np.array_equal(orc.distances(I, S, np.ones(40, np.uint8)), orc.distances(I, S))


def test_argmin_planted_permuted_tied():
    rng = np.random.default_rng(13)
    S = rng.random((11, 30)).astype(np.float32)
    planted = np.array([3, 0, 10, 7])
    I = S[planted].copy()
    bi, bd, sd, d = orc.match(I, S)
    assert np.array_equal(bi, planted) and np.all(bd == 0.0) and np.all(sd > 0)
    # permuting the reference set permutes the answer
    perm = rng.permutation(11)
    bi2, _, _, _ = orc.match(I, S[perm])
    assert np.array_equal(perm[bi2], planted)
    # exact tie -> lowest index; runner-up equals the best
    S2 = np.concatenate([S, S[3:4]])        # slice 11 duplicates slice 3
    bi3, bd3, sd3, _ = orc.match(I[:1], S2)
    assert bi3[0] == 3 and bd3[0] == sd3[0] == 0.0
    S3 = np.concatenate([S[3:4], S])        # now index 0 and 4 tie
    assert orc.match(I[:1], S3)[0][0] == 0
    # brute force in numpy agrees, including the runner-up
    I4 = rng.poisson(0.5, (6, 30)).astype(np.float32)
    bi4, bd4, sd4, d4 = orc.match(I4, S)
    nb, nd = orc.match_numpy(I4, S)
    assert np.array_equal(bi4, nb) and np.allclose(d4, nd, rtol=1e-13)
    assert np.allclose(sd4, np.sort(nd, axis=1)[:, 1], rtol=1e-13)
    # M == 1: no runner-up
    assert np.isinf(orc.match(I4, S[:1])[2]).all()


def test_end_to_end_tiny_planted_orientation():
    """Noise-free image built from reference slice m must match m with d = 0."""
    cfg = CONFIGS["tiny"]
    A = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(1, 8)
    refs = random_quaternions(10, seed=2)
    S = orc.intensity_slices(A, refs, pix, alpha=3.0)
    I = S[[4, 9]].astype(np.float32)
    bi, bd, _, _ = orc.match(I, I.dtype.type(1) * S.astype(np.float32))
    assert list(bi) == [4, 9] and np.all(bd == 0)
