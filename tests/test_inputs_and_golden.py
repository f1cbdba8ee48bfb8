"""Input-generator sanity and the oracle regression snapshot (-m "not gpu")."""
import json
import os
import sys

import numpy as np

from spf_inputs import (CONFIGS, make_model, make_detector, make_mask, random_quaternions,
                        planted_truth_quaternions, poisson_images, surrogate_slices, sample_pairs)

HERE = os.path.dirname(os.path.abspath(__file__))


def test_config_table_matches_baseline_json():
    with open(os.path.join(os.path.dirname(HERE), "BASELINE.json")) as f:
        text = " ".join(json.load(f)["configs"])
    base = [c for name, c in CONFIGS.items() if name != "paper_shaped"]       # the five rows of BASELINE.json:configs
    assert [c.P for c in base] == [1024, 16384, 65536, 65536, 65536]
    assert [c.N for c in base] == [21, 81, 151, 151, 201]
    assert [c.M for c in base] == [64, 1024, 10_000, 100_000, 20_000]
    assert [c.n_img for c in base] == [16, 1024, 10_000, 20_000, 2_000]
    ps = CONFIGS["paper_shaped"]
    assert (ps.P, ps.M, ps.n_img) == (128 * 128, 1_200_000, 1_000)
    for token in ("21^3", "81^3", "151^3", "201^3", "65,536", "100,000 reference", "eps 1e-9"):
        assert token in text


def test_detector_geometry():
    for panels, edge in ((1, 32), (4, 64)):
        q = make_detector(panels, edge)
        assert q.dtype == np.float32 and q.shape == (panels * edge * edge, 3)
        r = np.linalg.norm(q.astype(np.float64), axis=1)
        assert abs(r.max() - 0.9 * np.pi) < 1e-6
        # Ewald sphere: |q + k z|^2 = k^2 with k = 0.9 pi / max|q_unscaled|; q_z <= 0
        assert (q[:, 2] <= 0).all()
        k = -(r ** 2) / (2 * q[:, 2].astype(np.float64))
        assert np.allclose(k, k[0], rtol=1e-5)
        # inversion-symmetric lattice: for every pixel (u,v) there is (-u,-v)
        s = {(round(float(a), 4), round(float(b), 4)) for a, b in q[:, :2]}
        assert all((-a, -b) in s for a, b in s)


def test_mask_counts():
    m = make_mask(4, 128, 0.05)
    assert m.dtype == np.uint8 and m.shape == (65536,) and int((m == 0).sum()) == 3277
    assert make_mask(4, 64, 0.0) is None
    assert np.array_equal(m, make_mask(4, 128, 0.05))


def test_quaternions_and_poisson_are_seeded():
    q = random_quaternions(100, seed=2)
    assert q.dtype == np.float32 and np.allclose(np.linalg.norm(q, axis=1), 1, atol=1e-6) and (q[:, 0] >= 0).all()
    assert np.array_equal(q, random_quaternions(100, seed=2))
    t, idx = planted_truth_quaternions(50, q)
    assert (idx[:5] >= 0).all() and (idx[5:] == -1).all() and np.array_equal(t[:5], q[idx[:5]])
    lam = np.full((3, 1000), 0.15)
    I = poisson_images(lam)
    assert I.dtype == np.float32 and np.array_equal(I, poisson_images(lam)) and abs(I.mean() - 0.15) < 0.03
    assert np.array_equal(I, np.round(I)) and (poisson_images(-lam) == 0).all()
    S = surrogate_slices(5, make_detector(1, 16))
    assert S.dtype == np.float32 and S.shape == (5, 256) and (S >= 0).all()
    sm, sj = sample_pairs(7, 9, 20)
    assert sm.max() < 7 and sj.max() < 9


def test_small_model_is_even_real_normalised():
    A = make_model(21, 12, 5.0)
    assert A[10, 10, 10] == 1.0 and np.array_equal(A, A[::-1, ::-1, ::-1]) and A.max() == 1.0
    B = make_model(12, 5, 3.0)   # even N: n <-> -n symmetric on the paired sub-grid
    assert np.array_equal(B[1:, 1:, 1:], B[1:, 1:, 1:][::-1, ::-1, ::-1]) and B[6, 6, 6] == 1.0


def test_oracle_matches_its_regression_snapshot():
    sys.path.insert(0, os.path.join(HERE, "golden"))
    from make_golden import tiny_oracle_run
    with open(os.path.join(HERE, "golden", "tiny_oracle.json")) as f:
        gold = json.load(f)
    now = tiny_oracle_run()
    assert now["sel_m"] == gold["sel_m"] and now["sel_j"] == gold["sel_j"]
    assert now["best_idx"] == gold["best_idx"] and now["image_sums"] == gold["image_sums"]
    for k in ("c_re", "c_im", "best_dist", "second_dist"):
        a, b = np.array(now[k]), np.array(gold[k])
        assert np.abs(a - b).max() <= 1e-9 * max(1.0, np.abs(b).max())
    assert abs(now["alpha"] - gold["alpha"]) <= 1e-12 * gold["alpha"]
