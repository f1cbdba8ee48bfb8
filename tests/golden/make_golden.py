"""Writes tests/golden/tiny_oracle.json.  Calls ONLY oracle/ and spf_inputs/ (never the CUDA path)."""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from spf_inputs import (CONFIGS, make_model, make_detector, random_quaternions, planted_truth_quaternions,  # noqa: E402
                        photon_scale, poisson_images, sample_pairs)


def tiny_oracle_run():
    cfg = CONFIGS["tiny"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    truth, planted = planted_truth_quaternions(cfg.n_img, refs)
    c_ref = orc.slice_points(model, refs, pix)
    alpha = photon_scale(c_ref.real, None, cfg.photons)
    lam = alpha * orc.slice_points(model, truth, pix).real
    images = poisson_images(lam)
    slices32 = (alpha * c_ref.real).astype(np.float32)
    bi, bd, sd, _ = orc.match(images, slices32)
    sm, sj = sample_pairs(cfg.M, cfg.P, 32)
    return dict(alpha=alpha, sel_m=sm.tolist(), sel_j=sj.tolist(),
                c_re=c_ref[sm, sj].real.tolist(), c_im=c_ref[sm, sj].imag.tolist(),
                image_sums=images.sum(axis=1).tolist(), planted=planted.tolist(),
                best_idx=bi.tolist(), best_dist=bd.tolist(), second_dist=sd.tolist())


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_oracle.json")
    with open(out, "w") as f:
        json.dump(tiny_oracle_run(), f, indent=1)
    print("wrote", out)
