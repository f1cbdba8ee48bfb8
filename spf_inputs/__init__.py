"""Seeded synthetic inputs shared by the oracle tests and the CUDA tests / bench.

This package holds NONE of the method's arithmetic (no NUDFT, no NUFFT, no distances):
it only builds the arrays that are *inputs* to slicing and matching -- the model volume,
detector q-vectors, mask, quaternions, Poisson counts -- with the shapes and statistics of
BASELINE.json:configs.  Anything that needs slices (the Poisson means) receives them as
an argument from the caller.  Recipe: DESIGN.md "Synthetic inputs".
"""
from .generate import (CONFIGS, Config, make_atoms, make_density, make_model, make_detector, make_mask,
                       random_quaternions, planted_truth_quaternions, photon_scale, poisson_images,
                       surrogate_slices, sample_pairs)

__all__ = ["CONFIGS", "Config", "make_atoms", "make_density", "make_model", "make_detector", "make_mask",
           "random_quaternions", "planted_truth_quaternions", "photon_scale", "poisson_images",
           "surrogate_slices", "sample_pairs"]
