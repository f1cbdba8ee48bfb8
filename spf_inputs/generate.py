"""Seeded input generators (see package docstring: no method arithmetic lives here).

They stand in for the paper's skopi-simulated PDB-3IYF dataset, which is
not available; shapes follow PAPER.md:124,132 and BASELINE.json:configs.  All NumPy
randomness is numpy.random.Generator(PCG64(seed)); seeds: model 0, mask 1, reference
quaternions 2, truth quaternions 3, Poisson 4, surrogate slices 5, sampling 6.
"""
from dataclasses import dataclass
from typing import Optional

import numpy as np

SEED_MODEL, SEED_MASK, SEED_REF, SEED_TRUTH, SEED_POISSON, SEED_SURROGATE, SEED_SAMPLE = 0, 1, 2, 3, 4, 5, 6


@dataclass(frozen=True)
class Config:
    """One row of BASELINE.json:configs."""
    name: str
    N: int            # model edge
    n_atoms: int
    atom_radius: float
    panels: int       # 1 or 4 (2x2)
    panel_edge: int   # pixels per panel edge
    M: int            # reference orientations
    n_img: int
    photons: float    # mean photons per image
    eps: float
    masked_frac: float = 0.0

    @property
    def P(self) -> int:
        return self.panels * self.panel_edge * self.panel_edge


CONFIGS = {
    "tiny": Config("tiny", 21, 12, 5.0, 1, 32, 64, 16, 100.0, 1e-6),
    "small": Config("small", 81, 200, 25.0, 4, 64, 1024, 1024, 1e4, 1e-6),
    "paper_scale": Config("paper_scale", 151, 2000, 50.0, 4, 128, 10_000, 10_000, 1e4, 1e-6, 0.05),
    "matching_heavy": Config("matching_heavy", 151, 2000, 50.0, 4, 128, 100_000, 20_000, 1e4, 1e-6, 0.05),
    "slicing_heavy": Config("slicing_heavy", 201, 5000, 70.0, 4, 128, 20_000, 2_000, 1e4, 1e-9),
    # the paper's own per-node workload: 128 x 128-pixel images, 1,000 images
    # against 1,200,000 model orientations.  The model size is not stated; the Paper-scale model is reused.  The slice
    # array would be 79 GB, so this configuration runs through spf_slice_match (slices exist one chunk at a time).
    "paper_shaped": Config("paper_shaped", 151, 2000, 50.0, 1, 128, 1_200_000, 1_000, 1e4, 1e-6, 0.05),
}


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def make_atoms(n_atoms: int, radius: float, seed: int = SEED_MODEL) -> np.ndarray:
    """n_atoms positions uniform in a ball of `radius` voxels (r = R u^(1/3), isotropic direction)."""
    rng = _rng(seed)
    r = radius * rng.random(n_atoms) ** (1.0 / 3.0)
    d = rng.standard_normal((n_atoms, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    return r[:, None] * d


def make_density(N: int, atoms: np.ndarray, sigma: float = 1.0) -> np.ndarray:
    """rho[n] = sum_a exp(-|n - r_a|^2 / 2 sigma^2) on the N^3 grid, n = index - floor(N/2), fp64."""
    n = np.arange(N, dtype=np.float64) - N // 2
    rho = np.zeros((N * N, N), np.float64)
    chunk = 256
    for s in range(0, atoms.shape[0], chunk):
        a = atoms[s:s + chunk]
        g = [np.exp(-((n[None, :] - a[:, d:d + 1]) ** 2) / (2.0 * sigma * sigma)) for d in range(3)]
        gxy = (g[0][:, :, None] * g[1][:, None, :]).reshape(a.shape[0], N * N)
        rho += gxy.T @ g[2]
    return rho.reshape(N, N, N)


def make_model(N: int, n_atoms: int, radius: float, seed: int = SEED_MODEL, sigma: float = 1.0) -> np.ndarray:
    """The 3-D model the path slices: autocorrelation of a Gaussian-atom density.

    Linear (zero-padded FFT, fp64) autocorrelation of rho, cropped to the centred N^3 grid,
    symmetrised A <- (A[n] + A[-n]) / 2 where both exist, scaled to A[0] = 1, cast to fp32.
    The autocorrelation is wider than the grid in every config; the model is *defined* as
    what is on the grid.
    """
    import scipy.fft as sfft
    rho = make_density(N, make_atoms(n_atoms, radius, seed), sigma)
    F = sfft.rfftn(rho, s=(2 * N,) * 3, workers=-1)
    ac = sfft.irfftn(F.real ** 2 + F.imag ** 2, s=(2 * N,) * 3, workers=-1)
    del F, rho
    c = N // 2
    lag = (np.arange(N) - c) % (2 * N)
    A = ac[np.ix_(lag, lag, lag)]
    del ac
    # pair n with -n: index i <-> 2c - i, available for i in [lo, N) with lo = 0 (odd N) or 1 (even N)
    lo = 0 if N % 2 else 1
    sub = A[lo:, lo:, lo:]
    sub[...] = 0.5 * (sub + sub[::-1, ::-1, ::-1])
    A = A / A[c, c, c]
    return np.ascontiguousarray(A, dtype=np.float32)


def make_detector(panels: int, panel_edge: int, gap: int = 4, distance_ratio: float = 1.0,
                  q_frac_nyquist: float = 0.9) -> np.ndarray:
    """Pixel q-vectors in NUFFT units (radians per voxel), [P,3] fp32 (readings s4, s5).

    Flat detector normal to z at distance D = distance_ratio * total width; pixel centres on a
    unit lattice; 1 panel, or 2x2 panels separated by a `gap`-pixel cross.  Ewald sphere with
    k = 1:  q = (u, v, D) / |(u, v, D)| - z_hat,  then scaled so max |q| = q_frac_nyquist * pi.
    Pixel order: panel-major, row-major inside a panel.
    """
    e = panel_edge
    if panels == 1:
        width = float(e)
        origins = [(-e / 2.0, -e / 2.0)]
    elif panels == 4:
        width = 2.0 * e + gap
        origins = [(-width / 2.0, -width / 2.0), (-width / 2.0, gap / 2.0),
                   (gap / 2.0, -width / 2.0), (gap / 2.0, gap / 2.0)]
    else:
        raise ValueError("panels must be 1 or 4")
    D = distance_ratio * width
    uv = []
    ax = np.arange(e, dtype=np.float64) + 0.5
    for (u0, v0) in origins:
        uu, vv = np.meshgrid(u0 + ax, v0 + ax, indexing="ij")
        uv.append(np.stack([uu.ravel(), vv.ravel()], axis=1))
    uv = np.concatenate(uv, axis=0)
    k_out = np.concatenate([uv, np.full((uv.shape[0], 1), D)], axis=1)
    k_out /= np.linalg.norm(k_out, axis=1, keepdims=True)
    q = k_out - np.array([0.0, 0.0, 1.0])
    q *= q_frac_nyquist * np.pi / np.linalg.norm(q, axis=1).max()
    return np.ascontiguousarray(q, dtype=np.float32)


def detector_uv(panels: int, panel_edge: int, gap: int = 4) -> np.ndarray:
    """Pixel-centre lattice coordinates (u, v) in pixels, same order as make_detector."""
    e = panel_edge
    if panels == 1:
        origins = [(-e / 2.0, -e / 2.0)]
    else:
        width = 2.0 * e + gap
        origins = [(-width / 2.0, -width / 2.0), (-width / 2.0, gap / 2.0),
                   (gap / 2.0, -width / 2.0), (gap / 2.0, gap / 2.0)]
    ax = np.arange(e, dtype=np.float64) + 0.5
    uv = []
    for (u0, v0) in origins:
        uu, vv = np.meshgrid(u0 + ax, v0 + ax, indexing="ij")
        uv.append(np.stack([uu.ravel(), vv.ravel()], axis=1))
    return np.concatenate(uv, axis=0)


def make_mask(panels: int, panel_edge: int, masked_frac: float, seed: int = SEED_MASK, gap: int = 4,
              beamstop_radius: float = 8.0) -> Optional[np.ndarray]:
    """[P] uint8, 1 = use.  Beam-stop disc at the centre plus random dead pixels up to exactly
    round(masked_frac * P) masked pixels (reading s8).  None when masked_frac == 0."""
    if masked_frac <= 0.0:
        return None
    uv = detector_uv(panels, panel_edge, gap)
    P = uv.shape[0]
    mask = np.ones(P, np.uint8)
    mask[np.hypot(uv[:, 0], uv[:, 1]) < beamstop_radius] = 0
    target = int(round(masked_frac * P))
    n_dead = target - int((mask == 0).sum())
    if n_dead < 0:
        raise ValueError("beam stop alone exceeds masked_frac")
    alive = np.flatnonzero(mask)
    mask[_rng(seed).choice(alive, size=n_dead, replace=False)] = 0
    return mask


def random_quaternions(n: int, seed: int) -> np.ndarray:
    """n uniform random orientations: normalised 4-D Gaussians, sign fixed to w >= 0, fp32 (w,x,y,z)."""
    q = _rng(seed).standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    q[q[:, 0] < 0] *= -1.0
    return np.ascontiguousarray(q, dtype=np.float32)


def planted_truth_quaternions(n_img: int, ref_quats: np.ndarray, planted_frac: float = 0.1,
                              seed: int = SEED_TRUTH):
    """Truth orientations of the images.  The first round(planted_frac*n_img) are copies of random
    reference orientations (so a known answer exists with high probability -- a sanity statistic,
    not a correctness reference); the rest are fresh uniform random orientations.
    Returns (quats [n_img,4] fp32, planted_ref_index [n_img] int64, -1 where not planted)."""
    rng = _rng(seed)
    q = rng.standard_normal((n_img, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    q[q[:, 0] < 0] *= -1.0
    q = q.astype(np.float32)
    n_pl = int(round(planted_frac * n_img))
    idx = np.full(n_img, -1, np.int64)
    if n_pl:
        pick = rng.integers(0, ref_quats.shape[0], size=n_pl)
        q[:n_pl] = ref_quats[pick]
        idx[:n_pl] = pick
    return np.ascontiguousarray(q), idx


def photon_scale(ref_slices_re, mask, photons: float) -> float:
    """alpha = photons / mean_m sum_{j unmasked} Re c_mj over the reference slices (reading s6).
    Accepts a NumPy array or a torch tensor [M,P]."""
    keep = None if mask is None else np.flatnonzero(np.asarray(mask))
    if hasattr(ref_slices_re, "detach"):  # torch tensor (any device)
        import torch
        s = ref_slices_re if keep is None else ref_slices_re[:, torch.as_tensor(keep, device=ref_slices_re.device)]
        tot = float(s.double().sum(dim=1).mean().item())
    else:
        s = np.asarray(ref_slices_re, dtype=np.float64)
        s = s if keep is None else s[:, keep]
        tot = float(s.sum(axis=1).mean())
    return float(photons) / tot


def poisson_images(lam, seed: int = SEED_POISSON):
    """I_ij ~ Poisson(max(lam_ij, 0)) kept as raw counts in fp32.  NumPy in -> NumPy out (PCG64);
    torch tensor in -> torch tensor out on the same device (torch.Generator seeded with `seed`)."""
    if hasattr(lam, "detach"):
        import torch
        g = torch.Generator(device=lam.device)
        g.manual_seed(seed)
        return torch.poisson(lam.clamp_min(0).float(), generator=g)
    lam = np.maximum(np.asarray(lam, dtype=np.float64), 0.0)
    return _rng(seed).poisson(lam).astype(np.float32)


def surrogate_slices(M: int, pix_q: np.ndarray, seed: int = SEED_SURROGATE, device=None):
    """Stand-in model images for MATCH-ONLY tests at sizes where no CPU code can slice: a smooth
    radial fall-off 1 / (1 + (|q| / q0)^4) times unit-mean exponential speckle (the intensity
    statistics of a diffraction pattern), fp32 [M,P].  Not a slice of anything; spf_match takes
    images and slices as independent inputs, so its arithmetic is exercised all the same.
    device=None -> NumPy (PCG64); otherwise a torch tensor generated on `device`."""
    qn = np.linalg.norm(np.asarray(pix_q, dtype=np.float64), axis=1)
    base = 1.0 / (1.0 + (qn / (0.15 * np.pi)) ** 4)
    P = base.shape[0]
    if device is None:
        u = _rng(seed).random((M, P))
        return (base[None, :] * -np.log1p(-u)).astype(np.float32)
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    out = torch.empty((M, P), dtype=torch.float32, device=device)
    b = torch.as_tensor(base, dtype=torch.float32, device=device)
    step = max(1, (1 << 26) // P)
    for s in range(0, M, step):
        u = torch.rand((min(step, M - s), P), generator=g, device=device, dtype=torch.float32)
        out[s:s + u.shape[0]] = b[None, :] * -torch.log1p(-u)
    return out


def sample_pairs(M: int, P: int, n: int, seed: int = SEED_SAMPLE):
    """n random (orientation, pixel) index pairs for sampled oracle checks."""
    rng = _rng(seed)
    return rng.integers(0, M, size=n).astype(np.int64), rng.integers(0, P, size=n).astype(np.int64)
