"""Python face of the ORACLE (test infrastructure -- see the header of spf_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from paper_2109_05339_b200/ and the CUDA
path imports nothing from here.

Two layers:
  * ctypes wrappers around liboracle.so (spf_oracle.c, fp64, OpenMP over independent
    points / images) -- what the parity tests and the timed CPU baseline call;
  * a NumPy restatement of the same definitions (`*_numpy`), pure array expressions of
    the formulas, used on Tiny to cross-check the C code.

Definitions (readings in DESIGN.md):
  c_{m,j}  = sum_n A[n] exp(-i n . R(quat_m) q_j),   n = index - floor(N/2)
  S_{m,j}  = alpha * Re c_{m,j}
  d_{i,m}  = sum_{j unmasked} (I_{ij} - S_{mj})^2
  best_i   = argmin_m d_{i,m}  (lowest m on exact ties)
"""
import ctypes as C

import numpy as np

from .build import build_oracle

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build_oracle())
        i64, dbl, flt = C.c_int64, C.c_double, C.c_float
        P = C.POINTER
        lib.oracle_num_threads.restype = C.c_int
        lib.oracle_rotation_matrix.argtypes = [P(flt), P(dbl)]
        lib.oracle_nudft_direct.argtypes = [P(flt), C.c_int, P(dbl), i64, P(dbl)]
        lib.oracle_nudft.argtypes = [P(flt), C.c_int, P(dbl), i64, P(dbl)]
        lib.oracle_slice.argtypes = [P(flt), C.c_int, P(flt), i64, P(flt), i64, P(i64), P(i64), i64, C.c_int, P(dbl)]
        lib.oracle_distances.argtypes = [P(flt), i64, P(flt), i64, i64, P(C.c_uint8), P(dbl)]
        lib.oracle_distances_f64.argtypes = [P(flt), i64, P(dbl), i64, i64, P(C.c_uint8), P(dbl)]
        lib.oracle_argmin.argtypes = [P(dbl), i64, i64, P(i64), P(dbl), P(dbl)]
        for f in (lib.oracle_rotation_matrix, lib.oracle_nudft_direct, lib.oracle_nudft, lib.oracle_slice,
                  lib.oracle_distances, lib.oracle_distances_f64, lib.oracle_argmin):
            f.restype = None
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def _f32(a):
    a = np.ascontiguousarray(a)
    if a.dtype != np.float32:
        raise TypeError("the oracle takes the same fp32 arrays the GPU gets; got %s" % a.dtype)
    return a


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def rotation_matrix(quat) -> np.ndarray:
    """3x3 fp64 active Hamilton rotation matrix of an fp32 quaternion (w,x,y,z) (reading s2)."""
    q = _f32(np.asarray(quat, dtype=np.float32).reshape(4))
    R = np.empty(9, np.float64)
    _load().oracle_rotation_matrix(_p(q, C.c_float), _p(R, C.c_double))
    return R.reshape(3, 3)


def nudft(model, x, direct: bool = False) -> np.ndarray:
    """c(x) = sum_n A[n] exp(-i n.x) at fp64 points x [npts,3]; returns complex128 [npts]."""
    model = _f32(model)
    N = model.shape[0]
    assert model.shape == (N, N, N)
    x = np.ascontiguousarray(x, dtype=np.float64).reshape(-1, 3)
    out = np.empty((x.shape[0], 2), np.float64)
    fn = _load().oracle_nudft_direct if direct else _load().oracle_nudft
    fn(_p(model, C.c_float), N, _p(x, C.c_double), x.shape[0], _p(out, C.c_double))
    return out[:, 0] + 1j * out[:, 1]


def slice_points(model, quats, pix_q, sel_m=None, sel_j=None, direct: bool = False) -> np.ndarray:
    """Complex slices c_{m,j}.  With sel_m/sel_j: complex128 [nsel]; without: [M,P] (all pairs)."""
    model, quats, pix_q = _f32(model), _f32(quats).reshape(-1, 4), _f32(pix_q).reshape(-1, 3)
    N, M, P = model.shape[0], quats.shape[0], pix_q.shape[0]
    if sel_m is None:
        nsel, sm, sj = M * P, None, None
    else:
        sm = np.ascontiguousarray(sel_m, dtype=np.int64)
        sj = np.ascontiguousarray(sel_j, dtype=np.int64)
        assert sm.shape == sj.shape and sm.ndim == 1
        assert sm.min(initial=0) >= 0 and sm.max(initial=0) < M and sj.min(initial=0) >= 0 and sj.max(initial=0) < P
        nsel = sm.shape[0]
    out = np.empty((nsel, 2), np.float64)
    _load().oracle_slice(_p(model, C.c_float), N, _p(quats, C.c_float), M, _p(pix_q, C.c_float), P,
                         _p(sm, C.c_int64), _p(sj, C.c_int64), nsel, int(direct), _p(out, C.c_double))
    c = out[:, 0] + 1j * out[:, 1]
    return c if sel_m is not None else c.reshape(M, P)


def intensity_slices(model, quats, pix_q, alpha: float = 1.0) -> np.ndarray:
    """S_{m,j} = alpha * Re c_{m,j}, fp64 [M,P] (reading s3: a model image is Re c)."""
    return float(alpha) * slice_points(model, quats, pix_q).real


def distances(images, slices, mask=None) -> np.ndarray:
    """d[i,m] = sum_{j unmasked} (I_ij - S_mj)^2 in fp64; slices fp32 (GPU's input) or fp64 (oracle's own)."""
    images = _f32(images)
    n_img, P = images.shape
    slices = np.ascontiguousarray(slices)
    M = slices.shape[0]
    assert slices.shape == (M, P)
    mk = None
    if mask is not None:
        mk = np.ascontiguousarray(mask, dtype=np.uint8)
        assert mk.shape == (P,)
    d = np.empty((n_img, M), np.float64)
    if slices.dtype == np.float32:
        _load().oracle_distances(_p(images, C.c_float), n_img, _p(slices, C.c_float), M, P, _p(mk, C.c_uint8), _p(d, C.c_double))
    elif slices.dtype == np.float64:
        _load().oracle_distances_f64(_p(images, C.c_float), n_img, _p(slices, C.c_double), M, P, _p(mk, C.c_uint8), _p(d, C.c_double))
    else:
        raise TypeError(slices.dtype)
    return d


def argmin(dist):
    """(best_idx int64, best_dist, runner_up_dist) per row; lowest index on exact ties (reading s9)."""
    dist = np.ascontiguousarray(dist, dtype=np.float64)
    n_img, M = dist.shape
    bi = np.empty(n_img, np.int64)
    bd = np.empty(n_img, np.float64)
    sd = np.empty(n_img, np.float64)
    _load().oracle_argmin(_p(dist, C.c_double), n_img, M, _p(bi, C.c_int64), _p(bd, C.c_double), _p(sd, C.c_double))
    return bi, bd, sd


def match(images, slices, mask=None):
    """Brute-force orientation matching: distances then argmin.  Returns (idx, d_min, d_second, dist)."""
    d = distances(images, slices, mask)
    bi, bd, sd = argmin(d)
    return bi, bd, sd, d


# --------------------------------------------------------------------------------------
# NumPy restatement (pure array expressions of the same definitions; Tiny sizes only)
# --------------------------------------------------------------------------------------

def rotation_matrix_numpy(quat) -> np.ndarray:
    w, x, y, z = (np.asarray(quat, dtype=np.float64) / np.linalg.norm(np.asarray(quat, dtype=np.float64)))
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def nudft_numpy(model, x) -> np.ndarray:
    """sum over all voxels of A[n] exp(-i n.x), one complex exponential per (point, voxel)."""
    A = np.asarray(model, dtype=np.float64)
    N = A.shape[0]
    n = np.arange(N) - N // 2
    n1, n2, n3 = np.meshgrid(n, n, n, indexing="ij")
    nvec = np.stack([n1.ravel(), n2.ravel(), n3.ravel()], axis=1).astype(np.float64)  # [N^3, 3]
    x = np.asarray(x, dtype=np.float64).reshape(-1, 3)
    out = np.empty(x.shape[0], np.complex128)
    a = A.ravel()
    for p in range(x.shape[0]):
        out[p] = np.sum(a * np.exp(-1j * (nvec @ x[p])))
    return out


def slices_numpy(model, quats, pix_q) -> np.ndarray:
    quats = np.asarray(quats, dtype=np.float32).reshape(-1, 4)
    q = np.asarray(pix_q, dtype=np.float32).reshape(-1, 3).astype(np.float64)
    out = np.empty((quats.shape[0], q.shape[0]), np.complex128)
    for m in range(quats.shape[0]):
        R = rotation_matrix_numpy(quats[m])
        out[m] = nudft_numpy(model, q @ R.T)  # x_j = R q_j
    return out


def match_numpy(images, slices, mask=None):
    I = np.asarray(images, dtype=np.float64)
    S = np.asarray(slices, dtype=np.float64)
    if mask is not None:
        keep = np.asarray(mask).astype(bool)
        I, S = I[:, keep], S[:, keep]
    d = ((I[:, None, :] - S[None, :, :]) ** 2).sum(axis=2)
    return np.argmin(d, axis=1), d  # np.argmin returns the first (lowest) index on ties
