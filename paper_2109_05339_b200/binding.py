"""Thin ctypes binding of libspf (include/spf.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used for device memory and
streams.  There is no CPU fallback: if libspf.so is missing or no CUDA device is present the calls
raise.  Names follow the C ABI (spf_prepare_model / spf_slice / spf_match).
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# SPF_DEBUG=1 loads the build with device-side asserts (python -m paper_2109_05339_b200.build under the same variable)
LIB_PATH = os.path.join(_HERE, "libspf_debug.so" if os.environ.get("SPF_DEBUG", "0") == "1" else "libspf.so")

SPF_OUT_COMPLEX = 0
SPF_OUT_INTENSITY = 1

EXPORTS = ["spf_version", "spf_status_string", "spf_plan_kernel_width", "spf_plan_n_fine", "spf_create", "spf_destroy",
           "spf_get_info", "spf_last_error", "spf_set_detector_layout", "spf_prepare_model", "spf_slice", "spf_match",
           "spf_match_workspace_bytes", "spf_match_reference", "spf_orientation_match_host", "spf_debug_deapodisation",
           "spf_debug_fine_grid", "spf_set_option", "spf_launch_count", "spf_last_kernel_ms", "spf_last_match_products",
           "spf_check_fault", "spf_selftest", "spf_slice_match", "spf_slice_match_workspace_bytes", "spf_get_option", "spf_microbench"]


class SpfParams(C.Structure):
    _fields_ = [("n", C.c_int32), ("eps", C.c_double), ("upsampfac", C.c_double), ("n_fine", C.c_int32),
                ("device", C.c_int32)]


class SpfInfo(C.Structure):
    _fields_ = [("n", C.c_int32), ("n_fine", C.c_int32), ("w", C.c_int32), ("beta", C.c_double),
                ("n_padded", C.c_int32), ("grid_is_real", C.c_int32), ("prepared", C.c_int32), ("sm_count", C.c_int32)]


class SpfSelftestReport(C.Structure):
    _fields_ = [("passed", C.c_int32), ("ms_variant", C.c_float), ("ms_reference", C.c_float), ("worst_rel", C.c_double),
                ("detail", C.c_char * 192)]


class SpfError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("libspf status %d: %s" % (status, text))
        self.status = status


_lib = None


def load_library():
    """dlopen libspf.so (fails loudly when it has not been built: python paper_2109_05339_b200/build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libspf.so not built; run `python -m paper_2109_05339_b200.build` (needs nvcc)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, f32, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_float, C.c_size_t
    lib.spf_version.restype = C.c_char_p
    lib.spf_status_string.restype = C.c_char_p
    lib.spf_status_string.argtypes = [C.c_int]
    lib.spf_plan_kernel_width.restype = i32
    lib.spf_plan_kernel_width.argtypes = [C.c_double]
    lib.spf_plan_n_fine.restype = i32
    lib.spf_plan_n_fine.argtypes = [i32, C.c_double]
    lib.spf_create.argtypes = [C.POINTER(vp), C.POINTER(SpfParams)]
    lib.spf_destroy.argtypes = [vp]
    lib.spf_destroy.restype = None
    lib.spf_get_info.argtypes = [vp, C.POINTER(SpfInfo)]
    lib.spf_last_error.argtypes = [vp]
    lib.spf_last_error.restype = C.c_char_p
    lib.spf_set_detector_layout.argtypes = [vp, i32, i32, i32]
    lib.spf_prepare_model.argtypes = [vp, vp, vp]
    lib.spf_slice.argtypes = [vp, vp, i64, vp, i64, i32, f32, vp, vp]
    lib.spf_match.argtypes = [vp, vp, i64, vp, i64, i64, vp, vp, vp, vp, sz, vp]
    lib.spf_match_workspace_bytes.argtypes = [i64, i64, i64]
    lib.spf_match_workspace_bytes.restype = sz
    lib.spf_match_reference.argtypes = [vp, vp, i64, vp, i64, i64, vp, vp, vp, vp, vp]
    lib.spf_orientation_match_host.argtypes = [vp, vp, vp, i64, vp, i64, f32, vp, i64, vp, vp, vp, vp]
    lib.spf_debug_deapodisation.argtypes = [vp, vp]
    lib.spf_debug_fine_grid.argtypes = [vp, vp, vp]
    lib.spf_set_option.argtypes = [vp, C.c_char_p, i64]
    lib.spf_get_option.argtypes = [vp, C.c_char_p, C.POINTER(i64)]
    lib.spf_microbench.argtypes = [vp, C.c_char_p, C.POINTER(C.c_double), vp]
    lib.spf_launch_count.argtypes = [vp]
    lib.spf_launch_count.restype = i64
    lib.spf_last_kernel_ms.argtypes = [vp, i32, C.POINTER(C.c_float)]
    lib.spf_last_match_products.argtypes = [vp, C.POINTER(i32)]
    lib.spf_check_fault.argtypes = [vp, vp]
    lib.spf_selftest.argtypes = [vp, C.c_char_p, C.POINTER(SpfSelftestReport), vp]
    lib.spf_slice_match.argtypes = [vp, vp, i64, vp, i64, f32, vp, i64, vp, i64, vp, vp, vp, sz, vp]
    lib.spf_slice_match_workspace_bytes.argtypes = [i64, i64, i64]
    lib.spf_slice_match_workspace_bytes.restype = sz
    _lib = lib
    return lib


def spf_plan_kernel_width(eps: float) -> int:
    return int(load_library().spf_plan_kernel_width(eps))


def spf_plan_n_fine(n: int, upsampfac: float = 2.0) -> int:
    return int(load_library().spf_plan_n_fine(n, upsampfac))


def spf_match_workspace_bytes(n_img: int, M: int, P: int) -> int:
    return int(load_library().spf_match_workspace_bytes(n_img, M, P))


def _dev(t, dtype, what):
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor" % what)
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be contiguous %s, got %s" % (what, dtype, t.dtype))
    return C.c_void_p(t.data_ptr())


def _stream(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


class SpfContext:
    """Owns one spf_ctx.  Methods carry the C names; tensors in, tensors out."""

    def __init__(self, n: int, eps: float = 1e-6, upsampfac: float = 2.0, n_fine: int = 0, device: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("libspf needs a CUDA device (no CPU fallback)")
        self._lib = load_library()
        self._h = C.c_void_p()
        self.device = torch.device("cuda", device)
        p = SpfParams(n, eps, upsampfac, n_fine, device)
        rc = self._lib.spf_create(C.byref(self._h), C.byref(p))
        if rc != 0:
            raise SpfError(rc, (self._lib.spf_last_error(None) or b"").decode())
        self._ws = None

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.spf_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _check(self, rc):
        if rc != 0:
            raise SpfError(rc, (self._lib.spf_last_error(self._h) or b"").decode())

    @property
    def info(self) -> SpfInfo:
        out = SpfInfo()
        self._check(self._lib.spf_get_info(self._h, C.byref(out)))
        return out

    def spf_set_detector_layout(self, n_panels: int, rows: int, cols: int):
        self._check(self._lib.spf_set_detector_layout(self._h, n_panels, rows, cols))

    def spf_set_option(self, key: str, value: int):
        self._check(self._lib.spf_set_option(self._h, key.encode(), int(value)))

    def spf_get_option(self, key: str) -> int:
        v = C.c_int64()
        self._check(self._lib.spf_get_option(self._h, key.encode(), C.byref(v)))
        return int(v.value)

    def spf_microbench(self, what: str) -> float:
        """GB/s of one device figure (spf.h): "lds32", "lds128", "l2", "hbm_read", "hbm_copy"."""
        v = C.c_double()
        self._check(self._lib.spf_microbench(self._h, what.encode(), C.byref(v), _stream(self.device)))
        return float(v.value)

    def spf_check_fault(self):
        """Synchronise the current stream; raise SpfError(SPF_EFAULT) if a kernel's watchdog gave up."""
        self._check(self._lib.spf_check_fault(self._h, _stream(self.device)))

    def spf_selftest(self, variant: str) -> dict:
        """The library's own in-process check of one variant (spf.h); on success the library switches it on."""
        rep = SpfSelftestReport()
        self._check(self._lib.spf_selftest(self._h, variant.encode(), C.byref(rep), _stream(self.device)))
        return {"passed": bool(rep.passed), "ms_variant": float(rep.ms_variant), "ms_reference": float(rep.ms_reference),
                "worst_rel": float(rep.worst_rel), "detail": rep.detail.decode(errors="replace")}

    def spf_autotune(self, timeout_s: float = 240.0, classic_only: bool = False) -> dict:
        """Switch on the faster kernel variants that pass the library's own device check.  Each variant's check
        (spf_selftest, C) first runs in a CHILD process (selfcheck.py), least machinery first, stopping at the first child
        that dies -- a faulting variant cannot take this process's CUDA context with it; for every variant whose child
        passed, spf_selftest is then called on THIS context, which is what switches it on (the C library keeps the
        fastest verified slicer; tcgen05 supersedes mma.sync, CTA pairs supersede single CTAs).  classic_only=True limits the
        candidates to the classic-CUDA tier (slice_impl 3 / 4, match_impl 2): no tensor map, mbarrier, TMEM or tcgen05.
        The model must be prepared (the slicing checks slice the caller's own model).  Returns {variant: bool} plus
        "slice_impl" / "match_impl" / "match_cta_group" = the options now in force, and "detail" per variant."""
        from .selfcheck import verified_variants, CLASSIC
        report = {}
        ok = dict(verified_variants(self.device.index or 0, timeout_s, report, only=CLASSIC if classic_only else None))
        ok["detail"] = {}
        for v, passed in list(ok.items()):
            if v == "detail":
                continue
            if passed and v.startswith("slice") and not self.info.prepared:
                ok[v] = False
                ok["detail"][v] = "not switched on: the slicing checks slice the caller's model (call spf_prepare_model first)"
            elif passed:
                st = self.spf_selftest(v)
                ok[v] = st["passed"]
                ok["detail"][v] = st["detail"]
            else:
                ok["detail"][v] = "child check: " + str((report.get(v) or {}).get("detail", ""))[:160]
        for k in ("slice_impl", "match_impl", "match_cta_group"):
            ok[k] = self.spf_get_option(k)
        return ok

    def spf_launch_count(self) -> int:
        return int(self._lib.spf_launch_count(self._h))

    def spf_last_kernel_ms(self, which: int) -> float:
        ms = C.c_float()
        self._check(self._lib.spf_last_kernel_ms(self._h, which, C.byref(ms)))
        return float(ms.value)

    def spf_last_match_products(self) -> int:
        n = C.c_int32()
        self._check(self._lib.spf_last_match_products(self._h, C.byref(n)))
        return int(n.value)

    def spf_prepare_model(self, model: torch.Tensor):
        n = self.info.n
        if tuple(model.shape) != (n, n, n):
            raise ValueError("model must be [%d,%d,%d]" % (n, n, n))
        self._check(self._lib.spf_prepare_model(self._h, _dev(model, torch.float32, "model"), _stream(self.device)))

    def spf_slice(self, quats: torch.Tensor, pix_q: torch.Tensor, out_kind: int = SPF_OUT_INTENSITY, scale: float = 1.0,
                  out: torch.Tensor = None) -> torch.Tensor:
        M, P = quats.shape[0], pix_q.shape[0]
        if quats.shape != (M, 4) or pix_q.shape != (P, 3):
            raise ValueError("quats must be [M,4] and pix_q [P,3]")
        dt = torch.complex64 if out_kind == SPF_OUT_COMPLEX else torch.float32
        if out is None:
            out = torch.empty((M, P), dtype=dt, device=self.device)
        elif out.shape != (M, P):
            raise ValueError("out must be [M,P]")
        self._check(self._lib.spf_slice(self._h, _dev(quats, torch.float32, "quats"), M, _dev(pix_q, torch.float32, "pix_q"), P,
                                        out_kind, float(scale), _dev(out, dt, "out"), _stream(self.device)))
        return out

    def spf_match(self, images: torch.Tensor, slices: torch.Tensor, mask: torch.Tensor = None):
        n_img, P = images.shape
        M = slices.shape[0]
        if slices.shape != (M, P):
            raise ValueError("slices must be [M,P] with the images' P")
        need = spf_match_workspace_bytes(n_img, M, P)
        if self._ws is None or self._ws.numel() < need + 1024:
            self._ws = None
            self._ws = torch.empty(need + 1024, dtype=torch.uint8, device=self.device)
        ws_ptr = (self._ws.data_ptr() + 1023) & ~1023
        best_idx = torch.empty(n_img, dtype=torch.int32, device=self.device)
        best_dist = torch.empty(n_img, dtype=torch.float32, device=self.device)
        mk = None if mask is None else _dev(mask, torch.uint8, "mask")
        if mask is not None and mask.shape != (P,):
            raise ValueError("mask must be [P]")
        self._check(self._lib.spf_match(self._h, _dev(images, torch.float32, "images"), n_img, _dev(slices, torch.float32, "slices"),
                                        M, P, mk, _dev(best_idx, torch.int32, "best_idx"), _dev(best_dist, torch.float32, "best_dist"),
                                        C.c_void_p(ws_ptr), need, _stream(self.device)))
        return best_idx, best_dist

    def spf_slice_match(self, quats: torch.Tensor, pix_q: torch.Tensor, images: torch.Tensor, scale: float = 1.0,
                        mask: torch.Tensor = None, chunk_M: int = 1024):
        """Slicing and matching fused at the seam: slices exist only chunk_M orientations at a time (spf.h)."""
        M, P, n_img = quats.shape[0], pix_q.shape[0], images.shape[0]
        if quats.shape != (M, 4) or pix_q.shape != (P, 3) or images.shape != (n_img, P):
            raise ValueError("quats [M,4], pix_q [P,3], images [n_img,P]")
        chunk_M = max(1, min(int(chunk_M), M))
        need = int(self._lib.spf_slice_match_workspace_bytes(n_img, chunk_M, P))
        if self._ws is None or self._ws.numel() < need + 1024:
            self._ws = None
            self._ws = torch.empty(need + 1024, dtype=torch.uint8, device=self.device)
        ws_ptr = (self._ws.data_ptr() + 1023) & ~1023
        best_idx = torch.empty(n_img, dtype=torch.int32, device=self.device)
        best_dist = torch.empty(n_img, dtype=torch.float32, device=self.device)
        mk = None if mask is None else _dev(mask, torch.uint8, "mask")
        self._check(self._lib.spf_slice_match(self._h, _dev(quats, torch.float32, "quats"), M, _dev(pix_q, torch.float32, "pix_q"), P,
                                              float(scale), _dev(images, torch.float32, "images"), n_img, mk, chunk_M,
                                              _dev(best_idx, torch.int32, "best_idx"), _dev(best_dist, torch.float32, "best_dist"),
                                              C.c_void_p(ws_ptr), need, _stream(self.device)))
        return best_idx, best_dist

    def spf_match_reference(self, images: torch.Tensor, slices: torch.Tensor, mask: torch.Tensor = None):
        n_img, P = images.shape
        M = slices.shape[0]
        best_idx = torch.empty(n_img, dtype=torch.int32, device=self.device)
        best_dist = torch.empty(n_img, dtype=torch.float32, device=self.device)
        dist = torch.empty((n_img, M), dtype=torch.float32, device=self.device)
        mk = None if mask is None else _dev(mask, torch.uint8, "mask")
        self._check(self._lib.spf_match_reference(self._h, _dev(images, torch.float32, "images"), n_img,
                                                  _dev(slices, torch.float32, "slices"), M, P, mk,
                                                  _dev(best_idx, torch.int32, "best_idx"), _dev(best_dist, torch.float32, "best_dist"),
                                                  _dev(dist, torch.float32, "dist"), _stream(self.device)))
        return best_idx, best_dist, dist

    def spf_orientation_match_host(self, model: np.ndarray, quats: np.ndarray, pix_q: np.ndarray, images, scale: float = 1.0,
                                   mask: np.ndarray = None, want_slices: bool = False):
        """Host buffers in (NumPy arrays or pinned CPU tensors), host results out."""
        def host(a, dt, what):
            if isinstance(a, torch.Tensor):
                if a.is_cuda or a.dtype != getattr(torch, np.dtype(dt).name) or not a.is_contiguous():
                    raise TypeError("%s must be a contiguous CPU %s tensor" % (what, dt))
                return a, C.c_void_p(a.data_ptr())
            a = np.ascontiguousarray(a, dtype=dt)
            return a, C.c_void_p(a.ctypes.data)
        model, pm = host(model, np.float32, "model")
        quats, pq = host(quats, np.float32, "quats")
        pix_q, pp = host(pix_q, np.float32, "pix_q")
        images, pi = host(images, np.float32, "images")
        M, P, n_img = quats.shape[0], pix_q.shape[0], images.shape[0]
        pmask = None
        if mask is not None:
            mask, pmask = host(mask, np.uint8, "mask")
        best_idx = np.empty(n_img, np.int32)
        best_dist = np.empty(n_img, np.float32)
        slices = np.empty((M, P), np.float32) if want_slices else None
        self._check(self._lib.spf_orientation_match_host(self._h, pm, pq, M, pp, P, float(scale), pi, n_img, pmask,
                                                         C.c_void_p(best_idx.ctypes.data), C.c_void_p(best_dist.ctypes.data),
                                                         C.c_void_p(slices.ctypes.data) if want_slices else None))
        return (best_idx, best_dist, slices) if want_slices else (best_idx, best_dist)

    def spf_debug_deapodisation(self) -> np.ndarray:
        out = np.empty(self.info.n, np.float64)
        self._check(self._lib.spf_debug_deapodisation(self._h, C.c_void_p(out.ctypes.data)))
        return out

    def spf_debug_fine_grid(self) -> torch.Tensor:
        nf = self.info.n_fine
        out = torch.empty((nf, nf, nf), dtype=torch.complex64, device=self.device)
        self._check(self._lib.spf_debug_fine_grid(self._h, C.c_void_p(out.data_ptr()), _stream(self.device)))
        return out
