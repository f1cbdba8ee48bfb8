"""NumPy face of tests/emu/libspf_emu.so: libspf's C ABI with "device" pointers that are host pointers.
TEST INFRASTRUCTURE ONLY (see cuda_emu.h): used by tests/test_emu_kernels.py to execute the kernels' own source
on a box without a GPU.  Nothing in the product imports this."""
import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)
from build_emu import build_emu  # noqa: E402

SPF_OUT_COMPLEX, SPF_OUT_INTENSITY = 0, 1


class SpfParams(C.Structure):
    _fields_ = [("n", C.c_int32), ("eps", C.c_double), ("upsampfac", C.c_double), ("n_fine", C.c_int32), ("device", C.c_int32)]


class SpfInfo(C.Structure):
    _fields_ = [("n", C.c_int32), ("n_fine", C.c_int32), ("w", C.c_int32), ("beta", C.c_double),
                ("n_padded", C.c_int32), ("grid_is_real", C.c_int32), ("prepared", C.c_int32), ("sm_count", C.c_int32)]


class SelftestReport(C.Structure):
    _fields_ = [("passed", C.c_int32), ("ms_variant", C.c_float), ("ms_reference", C.c_float), ("worst_rel", C.c_double),
                ("detail", C.c_char * 192)]


class EmuError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("libspf (emulated) status %d: %s" % (status, text))
        self.status = status


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_emu())
        vp, i32, i64, f32, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_float, C.c_size_t
        L.spf_create.argtypes = [C.POINTER(vp), C.POINTER(SpfParams)]
        L.spf_destroy.argtypes = [vp]; L.spf_destroy.restype = None
        L.spf_get_info.argtypes = [vp, C.POINTER(SpfInfo)]
        L.spf_last_error.argtypes = [vp]; L.spf_last_error.restype = C.c_char_p
        L.spf_set_detector_layout.argtypes = [vp, i32, i32, i32]
        L.spf_set_option.argtypes = [vp, C.c_char_p, i64]
        L.spf_prepare_model.argtypes = [vp, vp, vp]
        L.spf_slice.argtypes = [vp, vp, i64, vp, i64, i32, f32, vp, vp]
        L.spf_match.argtypes = [vp, vp, i64, vp, i64, i64, vp, vp, vp, vp, sz, vp]
        L.spf_match_workspace_bytes.argtypes = [i64, i64, i64]; L.spf_match_workspace_bytes.restype = sz
        L.spf_match_reference.argtypes = [vp, vp, i64, vp, i64, i64, vp, vp, vp, vp, vp]
        L.spf_orientation_match_host.argtypes = [vp, vp, vp, i64, vp, i64, f32, vp, i64, vp, vp, vp, vp]
        L.spf_check_fault.argtypes = [vp, vp]
        L.spf_last_match_products.argtypes = [vp, C.POINTER(i32)]
        L.spf_debug_fine_grid.argtypes = [vp, vp, vp]
        L.spf_debug_deapodisation.argtypes = [vp, vp]
        L.spf_launch_count.argtypes = [vp]; L.spf_launch_count.restype = i64
        L.spf_slice_match.argtypes = [vp, vp, i64, vp, i64, f32, vp, i64, vp, i64, vp, vp, vp, sz, vp]
        L.spf_slice_match_workspace_bytes.argtypes = [i64, i64, i64]; L.spf_slice_match_workspace_bytes.restype = sz
        L.spf_selftest.argtypes = [vp, C.c_char_p, C.POINTER(SelftestReport), vp]
        L.spf_emu_last_fault.restype = C.c_char_p
        L.spf_emu_set_sm_count.argtypes = [C.c_int]
        L.spf_emu_counters.argtypes = [C.c_void_p, C.c_int]
        _lib = L
    return _lib


def counters(reset=True):
    """{tma_copies, mmas, launches, fiber_switches} since the last reset"""
    out = (C.c_long * 4)()
    lib().spf_emu_counters(out, int(reset))
    return {"tma_copies": out[0], "mmas": out[1], "launches": out[2], "fiber_switches": out[3]}


def smem_counters(reset=True):
    """Shared-memory wavefront accounting of the 16-byte-granular instructions since the last reset (a MODEL: 8 bank groups
    of 16 bytes per wavefront, warp-wide accesses served quarter-warp by quarter-warp, equal addresses merged):
    ldmatrix 8-row phases / the wavefronts they take, cp.async.16 quarter-warp groups / the wavefronts they take."""
    out = (C.c_long * 4)()
    lib().spf_emu_smem_counters(out, int(reset))
    return {"ldsm_phases": out[0], "ldsm_wavefronts": out[1], "cpasync_groups": out[2], "cpasync_wavefronts": out[3]}


def _p(a):
    return C.c_void_p(a.ctypes.data) if a is not None else None


class EmuContext:
    def __init__(self, n, eps=1e-6, sm_count=4):
        self.L = lib()
        self.L.spf_emu_set_sm_count(sm_count)
        self.h = C.c_void_p()
        p = SpfParams(n, eps, 2.0, 0, 0)
        rc = self.L.spf_create(C.byref(self.h), C.byref(p))
        if rc:
            raise EmuError(rc, (self.L.spf_last_error(None) or b"").decode())

    def close(self):
        if getattr(self, "h", None) and self.h.value:
            self.L.spf_destroy(self.h)
            self.h = C.c_void_p()

    __del__ = close

    def _check(self, rc):
        if rc:
            raise EmuError(rc, (self.L.spf_last_error(self.h) or b"").decode())
        f = (self.L.spf_emu_last_fault() or b"").decode()
        if f:
            self.L.spf_emu_clear_fault()
            raise EmuError(-99, "emulator fault: " + f)

    @property
    def info(self):
        out = SpfInfo()
        self._check(self.L.spf_get_info(self.h, C.byref(out)))
        return out

    def set_option(self, key, value):
        self._check(self.L.spf_set_option(self.h, key.encode(), int(value)))

    def set_detector_layout(self, panels, rows, cols):
        self._check(self.L.spf_set_detector_layout(self.h, panels, rows, cols))

    def selftest(self, variant):
        rep = SelftestReport()
        self._check(self.L.spf_selftest(self.h, variant.encode(), C.byref(rep), None))
        return {"passed": bool(rep.passed), "worst_rel": float(rep.worst_rel), "detail": rep.detail.decode(errors="replace")}

    def check_fault(self):
        self._check(self.L.spf_check_fault(self.h, None))

    def prepare_model(self, model):
        model = np.ascontiguousarray(model, np.float32)
        self._check(self.L.spf_prepare_model(self.h, _p(model), None))

    def deapodisation(self):
        out = np.empty(self.info.n, np.float64)
        self._check(self.L.spf_debug_deapodisation(self.h, _p(out)))
        return out

    def fine_grid(self):
        nf = self.info.n_fine
        out = np.empty((nf, nf, nf), np.complex64)
        self._check(self.L.spf_debug_fine_grid(self.h, _p(out), None))
        return out

    def slice(self, quats, pix, out_kind=SPF_OUT_INTENSITY, scale=1.0):
        quats, pix = np.ascontiguousarray(quats, np.float32), np.ascontiguousarray(pix, np.float32)
        M, P = quats.shape[0], pix.shape[0]
        out = np.full((M, P), np.nan, np.complex64 if out_kind == SPF_OUT_COMPLEX else np.float32)
        self._check(self.L.spf_slice(self.h, _p(quats), M, _p(pix), P, out_kind, float(scale), _p(out), None))
        self.check_fault()
        return out

    def match(self, images, slices, mask=None):
        images, slices = np.ascontiguousarray(images, np.float32), np.ascontiguousarray(slices, np.float32)
        n_img, P = images.shape
        M = slices.shape[0]
        need = self.L.spf_match_workspace_bytes(n_img, M, P)
        ws = np.full(need + 1024, 0xFF, np.uint8)
        wp = (ws.ctypes.data + 1023) & ~1023
        bi, bd = np.full(n_img, -7, np.int32), np.full(n_img, np.nan, np.float32)
        mk = None if mask is None else np.ascontiguousarray(mask, np.uint8)
        self._check(self.L.spf_match(self.h, _p(images), n_img, _p(slices), M, P, _p(mk), _p(bi), _p(bd), C.c_void_p(wp), need, None))
        self.check_fault()
        prods = C.c_int32()
        self._check(self.L.spf_last_match_products(self.h, C.byref(prods)))
        return bi, bd, int(prods.value)

    def slice_match(self, quats, pix, images, scale=1.0, mask=None, chunk_M=16):
        quats, pix, images = (np.ascontiguousarray(a, np.float32) for a in (quats, pix, images))
        M, P, n_img = quats.shape[0], pix.shape[0], images.shape[0]
        need = self.L.spf_slice_match_workspace_bytes(n_img, min(chunk_M, M), P)
        ws = np.full(need + 1024, 0xFF, np.uint8)
        wp = (ws.ctypes.data + 1023) & ~1023
        bi, bd = np.full(n_img, -7, np.int32), np.full(n_img, np.nan, np.float32)
        mk = None if mask is None else np.ascontiguousarray(mask, np.uint8)
        self._check(self.L.spf_slice_match(self.h, _p(quats), M, _p(pix), P, float(scale), _p(images), n_img, _p(mk), chunk_M,
                                           _p(bi), _p(bd), C.c_void_p(wp), need, None))
        self.check_fault()
        return bi, bd

    def match_reference(self, images, slices, mask=None):
        images, slices = np.ascontiguousarray(images, np.float32), np.ascontiguousarray(slices, np.float32)
        n_img, P = images.shape
        M = slices.shape[0]
        bi, bd = np.empty(n_img, np.int32), np.empty(n_img, np.float32)
        dist = np.empty((n_img, M), np.float32)
        mk = None if mask is None else np.ascontiguousarray(mask, np.uint8)
        self._check(self.L.spf_match_reference(self.h, _p(images), n_img, _p(slices), M, P, _p(mk), _p(bi), _p(bd), _p(dist), None))
        return bi, bd, dist

    def orientation_match_host(self, model, quats, pix, images, scale=1.0, mask=None):
        model, quats, pix, images = (np.ascontiguousarray(a, np.float32) for a in (model, quats, pix, images))
        M, P, n_img = quats.shape[0], pix.shape[0], images.shape[0]
        bi, bd = np.empty(n_img, np.int32), np.empty(n_img, np.float32)
        sl = np.empty((M, P), np.float32)
        mk = None if mask is None else np.ascontiguousarray(mask, np.uint8)
        self._check(self.L.spf_orientation_match_host(self.h, _p(model), _p(quats), M, _p(pix), P, float(scale), _p(images), n_img, _p(mk),
                                                      _p(bi), _p(bd), _p(sl)))
        return bi, bd, sl
