"""Dry-run harness: lets the GPU-side PYTHON code of this repository (paper_2109_05339_b200/binding.py, bench.py's
run_spf, __graft_entry__.smoke(), the -m gpu test functions) execute on a box without a GPU, against
tests/emu/libspf_emu.so.  TEST INFRASTRUCTURE ONLY.

Why: that glue had never executed anywhere (no GPU has been available to this repository), and a NameError in
bench.py would cost the one GPU run the driver makes at round end.  What is swapped, for the duration of
`with dry_run():` only:
  * binding.load_library loads the emulator build (same C ABI, "device" pointers are host pointers), binding._dev accepts
    CPU tensors, binding._stream passes the NULL stream;
  * `torch` as seen by bench.py / __graft_entry__ / binding is a thin proxy: torch.device("cuda", i) -> the CPU device,
    torch.cuda.{is_available, set_device, synchronize, Event, mem_get_info} -> stubs (events measure host time),
    pin_memory arguments are dropped; Tensor.cuda() / Tensor.pin_memory() return the tensor itself.
Everything else -- argument marshalling, workspace sizing, option calls, the order of library calls, the JSON line --
is the real code.  Nothing here is imported by the product.
"""
import contextlib
import os
import sys
import time
import types

HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)


class _Event:
    def __init__(self, enable_timing=False):
        self.t = None

    def record(self, stream=None):
        self.t = time.perf_counter()

    def synchronize(self):
        pass

    def elapsed_time(self, other):
        return 1e3 * (other.t - self.t)


class _TorchProxy(types.ModuleType):
    """`torch` with the CUDA device mapped onto the CPU (attribute access falls through to the real module)."""

    def __init__(self, real):
        super().__init__("torch")
        object.__setattr__(self, "_real", real)
        cuda = types.SimpleNamespace(
            is_available=lambda: True, set_device=lambda *_a, **_k: None, synchronize=lambda *_a, **_k: None,
            Event=_Event, mem_get_info=lambda *_a, **_k: (64 << 30, 180 << 30), device_count=lambda: 1,
            current_stream=lambda *_a, **_k: types.SimpleNamespace(cuda_stream=0),
            get_device_properties=lambda *_a, **_k: types.SimpleNamespace(uuid="emu", name="emulated B200"))
        object.__setattr__(self, "cuda", cuda)

    def device(self, *a, **k):
        return self._real.device("cpu")

    def _factory(self, name):
        fn = getattr(self._real, name)

        def wrapped(*a, **k):
            k.pop("pin_memory", None)
            if "device" in k and str(k["device"]).startswith("cuda"):
                k["device"] = "cpu"
            return fn(*a, **k)
        return wrapped

    def __getattr__(self, name):
        if name in ("empty", "zeros", "ones", "full", "rand", "randint", "randn", "as_tensor", "tensor", "arange", "Generator"):
            return self._factory(name)
        return getattr(self._real, name)


@contextlib.contextmanager
def dry_run(sm_count=4):
    import torch as real_torch
    from build_emu import build_emu
    import paper_2109_05339_b200.binding as b
    import ctypes as C
    proxy = _TorchProxy(real_torch)
    saved = {"lib_path": b.LIB_PATH, "lib": b._lib, "dev": b._dev, "stream": b._stream, "btorch": b.torch,
             "selftest": b.SpfContext.spf_selftest, "microbench": b.SpfContext.spf_microbench, "sys_torch": sys.modules["torch"], "t_cuda": real_torch.Tensor.cuda, "t_pin": real_torch.Tensor.pin_memory,
             "t_to": real_torch.Tensor.to}

    def _dev(t, dtype, what):
        if not isinstance(t, real_torch.Tensor):
            raise TypeError("%s must be a tensor" % what)
        if t.dtype != dtype or not t.is_contiguous():
            raise TypeError("%s must be contiguous %s, got %s" % (what, dtype, t.dtype))
        return C.c_void_p(t.data_ptr())

    def _to(self, *a, **k):
        a = tuple(("cpu" if (isinstance(x, str) and x.startswith("cuda")) else x) for x in a)
        if "device" in k and str(k["device"]).startswith("cuda"):
            k["device"] = "cpu"
        return saved["t_to"](self, *a, **k)

    def _selftest_small(self, variant):          # the emulator cannot afford the check's full-size cases
        self.spf_set_option("selftest_small", 1)
        return saved["selftest"](self, variant)

    def _microbench_small(self, what):           # functional run only: the figure means nothing under emulation
        self.spf_set_option("selftest_small", 1)
        return saved["microbench"](self, what)

    import paper_2109_05339_b200.selfcheck as sc
    saved["child"], saved["cache_env"] = sc.check_in_child, os.environ.get("SPF_SELFCHECK_CACHE")

    def _child_ok(variant, device=0, timeout_s=240.0):   # there is no device for a child process to check: pretend it passed
        return {"ok": True, "status": 0, "kind": "agrees", "detail": "dry run: child check skipped", "seconds": 0.0, "metrics": {}}

    try:
        sc.check_in_child = _child_ok
        sc._cache.clear()
        os.environ["SPF_SELFCHECK_CACHE"] = "off"
        b.SpfContext.spf_selftest, b.SpfContext.spf_microbench = _selftest_small, _microbench_small
        b.LIB_PATH, b._lib = build_emu(), None
        b._dev, b._stream, b.torch = _dev, (lambda device: None), proxy
        lib = b.load_library()
        lib.spf_emu_set_sm_count.argtypes = [C.c_int]
        lib.spf_emu_set_sm_count(sm_count)
        sys.modules["torch"] = proxy
        real_torch.Tensor.cuda = lambda self, *a, **k: self
        real_torch.Tensor.pin_memory = lambda self, *a, **k: self
        real_torch.Tensor.to = _to
        yield proxy
    finally:
        sc.check_in_child = saved["child"]
        sc._cache.clear()
        if saved["cache_env"] is None:
            os.environ.pop("SPF_SELFCHECK_CACHE", None)
        else:
            os.environ["SPF_SELFCHECK_CACHE"] = saved["cache_env"]
        b.SpfContext.spf_selftest, b.SpfContext.spf_microbench = saved["selftest"], saved["microbench"]
        b.LIB_PATH, b._lib, b._dev, b._stream, b.torch = saved["lib_path"], saved["lib"], saved["dev"], saved["stream"], saved["btorch"]
        sys.modules["torch"] = saved["sys_torch"]
        real_torch.Tensor.cuda, real_torch.Tensor.pin_memory, real_torch.Tensor.to = saved["t_cuda"], saved["t_pin"], saved["t_to"]
