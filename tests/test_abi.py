"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every symbol include/spf.h declares
(-m "not gpu": no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2109_05339_b200.build import build_lib
    return ctypes.CDLL(build_lib())


def _declared():
    text = open(os.path.join(ROOT, "include", "spf.h")).read()
    return sorted(set(re.findall(r"SPF_API[^;(]*?\b(spf_\w+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 18 and {"spf_prepare_model", "spf_slice", "spf_match"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "libspf.so does not export %s" % n
    from paper_2109_05339_b200 import EXPORTS
    assert sorted(EXPORTS) == names


def test_host_only_planning_calls(lib):
    lib.spf_plan_kernel_width.argtypes = [ctypes.c_double]
    lib.spf_plan_n_fine.argtypes = [ctypes.c_int32, ctypes.c_double]
    lib.spf_match_workspace_bytes.argtypes = [ctypes.c_int64] * 3
    lib.spf_match_workspace_bytes.restype = ctypes.c_size_t
    lib.spf_version.restype = ctypes.c_char_p
    lib.spf_status_string.restype = ctypes.c_char_p
    assert lib.spf_plan_kernel_width(1e-6) == 8 and lib.spf_plan_kernel_width(1e-9) == 10 and lib.spf_plan_kernel_width(1e-4) == 6
    assert lib.spf_plan_kernel_width(0.0) == -1
    assert [lib.spf_plan_n_fine(n, 2.0) for n in (21, 81, 151, 201)] == [42, 162, 320, 420]
    assert lib.spf_plan_n_fine(151, 1.5) == -1
    # two fp16 planes of each operand dominate the workspace
    ws = lib.spf_match_workspace_bytes(10_000, 10_000, 65_536)
    assert 2 * 2 * 2 * 10_000 * 65_536 <= ws <= 2 * 2 * 2 * 10_000 * 65_536 + (1 << 20)
    assert b"sm_100a" in lib.spf_version() and lib.spf_status_string(-4) == b"SPF_ESTATE"


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2109_05339_b200 import SpfContext
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        SpfContext(21)


def test_sass_uses_tcgen05_and_tma():
    """The built library carries the Blackwell-native instructions, not a legacy tensor path."""
    import shutil
    import subprocess
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    from paper_2109_05339_b200 import LIB_PATH
    sass = subprocess.run(["cuobjdump", "-sass", LIB_PATH], capture_output=True, text=True).stdout
    for mnemonic in ("UTCHMMA", "UTMALDG", "LDTM"):
        assert mnemonic in sass
    assert "HGMMA" not in sass
    # the legacy warp-level path (HMMA) exists in exactly one kernel family, the classic-CUDA matcher k_match_mma;
    # the tcgen05 matcher and everything else carry none
    per_fn = {}
    name = None
    for line in sass.splitlines():
        if "Function :" in line:
            name = line.split("Function :")[1].strip()
        elif name and "HMMA" in line and "UTCHMMA" not in line:
            per_fn[name] = per_fn.get(name, 0) + 1
    assert per_fn and all("k_match_mma" in fn for fn in per_fn), sorted(per_fn)
    assert any("UTCHMMA" in l for l in sass.splitlines())
