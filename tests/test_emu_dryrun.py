"""Dry run, on the CPU, of the Python code that will run on the GPU box: bench.py's CUDA arm, __graft_entry__.smoke(),
the ctypes binding and the `-m gpu` test functions themselves -- against the emulator build of the library
(tests/emu/fake_cuda.py).  None of that code had ever executed (no GPU has been available to this repository); a typo
in it would cost the single GPU run the driver makes at round end.  This is a check of the glue and of the TEST CODE,
not of the kernels (tests/test_emu_kernels.py) and not GPU parity.
"""
import argparse
import io
import json
import os
import sys
from contextlib import redirect_stdout

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "tests", "emu"))
sys.path.insert(0, os.path.join(ROOT, "tests"))
from fake_cuda import dry_run  # noqa: E402

FULL = os.environ.get("SPF_EMU_FULL", "1") == "1"      # default: every combination; 0: one representative per code path
full_only = pytest.mark.skipif(not FULL, reason="SPF_EMU_FULL=0: one representative per code path")


def test_bench_cuda_arm_runs_end_to_end_on_tiny():
    """bench.py run_spf, config tiny, library defaults: warm-up, timed region, kernel-time pass, e2e through the
    host-buffer call, oracle baseline, one JSON line with every key the contract names."""
    import bench
    args = argparse.Namespace(gpus=1, steps=2, warmup=3, impl="spf", config="tiny", no_cpu_baseline=False, no_e2e=False,
                              native=False, no_autotune=False, reference_kernels_only=False)
    out = io.StringIO()
    with dry_run(), redirect_stdout(out):
        bench.run_spf(args, bench.CONFIGS["tiny"])
    lines = [l for l in out.getvalue().splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches", "kernels", "breakdown_ms"):
        assert key in j, key
    assert j["n_gpus"] == 1 and j["steps"] == 2 and j["value"] > 0 and j["vs_baseline"] is None
    assert j["config"]["workload"] == "tiny" and j["config"]["w"] == 8
    assert j["config"]["kernel_variants"]["match"].startswith("mma.sync")    # the classic tensor-core matcher passed its in-process check
    sc = j["config"]["kernel_variants"]["selfcheck"]
    assert sc["slice_gcoop"] is True and sc["slice_coop_ld"] is True and sc["match_mma"] is True          # the classic warp-per-point slicers were checked in-process
    assert j["roofline"]["bound"] in ("smem", "tensor") and j["roofline"]["frac"] > 0
    assert j["kernels"]["gemm"]["roofline"]["kernel"] == "k_match_mma" and j["kernels"]["gemm"]["products"] == 2
    assert j["kernels"]["match_prep"]["roofline"]["bound"] == "hbm"
    assert j["gpu_launches"] == 2 * 13                              # 3 prepare, 1 slice, 9 match (common vector, 2 abs-max, 2 split, 2 mma, finalize, refine)
    assert j["e2e"]["value"] > 0 and j["e2e"]["h2d_bytes_per_step"] > 16 * 1024 * 4 and j["e2e"]["d2h_bytes_per_step"] == 16 * 8
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["value"] > 0
    assert j["planted_hit_rate"] is not None
    assert j["peaks"]["lds_gbs"] > 0 and j["peaks"]["l2_to_sm_gbs"] > 0 and "measured in this run" in j["peaks"]["sm_side_source"]
    assert "measured in this run" in j["kernels"]["slice"]["roofline"]["peak_source"]


def test_smoke_runs_on_the_emulator():
    import __graft_entry__ as ge
    with dry_run():
        ge.smoke()


@pytest.fixture(scope="module")
def gpu_tests():
    """The -m gpu test module and its `spf` / `tiny` fixtures' values, built by hand (the functions are called directly)."""
    import test_gpu_parity as t
    import paper_2109_05339_b200 as pkg
    from oracle import oracle as orc
    from spf_inputs import CONFIGS, make_model, make_detector, random_quaternions
    cfg = CONFIGS["tiny"]
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    refs = random_quaternions(cfg.M, seed=2)
    return t, pkg, (cfg, model, pix, refs, orc.slice_points(model, refs, pix))


def test_gpu_parity_test_functions_prepare_and_slice(gpu_tests):
    t, pkg, tiny = gpu_tests
    with dry_run():
        t.test_deapodisation_factors_match_quadrature(pkg)
        for N in (21, 16):
            t.test_fine_grid_is_the_nudft_of_the_deapodised_model(pkg, N)
        t.slice_tiny_full(pkg, tiny, 1, 0, True)
        t.test_slice_is_independent_of_the_patch_layout(pkg, tiny)
        for N, eps in ((16, 1e-6), (21, 1e-9), (12, 1e-4)):
            t.test_slice_general_model_widths_and_even_n(pkg, N, eps)
        t.test_slice_edge_cases(pkg, tiny)


@pytest.mark.parametrize("variant", ["simt", pytest.param("mma", marks=full_only), pytest.param("cg1", marks=full_only), "cg2"])
def test_gpu_parity_test_functions_match_and_end_to_end(gpu_tests, variant):
    t, pkg, tiny = gpu_tests
    with dry_run():
        t.match_vs_oracle_ragged_sizes(pkg, variant, 16, 64, 1024, False)
        t.match_vs_oracle_ragged_sizes(pkg, variant, 5, 300, 1000, True)
        t.match_planted_ties_and_general_values(pkg, variant)
        if variant == "simt":
            t.test_end_to_end_tiny_poisson(pkg, tiny)


def test_gpu_variant_test_functions(gpu_tests):
    """tests/test_gpu_variants.py's own functions for the warp-per-point slicers and the tcgen05 matcher (tiny sizes)."""
    t, pkg, tiny = gpu_tests
    import test_gpu_variants as v
    ok = {k: {"ok": True, "status": 0, "detail": ""} for k in ("slice_gcoop", "slice_coop_ld", "slice_coop", "match_cg1", "match_cg2")}
    with dry_run():
        for name, impl in (v.STAGED if FULL else v.STAGED[-1:]):
            v.test_staged_slice_tiny_full(pkg, tiny, ok, 0, True, name, impl)
            v.test_staged_slice_general_model(pkg, ok, 16, 1e-6, name, impl)
        v.test_staged_slice_equals_the_layout_free_result(pkg, tiny, ok)
        v.test_tcgen05_end_to_end_tiny(pkg, tiny, ok)


def test_gpu_classic_variant_test_functions(gpu_tests):
    """tests/test_gpu_parity_classic_variants.py's own functions (the default-on GPU tests of slice_impl 3 / 4 and the
    mma.sync matcher), tiny sizes."""
    t, pkg, tiny = gpu_tests
    import test_gpu_parity_classic_variants as c
    with dry_run():
        for impl in (c.CLASSIC_SLICERS if FULL else c.CLASSIC_SLICERS[-1:]):
            c.test_classic_slice_tiny_full(pkg, tiny, impl, 0, True)
            c.test_classic_slice_general_model(pkg, impl, 16, 1e-6)
            if FULL:
                c.test_classic_slice_tiny_full(pkg, tiny, impl, 1, False)
                c.test_classic_slice_general_model(pkg, impl, 21, 1e-9)
        c.test_mma_match_vs_oracle_ragged_sizes(pkg, 16, 64, 1024, False)
        if FULL:
            c.test_mma_match_vs_oracle_ragged_sizes(pkg, 5, 300, 1000, True)
            c.test_mma_match_planted_ties_and_general_values(pkg)
