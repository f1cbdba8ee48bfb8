"""Host-side logic of bench.py on CPU: sharding over ranks (world_size 2, gloo), the roofline
arithmetic, and the --impl reference line.  No CUDA call is made here."""
import json
import os
import subprocess
import sys
import types

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # each rank "measures" a different time; the job's time is the max over ranks
    t = bench.dist_max(10.0 + 5.0 * rank, dist)
    # every rank draws its own truth orientations, shares the reference set
    cfg = bench.CONFIGS["tiny"]
    _, _, _, refs, truth, planted = bench.host_inputs(cfg, rank)
    out[rank] = (t, bench.shard_units(cfg.n_img, world), refs.tobytes(), truth.tobytes())
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_images_and_take_the_max_time():
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, 29613, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0[0] == r1[0] == 15.0                  # max over ranks, seen by both
    assert r0[1] == r1[1] == 2 * 16                # weak scaling: units = n_img per rank x world
    assert r0[2] == r1[2]                          # reference orientations replicated
    assert r0[3] != r1[3]                          # images (truth orientations) differ per rank


def test_plain_gpus_2_relaunches_itself_under_torchrun():
    """`python bench.py --gpus 2` with no torchrun environment must run 2 ranks through the same entry the driver
    uses.  --impl hostcheck keeps it on the CPU: gloo rendezvous, max over ranks, one line."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "hostcheck", "--config", "tiny"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                       # rank 0 only
    j = json.loads(lines[0])
    assert j["n_gpus"] == 2 and j["ranks_seen_max_ms"] == 15.0 and j["units"] == 2 * 16
    assert "re-launching under torchrun" in p.stderr


def test_gpus_must_match_world_size():
    env = dict(os.environ, RANK="0", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--impl", "hostcheck"],
                       capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert p.returncode != 0 and "WORLD_SIZE" in p.stderr


def test_dist_max_without_a_process_group_is_the_identity():
    assert bench.dist_max(3.5, None) == 3.5


def test_physical_gpu_index(monkeypatch):
    monkeypatch.delenv("CUDA_VISIBLE_DEVICES", raising=False)
    assert bench.physical_gpu_index(0) == "0"
    monkeypatch.setenv("CUDA_VISIBLE_DEVICES", "5,7")
    assert bench.physical_gpu_index(1) == "7"


def test_roofline_arithmetic_matches_design_md():
    cfg = bench.CONFIGS["paper_scale"]
    info = types.SimpleNamespace(w=7, grid_is_real=1, n_fine=320, sm_count=148)
    peaks = {"hbm_gbs": 6543.4, "tensor_tflops": 1361.5, "sm_max_mhz": 1965.0, "source": "measured"}
    k_ms = {"slice": [12.0, 12.0], "gemm": [38.5], "match_prep": [4.8]}
    k = bench.roofline_objects(cfg, info, k_ms, 2, peaks, {"sm_mhz": 1312.0})
    s = k["slice"]["roofline"]
    assert s["bound"] == "smem" and s["unit"] == "GB/s" and abs(s["peak"] - 148 * 128 * 1.965e9 / 1e9) < 1e-6
    assert "NOMINAL" in s["peak_source"] and abs(s["frac_of_nominal"] - s["frac"]) < 1e-12
    km = bench.roofline_objects(cfg, info, k_ms, 2, dict(peaks, lds_gbs=30000.0), {"sm_mhz": 1312.0})["slice"]["roofline"]
    assert km["peak"] == 30000.0 and "measured in this run" in km["peak_source"] and abs(km["frac"] - s["achieved"] / 30000.0) < 1e-12
    assert abs(s["achieved"] - 10_000 * 65_536 * 343 * 4 / 12e-3 / 1e9) < 1e-3
    assert abs(s["frac"] - s["achieved"] / s["peak"]) < 1e-12
    alu = k["slice"]["alu"]
    assert abs(alu["peak"] - 148 * 128 * 2 * 1.965e9 / 1e12) < 1e-9
    assert abs(alu["achieved"] - 10_000 * 65_536 * 343 * 2 / 12e-3 / 1e12) < 1e-6
    g = k["gemm"]["roofline"]
    assert g["bound"] == "tensor" and g["peak"] == 1361.5
    assert abs(g["achieved"] - 2 * 2.0 * 1e4 * 1e4 * 65_536 / 38.5e-3 / 1e12) < 1e-6
    assert k["match_prep"]["roofline"]["bound"] == "hbm"
    # a complex grid doubles the FMA count per point
    info.grid_is_real = 0
    k2 = bench.roofline_objects(cfg, info, k_ms, 3, peaks, {"sm_mhz": None})
    assert abs(k2["slice"]["roofline"]["achieved"] - 2 * s["achieved"]) < 1e-3
    assert abs(k2["slice"]["alu"]["achieved"] - 2 * alu["achieved"]) < 1e-6
    assert abs(k2["gemm"]["roofline"]["achieved"] - 1.5 * g["achieved"]) < 1e-6
    # CUDA-core matcher (products == 0): ALU roofline against the plain fp32 FMA peak, no operand-preparation entry
    k3 = bench.roofline_objects(cfg, info, k_ms, 0, peaks, {"sm_mhz": None})
    r3 = k3["gemm"]["roofline"]
    assert r3["bound"] == "alu" and abs(r3["peak"] - alu["peak"]) < 1e-9 and r3["mix_ceiling"] == 0.75
    assert abs(r3["achieved"] - 3.0 * 1e4 * 1e4 * 65_536 / 38.5e-3 / 1e12) < 1e-6
    assert k3["match_prep"]["roofline"] is None and k3["match_prep"]["ms"] is None


def test_reference_arm_prints_one_contract_line():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["unit"] == "images/s" and j["value"] > 0
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1
    assert j["e2e"] == {"value": j["value"], "unit": "images/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert j["config"]["workload"] == "tiny" and j["gpu_launches"] == 0


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert p.returncode == 0 and p.stdout.strip() == ""
