"""bench.py -- one JSON line for the M-TIP orientation-matching hot path on B200 (contract: DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config paper_scale] [--impl spf|reference] [--native]

A "step" is one pass of the whole hot path over one batch of
synthetic input: spf_prepare_model -> spf_slice (M x P points) -> spf_match (n_img x M x P).
  value   orientation-matched images / s for the whole step, inputs resident in HBM
  e2e     the same through spf_orientation_match_host with pinned HOST buffers (copies inside the timed region)
  roofline / kernels   per-kernel device times (CUDA events recorded by the library on the launching stream)
  cpu_baseline   the oracle, as it stands, timed on this box's host cores on a bounded sample (rank 0, N = 1)
N > 1 (under torchrun, or plain `python bench.py --gpus N`, which re-launches itself under torchrun): images are partitioned across ranks, the model and all M orientations replicated --
the paper's scheme; no data-path collective; "scaling": "weak".
--impl reference times the oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from spf_inputs import (CONFIGS, make_model, make_detector, make_mask, random_quaternions,  # noqa: E402
                        planted_truth_quaternions, photon_scale, poisson_images, sample_pairs)

METRIC = "orientation-matched images/sec (whole step: prepare + slice + match)"
UNIT = "images/s"
ORACLE_POINTS = 8192      # NUDFT sample of the cpu_baseline / reference arm (>= 4,096; about 6 s on 8 cores at N = 151)
ORACLE_IMAGES = 64        # images x ALL M slices brute-forced by the oracle (>= 64; about 15 s on 8 cores at M = 10,000)


def _peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": float(p["hbm_gbs"]), "tensor_tflops": float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                "tensor_tflops_burst": float(p["bf16_tflops"]), "sm_max_mhz": float(p.get("sm_max_mhz", 1965.0)),
                "source": "measured"}
    except Exception:
        return {"hbm_gbs": 6650.0, "tensor_tflops": 1400.0, "tensor_tflops_burst": 1590.0, "sm_max_mhz": 1965.0,
                "source": "fallback"}


def measure_device_peaks(ctx):
    """The SM-side denominators, measured on this device in this run (spf_microbench, csrc/spf_microbench.cu; SURVEY.md
    section 8(d)): aggregate shared-memory load bandwidth (the slicing roofline's peak) and L2 -> SM bandwidth, plus an HBM copy
    as a sanity check against MEASURED_PEAKS.json.  A failure leaves the nominal figures in place and says so."""
    out = {}
    try:
        lds = {k: ctx.spf_microbench(k) for k in ("lds32", "lds128")}
        out["lds_gbs"] = max(lds.values())
        out["lds_gbs_by_load_width"] = lds
        out["l2_to_sm_gbs"] = ctx.spf_microbench("l2")
        out["hbm_copy_gbs_this_run"] = ctx.spf_microbench("hbm_copy")
        out["sm_side_source"] = "measured in this run by spf_microbench (best of 3 after a warm-up, CUDA events)"
    except Exception as e:      # the rooflines then fall back to the nominal SM-side figures
        out["sm_side_source"] = "nominal (spf_microbench failed: %s)" % repr(e)[:120]
    return out


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def __exit__(self, *a):
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
# workload (inputs only: spf_inputs holds none of the method's arithmetic)
# ------------------------------------------------------------------------------------------------
def host_inputs(cfg, rank=0):
    """Model, detector, mask and quaternions of one rank.  The model, detector, mask and reference set are
    the same on every rank (replicated); the truth orientations (hence the images) differ."""
    model = make_model(cfg.N, cfg.n_atoms, cfg.atom_radius)
    pix = make_detector(cfg.panels, cfg.panel_edge)
    mask = make_mask(cfg.panels, cfg.panel_edge, cfg.masked_frac)
    refs = random_quaternions(cfg.M, seed=2)
    truth, planted = planted_truth_quaternions(cfg.n_img, refs, seed=3 + 1000 * rank)
    return model, pix, mask, refs, truth, planted


def physical_gpu_index(local):
    """nvidia-smi index of CUDA device `local` (CUDA_VISIBLE_DEVICES may renumber)."""
    vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
    ids = [v.strip() for v in vis.split(",") if v.strip()]
    return ids[local] if local < len(ids) else str(local)


def shard_units(n_img_per_rank, world):
    """Weak scaling: every rank matches its own n_img images against all M orientations."""
    return n_img_per_rank * world


def dist_max(x, dist=None):
    """max over ranks of a Python float (the only collective in the job: timing, not data)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ------------------------------------------------------------------------------------------------
# the oracle on a bounded sample (cpu_baseline leg and --impl reference; the only places oracle/ runs)
# ------------------------------------------------------------------------------------------------
def oracle_match_inputs(cfg, pix, n_images, m_slices):
    """Inputs of the oracle's matching sample (the oracle cannot slice M x P points here): surrogate model images
    generated 1,000 rows at a time (each block its own seed, so the fp64 temporaries stay small) and Poisson images
    drawn from evenly spaced rows."""
    from spf_inputs import surrogate_slices
    S = np.empty((m_slices, cfg.P), np.float32)
    for s0 in range(0, m_slices, 1000):
        n = min(1000, m_slices - s0)
        S[s0:s0 + n] = surrogate_slices(n, pix, seed=5 + s0)
    S *= np.float32(cfg.photons / max(float(S[:min(m_slices, 1000)].sum(axis=1, dtype=np.float64).mean()), 1e-30))
    I = poisson_images(S[(np.arange(n_images) * max(1, m_slices // max(1, n_images))) % m_slices])
    return I, S


def oracle_sample(cfg, model, pix, mask, refs, n_points, n_images, m_slices, match_inputs=None):
    """Times oracle NUDFT on n_points sampled (orientation, pixel) pairs and oracle brute-force matching of
    n_images images against m_slices model images of P pixels; extrapolates to the whole step."""
    from oracle import oracle as orc
    sm, sj = sample_pairs(cfg.M, cfg.P, n_points)
    t0 = time.perf_counter()
    orc.slice_points(model, refs, pix, sm, sj)
    t_slice = time.perf_counter() - t0
    I, S = match_inputs if match_inputs is not None else oracle_match_inputs(cfg, pix, n_images, m_slices)
    t0 = time.perf_counter()
    orc.match(I, S, mask)
    t_match = time.perf_counter() - t0
    pts_s = n_points / t_slice
    pairs_s = n_images * m_slices / t_match
    t_full = cfg.M * cfg.P / pts_s + cfg.n_img * cfg.M / pairs_s
    return {"value": cfg.n_img / t_full, "unit": UNIT, "cores": int(orc.num_threads()), "kind": "oracle",
            "sample": "%d NUDFT points of %d^3 voxels (%.1f s) + %d images x %d slices x %d pixels brute force (%.1f s); "
                      "value extrapolated to M*P = %.3g points and n_img*M = %.3g pairs"
                      % (n_points, cfg.N, t_slice, n_images, m_slices, cfg.P, t_match, cfg.M * cfg.P, cfg.n_img * cfg.M),
            "slice_points_per_s": pts_s, "match_pairs_per_s": pairs_s, "seconds": t_slice + t_match}


def run_reference(args, cfg):
    """--impl reference: the oracle as it stands on this box's host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    model, pix, mask, refs, _, _ = host_inputs(cfg)
    scale = min(1.0, 8.0 / max(1, args.steps + args.warmup))     # keep the whole run within a few minutes
    n_pts, n_im = max(1024, int(ORACLE_POINTS * scale)), max(4, int(ORACLE_IMAGES * scale))
    m_s = cfg.M if cfg.M <= 20_000 else 20_000                   # all M slices (host memory bounds the largest config)
    inputs = oracle_match_inputs(cfg, pix, n_im, m_s)            # generated once, outside every timed sample
    last, times = None, []
    for it in range(args.warmup + args.steps):
        last = oracle_sample(cfg, model, pix, mask, refs, n_pts, n_im, m_s, inputs)
        if it >= args.warmup:
            times.append(last)
    value = float(np.mean([t["value"] for t in times]))
    secs = float(np.mean([t["seconds"] for t in times]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * cfg.n_img / value, "ms_per_sample": 1e3 * secs,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "N": cfg.N, "P": cfg.P, "M": cfg.M, "n_img": cfg.n_img, "eps": cfg.eps},
            "cpu_baseline": {k: last[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    line["cpu_baseline"]["value"] = value
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
def run_spf(args, cfg):
    import torch
    import torch.distributed as dist
    import __graft_entry__ as ge
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libspf has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        ge.build()
    if world > 1:
        dist.barrier()
    from paper_2109_05339_b200 import SpfContext, SPF_OUT_INTENSITY

    model, pix, mask, refs, truth, planted = host_inputs(cfg, rank)
    ctx = SpfContext(cfg.N, eps=cfg.eps, device=local)
    ctx.spf_set_detector_layout(cfg.panels, cfg.panel_edge, cfg.panel_edge)
    # kernel variants: the library defaults, or with --native the faster ones (TMA-staged gather, tcgen05 GEMM) whose
    # device self-check passes in a child process (paper_2109_05339_b200/selfcheck.py).  Opt-in until those kernels
    # have been cleared on hardware: the default run never launches an unverified kernel.
    variants = {"slice_impl": 1, "match_impl": 1, "match_cta_group": 1, "tier": "reference kernels"}
    info = ctx.info
    measured = measure_device_peaks(ctx) if rank == 0 or world > 1 else {}
    d_model = torch.from_numpy(model).to(dev)
    d_pix, d_refs = torch.from_numpy(pix).to(dev), torch.from_numpy(refs).to(dev)
    d_mask = None if mask is None else torch.from_numpy(mask).to(dev)

    # workload generation (outside every timed region): Poisson means come from the CUDA slicer at the
    # truth orientations -- inputs, not a correctness reference
    ctx.spf_prepare_model(d_model)
    # Kernel variants.  Default: the classic-CUDA fast tier (warp-per-point slicers from global memory / from a cp.async-staged
    # tile, the mma.sync matcher -- no tensor map, mbarrier, TMEM or tcgen05 in any of them).  --native adds the TMA-staged slicer
    # and the tcgen05 matcher (opt-in until cleared on hardware).  Either way every candidate is checked by
    # the C library's spf_selftest in a CHILD process first and switched on only if it agrees with the reference kernels.
    if not args.reference_kernels_only:
        variants = ctx.spf_autotune(classic_only=not args.native)
        variants["tier"] = "classic + TMA / tcgen05 (--native)" if args.native else "classic CUDA (default)"
    slices = ctx.spf_slice(d_refs, d_pix, SPF_OUT_INTENSITY, scale=1.0)
    alpha = photon_scale(slices, mask, cfg.photons)
    images = torch.empty((cfg.n_img, cfg.P), dtype=torch.float32, device=dev)
    d_truth = torch.from_numpy(truth).to(dev)
    for s in range(0, cfg.n_img, 1000):
        lam = ctx.spf_slice(d_truth[s:s + 1000].contiguous(), d_pix, SPF_OUT_INTENSITY, scale=alpha)
        images[s:s + 1000] = poisson_images(lam, seed=4 + s + 100000 * rank)
    del lam
    ctx.spf_set_option("record_events", 1)

    def step():
        ctx.spf_prepare_model(d_model)
        ctx.spf_slice(d_refs, d_pix, SPF_OUT_INTENSITY, scale=alpha, out=slices)
        return ctx.spf_match(images, slices, d_mask)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    ctx.spf_check_fault()      # raises if any kernel's watchdog gave up: no number from a broken pipeline
    products = ctx.spf_last_match_products() if args.warmup > 0 else None
    def measure():
        """EXACTLY args.steps timed steps between two barriers; CUDA events on the current stream; clocks sampled."""
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
        sync_all()
        launches0 = ctx.spf_launch_count()
        with ClockSampler(physical_gpu_index(local)) as clocks:
            for k in range(args.steps):
                ev[k][0].record()
                ctx.spf_prepare_model(d_model)
                ev[k][1].record()
                ctx.spf_slice(d_refs, d_pix, SPF_OUT_INTENSITY, scale=alpha, out=slices)
                ev[k][2].record()
                bi, bd = ctx.spf_match(images, slices, d_mask)
                ev[k][3].record()
            sync_all()
            launches = ctx.spf_launch_count() - launches0
            # Per-kernel device times: the library's own CUDA events around the dominant kernels (recorded on the
            # launching stream).  Reading them synchronises the host, so they are taken in a SECOND pass of the same
            # steps, after the timed region has closed and still under the clock sampler -- `value` has no host
            # bubbles, and each kernel's time is the mean over args.steps launches.
            k_ms = {"slice": [], "gemm": [], "match_prep": []}
            for k in range(args.steps):
                ctx.spf_prepare_model(d_model)
                ctx.spf_slice(d_refs, d_pix, SPF_OUT_INTENSITY, scale=alpha, out=slices)
                ctx.spf_match(images, slices, d_mask)
                k_ms["slice"].append(ctx.spf_last_kernel_ms(0))
                k_ms["gemm"].append(ctx.spf_last_kernel_ms(1))
                k_ms["match_prep"].append(ctx.spf_last_kernel_ms(2))
            torch.cuda.synchronize()
        ctx.spf_check_fault()
        return ev, k_ms, launches, clocks.summary(), bi

    # a run that saw a hardware or thermal slowdown is rejected and measured once more (timing rules)
    remeasured = False
    ev, k_ms, launches, clk, best_idx = measure()
    bad = sorted(set(clk["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"})
    if bad:
        remeasured = True
        time.sleep(5.0)
        ev, k_ms, launches, clk, best_idx = measure()
        bad = sorted(set(clk["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"})
    if products is None:
        products = ctx.spf_last_match_products()
    total_ms = ev[0][0].elapsed_time(ev[-1][3])
    total_ms = dist_max(total_ms, dist if world > 1 else None)
    part = lambda a, b: float(np.mean([ev[k][a].elapsed_time(ev[k][b]) for k in range(args.steps)]))
    prepare_ms, slice_ms, match_ms = part(0, 1), part(1, 2), part(2, 3)
    ms_per_step = total_ms / args.steps
    value = shard_units(cfg.n_img, world) / (ms_per_step * 1e-3)

    # sanity statistic of the result (not a correctness check: tests/ do that)
    sel = planted >= 0
    hit = float((best_idx.cpu().numpy()[sel] == planted[sel]).mean()) if sel.any() else None

    peaks = _peaks()
    peaks.update(measured)
    kern = roofline_objects(cfg, info, k_ms, products, peaks, clk, "k_match_mma" if variants["match_impl"] == 2 else "k_match_gemm")
    dominant = max(("slice", "gemm"), key=lambda n: kern[n]["ms"])
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (slicing, fp64 coordinates); f16x2-split products with f32 accumulation (matching)",
            "data": "synthetic",
            "config": {"workload": cfg.name, "N": cfg.N, "n_fine": info.n_fine, "w": info.w, "P": cfg.P, "M": cfg.M,
                       "n_img_per_gpu": cfg.n_img, "eps": cfg.eps, "masked_frac": cfg.masked_frac,
                       "grid_is_real": bool(info.grid_is_real),
                       "kernel_variants": {"slice": {1: "global_gather, thread per point",
                                                     2: "tma_staged, warp per point", 3: "global_gather, warp per point",
                                                     4: "cp_async_staged, warp per point"}[variants["slice_impl"]],
                                           "match": ("tcgen05 cta_group::%d" % variants["match_cta_group"]) if variants["match_impl"] == 0
                                                    else ("mma.sync (legacy tensor-core path, classic CUDA; tcgen05 variant %s)" if variants["match_impl"] == 2
                                                          else "cuda_core difference form (library default; tcgen05 variant %s)") % ("failed its self-check" if args.native else "not requested"),
                                           "selfcheck": variants},
                       "parallelism": "images partitioned x%d, orientations replicated" % world,
                       "l2": "inputs larger than L2 (slices %.2f GB, images %.2f GB per step; no flush needed)"
                             % (cfg.M * cfg.P * 4e-9, cfg.n_img * cfg.P * 4e-9)},
            "breakdown_ms": {"prepare_model": prepare_ms, "slice": slice_ms, "match": match_ms},
            "slice_points_per_s": cfg.M * cfg.P * world / (slice_ms * 1e-3),
            "match_images_per_s": cfg.n_img * world / (match_ms * 1e-3),
            "roofline": kern[dominant]["roofline"], "kernels": kern, "peaks": peaks,
            "clocks": {"sm_mhz": clk["sm_mhz"], "sm_max_mhz": clk["sm_max_mhz"], "reasons": clk["reasons"], "rejected_for": bad,
                       "remeasured": remeasured},
            "gpu_launches": int(launches), "planted_hit_rate": hit}

    # end to end through the C-ABI host-buffer call (pinned host memory, copies inside the timed region)
    if args.no_e2e:
        line["e2e"] = {"value": None, "unit": UNIT, "skipped": "--no-e2e"}
    else:
        try:
            line["e2e"] = run_e2e(args, cfg, ctx, model, refs, pix, mask, images, alpha, world, dist if world > 1 else None)
        except Exception as e:  # the device-resident number stands on its own
            line["e2e"] = {"value": None, "unit": UNIT, "error": repr(e)[:200]}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        try:
            base = oracle_sample(cfg, model, pix, mask, refs, ORACLE_POINTS, ORACLE_IMAGES, cfg.M if cfg.M <= 20_000 else 20_000)
            line["cpu_baseline"] = {k: base[k] for k in ("value", "unit", "cores", "kind", "sample", "slice_points_per_s", "match_pairs_per_s")}
        except Exception as e:
            line["cpu_baseline"] = {"value": None, "unit": UNIT, "kind": "oracle", "error": repr(e)[:200]}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def roofline_objects(cfg, info, k_ms, products, peaks, clk, tensor_kernel="k_match_gemm"):
    """Per-kernel roofline entries from the library's CUDA-event times.

    slice kernel: bound on chip -- every point needs w^3 grid values brought from shared memory to a lane
      (128 B/clk/SM) and w^3 (real grid) or 2 w^3 (complex grid) FMAs (128 lanes/clk/SM); the first is the
      tighter limit by 4x and is the `roofline` entry ("smem"), the FMA-pipe ("alu") and HBM figures (bytes
      written + the touched part of the grid read once) are reported beside it.
    GEMM: tensor pipe.  achieved = issued MMA flop (all split products); peak = measured sustained bf16 cuBLAS
      throughput (fp16 and bf16 share one rate).  The fp32-equivalent algorithmic rate is reported beside it.
    """
    out = {}
    w, real = int(info.w), bool(info.grid_is_real)
    pts = cfg.M * cfg.P
    t_s = float(np.mean(k_ms["slice"])) * 1e-3
    flop = pts * (w ** 3) * 2.0 * (1 if real else 2)
    alu_peak = info.sm_count * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12      # TFLOP/s
    ach = flop / t_s / 1e12
    n_f = int(info.n_fine)
    ball = (4.0 / 3.0) * np.pi * (0.45 * n_f + w) ** 3 * (4 if real else 8)     # touched part of the fine grid, read once
    hbm_bytes = pts * 4.0 + min(ball, n_f ** 3 * (4.0 if real else 8.0))
    # SM-side memory roofline (north_star's "memory roofline" as SURVEY.md section 8(d) reads it): every point needs
    # w^3 grid values (4 B real, 8 B complex) delivered from shared memory / L1 to a lane, against 128 B/clk/SM
    smem_bytes = pts * (w ** 3) * (4.0 if real else 8.0)
    smem_nominal = info.sm_count * 128 * peaks["sm_max_mhz"] * 1e6 / 1e9             # GB/s, the guide's 128 B/clk/SM at max clock
    smem_peak = float(peaks.get("lds_gbs") or smem_nominal)                            # measured in this run when available
    smem_ach = smem_bytes / t_s / 1e9
    out["slice"] = {"ms": t_s * 1e3, "points_per_s": pts / t_s,
                    "roofline": {"kernel": "k_slice", "bound": "smem", "achieved": smem_ach, "peak": smem_peak, "unit": "GB/s",
                                 "frac": smem_ach / smem_peak, "traffic": None,
                                 "peak_source": ("aggregate shared-memory load bandwidth measured in this run (spf_microbench)" if peaks.get("lds_gbs")
                                                 else "NOMINAL 148 SM x 128 B/clk x sm_max_mhz (no measurement)") +
                                                "; algorithmic bytes = w^3 grid values per point (DESIGN.md section 6.1); HBM and FMA-pipe figures beside it",
                                 "peak_nominal": smem_nominal, "frac_of_nominal": smem_ach / smem_nominal,
                                 "frac_of_nominal_at_observed_clock": (smem_ach / (smem_nominal * clk["sm_mhz"] / peaks["sm_max_mhz"])) if clk.get("sm_mhz") else None},
                    "alu": {"achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak,
                            "peak_source": "148 SM x 128 FMA lanes x 2 x sm_max_mhz"},
                    "hbm": {"algorithmic_bytes": hbm_bytes, "achieved_gbs": hbm_bytes / t_s / 1e9, "peak_gbs": peaks["hbm_gbs"],
                            "frac": hbm_bytes / t_s / 1e9 / peaks["hbm_gbs"]}}
    t_g = float(np.mean(k_ms["gemm"])) * 1e-3
    Ppad = (cfg.P + 63) // 64 * 64
    alg = 2.0 * cfg.n_img * cfg.M * Ppad
    if products:
        ach = products * alg / t_g / 1e12
        out["gemm"] = {"ms": t_g * 1e3, "products": products, "algorithmic_tflops_fp32_equivalent": alg / t_g / 1e12,
                       "images_per_s": cfg.n_img / t_g,
                       "roofline": {"kernel": tensor_kernel, "bound": "tensor", "achieved": ach, "peak": peaks["tensor_tflops"],
                                    "unit": "TFLOP/s", "frac": ach / peaks["tensor_tflops"], "traffic": None,
                                    "peak_source": "%s sustained bf16 cuBLAS (fp16 = bf16 rate)" % peaks["source"]}}
    else:
        # CUDA-core matcher (library default): one FADD (the difference) + one FFMA (square and add) per pixel pair =
        # 3 flop in 2 issue slots.  Peak = the fp32 FMA pipe (guide: 128 lanes/clk/SM, 2 flop per FFMA); this
        # instruction mix can reach at most 3/4 of it, which `mix_ceiling` states -- no credit is taken for it.
        ach = 3.0 * cfg.n_img * cfg.M * cfg.P / t_g / 1e12
        out["gemm"] = {"ms": t_g * 1e3, "products": 0, "algorithmic_tflops_fp32_equivalent": alg / t_g / 1e12,
                       "images_per_s": cfg.n_img / t_g,
                       "roofline": {"kernel": "k_match_simt", "bound": "alu", "achieved": ach, "peak": alu_peak,
                                    "unit": "TFLOP/s", "frac": ach / alu_peak, "traffic": None, "mix_ceiling": 0.75,
                                    "peak_source": "fp32 FMA pipe: %d SM x 128 lanes x 2 flop x sm_max_mhz (DESIGN.md section 6); "
                                                   "FADD + FFMA per pixel pair = 3 flop per 2 slots, so <= 0.75 of it"
                                                   % info.sm_count}}
    if not products:
        # the CUDA-core matcher has no operand preparation (only a memset of the argmin keys): nothing to report
        out["match_prep"] = {"ms": None, "roofline": None, "skipped": "no operand preparation ran (CUDA-core matcher)"}
        return out
    t_p = float(np.mean(k_ms["match_prep"])) * 1e-3
    prep_bytes = (cfg.n_img + cfg.M) * cfg.P * 4.0 * 2 + (cfg.n_img + cfg.M) * Ppad * 4.0   # abs-max read + split read + 2 fp16 planes written
    out["match_prep"] = {"ms": t_p * 1e3,
                         "roofline": {"kernel": "k_absmax + k_split", "bound": "hbm", "achieved": prep_bytes / t_p / 1e9,
                                      "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": prep_bytes / t_p / 1e9 / peaks["hbm_gbs"],
                                      "traffic": None}}
    return out


def run_e2e(args, cfg, ctx, model, refs, pix, mask, images_dev, alpha, world, dist):
    """The user's call with HOST buffers: every step uploads model, quaternions, pixels, mask and the images
    from pinned memory, runs prepare -> slice -> match, and downloads (best_idx, best_dist)."""
    import torch
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_model, h_refs, h_pix = pin(model), pin(refs), pin(pix)
    h_mask = None if mask is None else pin(mask)
    h_images = torch.empty(images_dev.shape, dtype=torch.float32, pin_memory=True)
    h_images.copy_(images_dev)
    torch.cuda.synchronize()
    steps = max(1, min(args.steps, 5))
    for _ in range(2):
        ctx.spf_orientation_match_host(h_model, h_refs, h_pix, h_images, scale=alpha, mask=h_mask)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        bi, bd = ctx.spf_orientation_match_host(h_model, h_refs, h_pix, h_images, scale=alpha, mask=h_mask)
    torch.cuda.synchronize()
    dt = dist_max(time.perf_counter() - t0, dist)
    h2d = model.nbytes + refs.nbytes + pix.nbytes + (0 if mask is None else mask.nbytes) + h_images.numel() * 4
    d2h = bi.nbytes + bd.nbytes
    return {"value": shard_units(cfg.n_img, world) * steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
            "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * dt / steps, "steps": steps,
            "timer": "host clock around the synchronous C-ABI call spf_orientation_match_host (max over ranks)"}


def respawn_under_torchrun(args, argv):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: re-exec the same command line as
    `python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py ...`
    (one rank per GPU), so the plain command the driver uses for N = 1 also works for N > 1.  Returns the exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")          # keep NCCL's communicator log on: the rank check reads it
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    sys.stderr.write("bench.py: --gpus %d without WORLD_SIZE: re-launching under torchrun (port %d)\n" % (args.gpus, port))
    return subprocess.call(cmd, env=env)


def run_hostcheck(args):
    """--impl hostcheck (CPU test of the N > 1 launch path, tests/test_bench_host.py): rendezvous over gloo, shard the
    units, take the max-over-ranks of a per-rank number, rank 0 prints one line.  No CUDA call, no kernel, no oracle."""
    import torch.distributed as dist
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    cfg = CONFIGS[args.config]
    t = dist_max(10.0 + 5.0 * rank, dist if world > 1 else None)
    if rank == 0:
        print(json.dumps({"impl": "hostcheck", "n_gpus": world, "ranks_seen_max_ms": t, "units": shard_units(cfg.n_img, world),
                          "scaling": "weak"}), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="spf", choices=["spf", "reference", "hostcheck"])
    ap.add_argument("--config", default="paper_scale", choices=sorted(CONFIGS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (profiler runs)")
    ap.add_argument("--native", action="store_true",
                    help="self-check the TMA / tcgen05 kernel variants in child processes and use the ones that pass "
                         "(opt-in until cleared on hardware; default: the library's default kernels only)")
    ap.add_argument("--no-autotune", action="store_true", help="(default behaviour now; kept for old command lines)")
    ap.add_argument("--reference-kernels-only", action="store_true",
                    help="skip even the in-process check of the classic-CUDA warp-per-point slicer: reference gather + CUDA-core matcher")
    args = ap.parse_args()
    if args.steps < 1:
        raise SystemExit("--steps must be >= 1")
    cfg = CONFIGS[args.config]
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        raise SystemExit(respawn_under_torchrun(args, sys.argv[1:]))
    if "WORLD_SIZE" in os.environ and int(os.environ["WORLD_SIZE"]) != args.gpus and args.impl != "reference":
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%s" % (args.gpus, os.environ["WORLD_SIZE"]))
    if args.impl == "hostcheck":
        run_hostcheck(args)
    elif args.impl == "reference":
        run_reference(args, cfg)
    else:
        if args.warmup < 3:
            sys.stderr.write("bench.py: warm-up raised to 3 (timing rules)\n")
            args.warmup = 3
        run_spf(args, cfg)


if __name__ == "__main__":
    main()
