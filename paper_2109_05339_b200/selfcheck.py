"""Device self-check of libspf's kernel variants.

libspf has several implementations of each hot kernel: one with the least machinery (plain global
gather; CUDA-core difference-form matcher) and faster ones (warp-per-point gather from global memory;
TMA-staged shared-memory gather, one warp per point; tcgen05 GEMM on single CTAs or cta_group::2 pairs).  The library starts on the first;
`SpfContext.spf_autotune()` switches on the faster ones that pass this self-check on the device at
hand, and among the slicing variants that pass, the one the check timed fastest.

A check runs in a CHILD process (`python -m paper_2109_05339_b200.selfcheck <variant>`): a kernel
that faults poisons its CUDA context, and the caller's must survive that.  The child compares the
variant with another computation made by the library's own kernels on the same device -- the
staged gather with the global gather, the tensor-core matcher with the CUDA-core difference-form
matcher (`spf_match_reference`) -- on seeded random inputs that span several tiles and a ragged
tail.  This is a consistency check between two CUDA paths, not parity: parity against the oracle
is what tests/ does.  Nothing here touches `oracle/`.

Exit status of the child: 0 = variant agrees, 1 = disagrees with the reference kernels or the library's
watchdog reported SPF_EFAULT (a verdict about the kernel), 3 = the check itself could not run (import error,
out of memory, any other exception: no verdict), anything else (signal, time-out) = the process died or hung.

Containment: `verified_variants` stops at the FIRST child that died or hung -- a kernel that raises an SM
exception must not be followed by four more launches of unverified kernels on the same device -- and marks
every remaining variant unverified.  Only verdicts (status 0 and 1) are cached on disk; a time-out or an
infrastructure error is retried by the next process.

The whole mechanism is OPT-IN (SpfContext.spf_autotune, bench.py --native, SPF_NATIVE=1 for tests/ and
smoke()): until a variant has passed on hardware the library's defaults are the only kernels launched.
"""
import json
import os
import subprocess
import sys
import time

# least machinery first: classic CUDA (no TMA / mbarrier / tcgen05), then TMA + mbarrier, then tcgen05, CTA pairs last
VARIANTS = ("slice_gcoop", "slice_coop", "match_cg1", "match_cg2")
SLICE_IMPL = {"slice_coop": 2, "slice_gcoop": 3}
_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
_cache = {}


def _check_slice_staged(device: int, impl: int):
    import torch
    from .binding import SpfContext, SPF_OUT_COMPLEX
    dev = torch.device("cuda", device)
    g = torch.Generator(device="cpu"); g.manual_seed(11)
    worst = 0.0
    for n, eps, even in ((24, 1e-6, True), (21, 1e-6, False), (20, 1e-9, True)):
        A = torch.randn((n, n, n), generator=g, dtype=torch.float32)
        if even:   # A[n] == A[-n] about index floor(n/2): exercises the real-grid kernels
            c = n // 2
            idx = (2 * c - torch.arange(n)) % n
            Af = A[idx][:, idx][:, :, idx]
            A = 0.5 * (A + Af)
            if n % 2 == 0:
                A[0] = 0; A[:, 0] = 0; A[:, :, 0] = 0
        rows = cols = 40     # 1,600 pixels: 8 x 16 lattice patches with ragged edges
        u = (torch.arange(cols, dtype=torch.float64) - (cols - 1) / 2) / cols
        v = (torch.arange(rows, dtype=torch.float64) - (rows - 1) / 2) / rows
        vv, uu = torch.meshgrid(v, u, indexing="ij")
        k = torch.stack([uu, vv, torch.ones_like(uu)], -1)
        q = k / k.norm(dim=-1, keepdim=True) - torch.tensor([0.0, 0.0, 1.0], dtype=torch.float64)
        pix = (q * (0.9 * torch.pi / q.norm(dim=-1).max())).reshape(-1, 3).to(torch.float32)
        quats = torch.randn((37, 4), generator=g, dtype=torch.float32)
        ctx = SpfContext(n, eps=eps, device=device)
        ctx.spf_set_detector_layout(1, rows, cols)
        ctx.spf_prepare_model(A.to(dev))
        assert bool(ctx.info.grid_is_real) == even
        outs = []
        for which in (1, impl):
            ctx.spf_set_option("slice_impl", which)
            outs.append(ctx.spf_slice(quats.to(dev), pix.to(dev), SPF_OUT_COMPLEX))
            ctx.spf_check_fault()
        err = float((outs[1] - outs[0]).abs().pow(2).sum().sqrt() / outs[0].abs().pow(2).sum().sqrt())
        worst = max(worst, err)
        # the two variants differ only in how the kernel weights are evaluated (polynomial fit vs exp/sqrt)
        if not err <= 3e-6:
            raise AssertionError("staged vs global gather: relative L2 %.3e (n=%d eps=%g)" % (err, n, eps))
        ctx.close()
    return "slice_impl %d == global gather to %.1e" % (impl, worst), _time_slice(device, impl)


def _time_slice(device: int, impl: int) -> dict:
    """Milliseconds of spf_slice for 64 orientations x 65,536 pixels (4 panels of 128 x 128, about 0.9 fine cells
    per pixel as at Paper-scale) of a 128^3 even model (real grid of 266^3 cells = 75 MB: beyond L1, inside L2,
    w = 7), global gather and variant `impl`, best of 3 (CUDA events on the current stream)."""
    import torch
    from .binding import SpfContext, SPF_OUT_INTENSITY
    dev = torch.device("cuda", device)
    g = torch.Generator(device="cpu"); g.manual_seed(3)
    n = 128
    A = torch.randn((n, n, n), generator=g, dtype=torch.float32)
    idx = (2 * (n // 2) - torch.arange(n)) % n
    A = 0.5 * (A + A[idx][:, idx][:, :, idx])
    A[0] = 0; A[:, 0] = 0; A[:, :, 0] = 0
    edge = 128
    t = (torch.arange(edge, dtype=torch.float64) - (edge - 1) / 2) / (2 * edge)
    pix = []
    for cy in (-0.26, 0.26):
        for cx in (-0.26, 0.26):
            vv, uu = torch.meshgrid(t + cy, t + cx, indexing="ij")
            k = torch.stack([uu, vv, torch.ones_like(uu)], -1)
            pix.append((k / k.norm(dim=-1, keepdim=True) - torch.tensor([0.0, 0.0, 1.0], dtype=torch.float64)).reshape(-1, 3))
    pix = torch.cat(pix)
    pix = (pix * (0.9 * torch.pi / pix.norm(dim=-1).max())).to(torch.float32).to(dev)
    n_or = 64
    quats = torch.randn((n_or, 4), generator=g, dtype=torch.float32).to(dev)
    ctx = SpfContext(n, eps=1e-6, device=device)
    ctx.spf_set_detector_layout(4, edge, edge)
    ctx.spf_prepare_model(A.to(dev))
    out = torch.empty((n_or, pix.shape[0]), dtype=torch.float32, device=dev)
    ms = {}
    for which in (1, impl):
        ctx.spf_set_option("slice_impl", which)
        best = float("inf")
        for rep in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.spf_slice(quats, pix, SPF_OUT_INTENSITY, out=out)
            e1.record()
            e1.synchronize()
            if rep:
                best = min(best, e0.elapsed_time(e1))
        ctx.spf_check_fault()
        ms["global" if which == 1 else "variant"] = best
    ctx.close()
    return {"slice_ms_global": ms["global"], "slice_ms": ms["variant"], "points": n_or * int(pix.shape[0])}


def _check_match(device: int, cta_group: int) -> str:
    import torch
    from .binding import SpfContext
    dev = torch.device("cuda", device)
    g = torch.Generator(device="cpu"); g.manual_seed(5 + cta_group)
    ctx = SpfContext(8, device=device)
    ctx.spf_set_option("match_impl", 0)             # the tcgen05 kernel (the library default is the CUDA-core matcher)
    ctx.spf_set_option("match_cta_group", cta_group)
    worst = 0.0
    for n_img, M, P, counts in ((300, 513, 2048, True), (130, 257, 200, False), (5, 40, 4100, True)):
        S = torch.rand((M, P), generator=g) * torch.rand((M, 1), generator=g) * 3.0
        pick = torch.randint(0, M, (n_img,), generator=g)
        I = torch.poisson(S[pick], generator=g) if counts else S[pick] + 0.1 * torch.rand((n_img, P), generator=g)
        mask = (torch.rand(P, generator=g) > 0.2).to(torch.uint8)
        for mk in (None, mask):
            dI, dS = I.to(dev).contiguous(), S.to(dev).contiguous()
            dm = None if mk is None else mk.to(dev)
            ri, rd, dist = ctx.spf_match_reference(dI, dS, dm)
            keep = torch.ones(P, device=dev) if dm is None else dm.float()
            nrm = (dI * dI * keep).sum(1) + ((dS * dS * keep).sum(1))[ri.long()]
            for refine in (1, 0):
                ctx.spf_set_option("match_refine", refine)
                bi, bd = ctx.spf_match(dI, dS, dm)
                ctx.spf_check_fault()
                torch.cuda.synchronize(dev)
                # refine = 1 (the library's result): 1e-4 of d against the CUDA-core difference-form reference.
                # refine = 0 exposes the epilogue's own a_i + b_m - 2 G: a sanity bound on the contraction itself,
                # 1e-4 d plus 2e-6 of the norms (the expansion's fp32 cancellation floor); not a parity bar.
                tol = 1e-4 * rd if refine else 1e-4 * rd + 2e-6 * nrm
                rel = ((bd - rd).abs() / rd.clamp_min(1e-30)).max().item()
                if refine:
                    worst = max(worst, rel)
                if not bool(((bd - rd).abs() <= tol).all()):
                    raise AssertionError("cta_group %d (refine %d): distance differs from the CUDA-core matcher by %.3e" % (cta_group, refine, rel))
                # argmin may differ only where the reference's own margin is within tolerance
                d_at = dist.gather(1, bi.long().clamp(0, M - 1)[:, None])[:, 0]
                bad = (bi != ri) & ((d_at - rd) > tol)
                if bool(bad.any()) or bool((bi < 0).any()) or bool((bi >= M).any()):
                    raise AssertionError("cta_group %d (refine %d): argmin differs from the CUDA-core matcher" % (cta_group, refine))
    ctx.close()
    return "cta_group::%d == CUDA-core matcher, distances to %.1e" % (cta_group, worst)


def run_variant(variant: str, device: int = 0):
    """Returns (one-line description, metrics dict)."""
    if variant in SLICE_IMPL:
        return _check_slice_staged(device, SLICE_IMPL[variant])
    if variant == "match_cg1":
        return _check_match(device, 1), {}
    if variant == "match_cg2":
        return _check_match(device, 2), {}
    raise ValueError("unknown variant %r (one of %s)" % (variant, ", ".join(VARIANTS)))


def check_in_child(variant: str, device: int = 0, timeout_s: float = 240.0) -> dict:
    """Run one variant's check in a child process.  Returns {"ok", "status", "detail", "seconds"}."""
    t0 = time.time()
    cmd = [sys.executable, "-m", "paper_2109_05339_b200.selfcheck", variant, "--device", str(device)]
    try:
        p = subprocess.run(cmd, cwd=_ROOT, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=timeout_s)
        status, out = p.returncode, p.stdout
    except subprocess.TimeoutExpired as e:
        status, out = -999, (e.stdout or "") if isinstance(e.stdout, str) else ""
        out += "\n[selfcheck] timed out after %.0f s" % timeout_s
    lines = [ln for ln in out.strip().splitlines() if ln.strip()]
    metrics = {}
    for ln in lines:
        if ln.startswith("[selfcheck-json] "):
            try:
                metrics = json.loads(ln[len("[selfcheck-json] "):])
            except ValueError:
                pass
    tail = [ln for ln in lines if not ln.startswith("[selfcheck-json] ")][-3:]
    kind = "agrees" if status == 0 else ("disagrees" if status == 1 else ("no_verdict" if status == 3 else "died"))
    return {"ok": status == 0, "status": status, "kind": kind, "detail": " | ".join(tail)[-400:],
            "seconds": round(time.time() - t0, 1), "metrics": metrics}


def fastest_slice_impl(report: dict) -> int:
    """slice_impl to use given a verified_variants report: the verified variant with the lowest timed
    spf_slice, provided it beat the global gather in its own child's timing; else 1 (global gather)."""
    best, best_ms = 1, None
    for v, impl in SLICE_IMPL.items():
        r = report.get(v) or {}
        m = r.get("metrics") or {}
        if not r.get("ok") or "slice_ms" not in m:
            continue
        if m["slice_ms"] < m.get("slice_ms_global", float("inf")) and (best_ms is None or m["slice_ms"] < best_ms):
            best, best_ms = impl, m["slice_ms"]
    return best


def _disk_cache_path(device: int) -> str:
    """One file per (library build, GPU) under <repository>/gpurun_out/selfcheck/: a later PROCESS of the same
    job reuses the verdicts instead of launching a variant that already faulted once more (every bench /
    test / profiler process would otherwise repeat the fault).  Keyed by the SHA-1 of libspf.so and the GPU's
    UUID, so a rebuilt library or another device is always checked afresh; the directory lives inside the
    working copy, so nothing carries over from an earlier job on a reused machine.
    SPF_SELFCHECK_CACHE=off disables it, any other value is the directory to use."""
    import hashlib
    where = os.environ.get("SPF_SELFCHECK_CACHE", "")
    if where.lower() == "off":
        return ""
    from .binding import LIB_PATH
    try:
        with open(LIB_PATH, "rb") as f:
            h = hashlib.sha1(f.read()).hexdigest()[:16]
        import torch
        uuid = str(getattr(torch.cuda.get_device_properties(device), "uuid", "gpu%d" % device))
        where = where or os.path.join(_ROOT, "gpurun_out", "selfcheck")
        os.makedirs(where, exist_ok=True)
    except Exception:
        return ""
    return os.path.join(where, "libspf_selfcheck_%s_%s.json" % (h, uuid.replace("/", "_")))


def verified_variants(device: int = 0, timeout_s: float = 240.0, report: dict = None) -> dict:
    """{variant: passed} for every variant, each checked once per library build and GPU (cached in the
    process and on disk)."""
    path = _disk_cache_path(device)
    disk = {}
    if path and os.path.exists(path):
        try:
            with open(path) as f:
                disk = json.load(f)
        except Exception:
            disk = {}
    out = {}
    stopped_by = None
    for v in VARIANTS:
        key = (v, device)
        if key not in _cache:
            if stopped_by is not None:
                # not cached (in the process or on disk): a later process starts again from the variant that died
                r = {"ok": False, "status": None, "kind": "not_run", "seconds": 0.0, "metrics": {},
                     "detail": "not launched: the check of %s died or hung before it" % stopped_by}
                sys.stderr.write("[libspf selfcheck] %-12s NOT RUN (%s)\n" % (v, r["detail"]))
                out[v] = False
                if report is not None:
                    report[v] = r
                continue
            if v in disk and isinstance(disk[v], dict) and disk[v].get("kind") in ("agrees", "disagrees"):
                _cache[key] = disk[v]
                sys.stderr.write("[libspf selfcheck] %-12s %s (cached verdict from %s)\n" % (v, "ok" if disk[v]["ok"] else "FAILED", path))
            else:
                r = check_in_child(v, device, timeout_s)
                sys.stderr.write("[libspf selfcheck] %-12s %s (%s, %.1f s)\n" % (
                    v, "ok" if r["ok"] else "FAILED status %s (%s)" % (r["status"], r["kind"]), r["detail"], r["seconds"]))
                if r["kind"] == "died":
                    stopped_by = v
                if r["kind"] in ("agrees", "disagrees", "died"):
                    _cache[key] = r          # a kernel that died is not launched again by THIS process ...
                if r["kind"] in ("agrees", "disagrees"):
                    disk[v] = r              # ... but only verdicts persist across processes
                    if path:
                        try:
                            with open(path + ".tmp", "w") as f:
                                json.dump(disk, f)
                            os.replace(path + ".tmp", path)
                        except Exception:
                            pass
                out[v] = r["ok"]
                if report is not None:
                    report[v] = r
                continue
        elif _cache[key].get("kind") == "died":
            stopped_by = stopped_by or v
        out[v] = _cache[key]["ok"]
        if report is not None:
            report[v] = _cache[key]
    return out


if __name__ == "__main__":
    import argparse
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("variant", choices=VARIANTS + ("all",))
    ap.add_argument("--device", type=int, default=0)
    a = ap.parse_args()
    if a.variant == "all":
        rep = {}
        verified_variants(a.device, report=rep)
        print(json.dumps(rep))
        sys.exit(0 if all(r["ok"] for r in rep.values()) else 1)
    try:
        text, metrics = run_variant(a.variant, a.device)
        print("[selfcheck-json] " + json.dumps(metrics))
        print("[selfcheck] %s: %s" % (a.variant, text))
    except AssertionError as e:   # the variant disagrees with the reference kernels: a verdict
        print("[selfcheck] %s FAILED: %s: %s" % (a.variant, type(e).__name__, e))
        sys.exit(1)
    except Exception as e:
        # SPF_EFAULT (the kernel's watchdog gave up) is a verdict about the kernel; anything else (import error,
        # out of memory, a CUDA error from an unrelated call) is not
        print("[selfcheck] %s FAILED: %s: %s" % (a.variant, type(e).__name__, e))
        sys.exit(1 if getattr(e, "status", None) == -5 else 3)
