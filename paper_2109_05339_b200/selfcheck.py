"""Device self-check of libspf's kernel variants.

libspf has several implementations of each hot kernel: one with the least machinery (plain global
gather; CUDA-core difference-form matcher) and faster ones (warp-per-point gather from global memory;
TMA-staged shared-memory gather, one warp per point; tcgen05 GEMM on single CTAs or cta_group::2 pairs).  The library starts on the first;
`SpfContext.spf_autotune()` switches on the faster ones that pass this self-check on the device at
hand, and among the slicing variants that pass, the one the check timed fastest.

A check runs in a CHILD process (`python -m paper_2109_05339_b200.selfcheck <variant>`): a kernel
that faults poisons its CUDA context, and the caller's must survive that.  The child calls the C library's own
check, `spf_selftest` (include/spf.h, csrc/spf_selftest.cu): the variant against another computation made by the
library's reference kernels on the same device -- the warp-per-point gathers against the one-thread-per-point
gather, the tensor-core matcher against the CUDA-core difference-form reference -- on seeded inputs that span
several tiles and a ragged tail.  All comparison logic is in C; this module only provides the process boundary,
the ordering and the verdict cache.  It is a consistency check between two CUDA paths, not parity: parity
against the oracle is what tests/ does.  Nothing here touches `oracle/`.

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
VARIANTS = ("slice_gcoop", "slice_coop_ld", "match_mma", "slice_coop", "match_cg1", "match_cg2")
CLASSIC = ("slice_gcoop", "slice_coop_ld", "match_mma")      # classic CUDA only: no tensor map, mbarrier, TMEM or tcgen05
SLICE_IMPL = {"slice_coop": 2, "slice_gcoop": 3, "slice_coop_ld": 4}
_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
_cache = {}


def _even_model(n: int, seed: int, even: bool):
    """Seeded random model; `even` makes it exactly even about index floor(n/2) (real fine grid)."""
    import torch
    g = torch.Generator(device="cpu"); g.manual_seed(seed)
    A = torch.randn((n, n, n), generator=g, dtype=torch.float32)
    if even:
        idx = (2 * (n // 2) - torch.arange(n)) % n
        A = 0.5 * (A + A[idx][:, idx][:, :, idx])
        if n % 2 == 0:
            A[0] = 0; A[:, 0] = 0; A[:, :, 0] = 0
    return A


def _check_slice(device: int, variant: str):
    """The comparison itself is the C library's (spf_selftest, csrc/spf_selftest.cu): this only chooses the models
    it is run on -- real and complex fine grid, w = 8 and w = 10, and a 128^3 model (a 266^3-cell grid: beyond L1,
    inside L2) whose timing decides between the slicing variants."""
    import torch
    from .binding import SpfContext
    dev = torch.device("cuda", device)
    worst, metrics = 0.0, {}
    for n, eps, even, timed in ((24, 1e-6, True, False), (21, 1e-6, False, False), (20, 1e-9, True, False), (128, 1e-6, True, True)):
        ctx = SpfContext(n, eps=eps, device=device)
        ctx.spf_prepare_model(_even_model(n, 11 + n, even).to(dev))
        assert bool(ctx.info.grid_is_real) == even
        r = ctx.spf_selftest(variant)
        ctx.close()
        if not r["passed"]:
            raise AssertionError(r["detail"])
        worst = max(worst, r["worst_rel"])
        if timed:
            metrics = {"slice_ms_global": r["ms_reference"], "slice_ms": r["ms_variant"]}
    return "%s == reference gather to %.1e" % (variant, worst), metrics


def _check_match(device: int, variant: str) -> str:
    from .binding import SpfContext
    ctx = SpfContext(8, device=device)
    r = ctx.spf_selftest(variant)
    ctx.close()
    if not r["passed"]:
        raise AssertionError(r["detail"])
    return r["detail"]


def run_variant(variant: str, device: int = 0):
    """Returns (one-line description, metrics dict)."""
    if variant in SLICE_IMPL:
        return _check_slice(device, variant)
    if variant in ("match_mma", "match_cg1", "match_cg2"):
        return _check_match(device, variant), {}
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


def verified_variants(device: int = 0, timeout_s: float = 240.0, report: dict = None, only=None) -> dict:
    """{variant: passed} for every variant (or for the subset `only`, in VARIANTS order), each checked once per
    library build and GPU (cached in the process and on disk)."""
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
    for v in (VARIANTS if only is None else [x for x in VARIANTS if x in only]):
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
