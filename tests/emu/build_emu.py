"""Build tests/emu/libspf_emu.so: libspf's own CUDA sources compiled with g++ against the functional emulator
(cuda_emu.h, ptx_emu.cuh, emu_runtime.cpp).  TEST INFRASTRUCTURE ONLY -- nothing in the product loads the result.

The kernel sources are used as they are, after a purely mechanical rewrite into tests/emu/gen/ (git-ignored):
  * `#include <cuda.h> / <cuda_runtime.h> / <cufft.h> / <cuda_fp16.h>`  ->  `#include "cuda_emu.h"`
  * `kernel<<<grid, block, smem, stream>>>(args);`                      ->  `emu::launch(kernel, grid, block, smem, 1, args);`
  * `extern __shared__ [__align__(n)] T name[];`                        ->  `T *name = (T *)emu::dyn_smem();`
  * ptx_sm100.cuh: every function whose body is inline PTX (`asm volatile`) is dropped and ptx_emu.cuh supplies a
    functional stand-in of the same name; the functions that are plain C++ there (the bounded wait, the abort
    drain, the descriptor builders) are compiled unchanged.
"""
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2109_05339_b200", "csrc")
GEN = os.path.join(HERE, "gen")
LIB = os.path.join(HERE, "libspf_emu.so")
SOURCES = ["spf_api.cu", "spf_prepare.cu", "spf_slice.cu", "spf_match.cu", "spf_selftest.cu", "spf_microbench.cu"]
HEADERS = ["spf_internal.cuh", "ptx_sm100.cuh", "spf_slice_math.cuh", "spf_match_math.cuh"]
EMU_FILES = ["cuda_emu.h", "ptx_emu.cuh", "emu_runtime.cpp", "build_emu.py", os.path.join("selftest", "emu_faults.cu"), os.path.join("selftest", "emu_probes.cu")]
# the emulator's own self-test: deliberately broken kernels, and one-instruction probes compared with CuTe's tables
EXTRA = [os.path.join(HERE, "selftest", "emu_faults.cu"), os.path.join(HERE, "selftest", "emu_probes.cu")]


def _match_close(text, start, open_ch, close_ch):
    """index just past the bracket that closes the one at text[start]"""
    depth = 0
    for i in range(start, len(text)):
        if text[i] == open_ch:
            depth += 1
        elif text[i] == close_ch:
            depth -= 1
            if depth == 0:
                return i + 1
    raise ValueError("unbalanced %s" % open_ch)


def rewrite_launches(text):
    out, pos = [], 0
    while True:
        i = text.find("<<<", pos)
        if i < 0:
            out.append(text[pos:])
            return "".join(out)
        j = i
        while j > 0 and (text[j - 1].isalnum() or text[j - 1] in "_:"):
            j -= 1
        k = text.index(">>>", i)
        cfg = text[i + 3:k]
        a0 = k + 3
        assert text[a0] == "(", text[i - 20:a0 + 20]
        a1 = _match_close(text, a0, "(", ")")
        args = text[a0 + 1:a1 - 1].strip()
        # split the launch configuration at top-level commas
        parts, depth, cur = [], 0, ""
        for ch in cfg:
            if ch in "([":
                depth += 1
            elif ch in ")]":
                depth -= 1
            if ch == "," and depth == 0:
                parts.append(cur.strip()); cur = ""
            else:
                cur += ch
        parts.append(cur.strip())
        grid, block = parts[0], parts[1]
        smem = parts[2] if len(parts) > 2 else "0"
        out.append(text[pos:j])
        out.append("emu::launch(%s, dim3(%s), dim3(%s), (size_t)(%s), 1%s)" % (text[j:i], grid, block, smem, (", " + args) if args else ""))
        pos = a1


def strip_asm_functions(text):
    """drop every function definition whose body contains `asm volatile` (and a `template <...>` line right above it)"""
    out, pos = [], 0
    pat = re.compile(r"(?:template\s*<[^>\n]*>\s*\n)?__device__ __forceinline__ [^;{}()]*\([^{};]*\)\s*\{")
    while True:
        m = pat.search(text, pos)
        if not m:
            out.append(text[pos:])
            return "".join(out)
        end = _match_close(text, m.end() - 1, "{", "}")
        body = text[m.end():end]
        out.append(text[pos:m.start()])
        if "asm volatile" not in body:
            out.append(text[m.start():end])
        pos = end


def transform(name, text):
    text = re.sub(r'#include <(cuda|cuda_runtime|cufft|cuda_fp16)\.h>', '#include "cuda_emu.h"', text)
    text = text.replace('#include "../../include/spf.h"', '#include "%s"' % os.path.join(ROOT, "include", "spf.h"))
    text = re.sub(r'extern __shared__ (?:__align__\(\d+\) )?(\w+) (\w+)\[\];', r'\1 *\2 = (\1 *)emu::dyn_smem();', text)
    if name == "ptx_sm100.cuh":
        text = strip_asm_functions(text)
        text = text.replace("namespace ptx {", '#include "ptx_emu.cuh"\nnamespace ptx {', 1)
        assert "asm volatile" not in text
    if name.endswith(".cu"):
        text = rewrite_launches(text)
        assert "<<<" not in text
    return text


def build_emu(force: bool = False) -> str:
    global LIB
    asan = os.environ.get("SPF_EMU_ASAN", "0") == "1"      # AddressSanitizer build (run python under LD_PRELOAD=libasan.so)
    if asan:
        LIB = os.path.join(HERE, "libspf_emu_asan.so")
    srcs = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, f) for f in EMU_FILES]
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(p) for p in srcs):
        return LIB
    os.makedirs(GEN, exist_ok=True)
    for f in SOURCES + HEADERS:
        with open(os.path.join(CSRC, f)) as fh:
            text = transform(f, fh.read())
        with open(os.path.join(GEN, f.replace(".cu", ".cpp") if f.endswith(".cu") else f), "w") as fh:
            fh.write(text)
    for f in EXTRA:
        with open(f) as fh:
            text = transform(os.path.basename(f), fh.read())
        with open(os.path.join(GEN, os.path.basename(f).replace(".cu", ".cpp")), "w") as fh:
            fh.write(text)
    # the watchdog's bounds count emulator ticks (one per fiber switch), not SM clocks: keep them small so that a
    # pipeline that deadlocks under emulation reports SPF_EFAULT within seconds
    flags = ["-O2", "-g", "-std=c++17", "-fPIC", "-fvisibility=hidden", "-fno-strict-aliasing", "-DSPF_EMU", "-DSPF_DEBUG", "-U_FORTIFY_SOURCE", "-D_FORTIFY_SOURCE=0",
             "-DSPF_WAIT_CYCLES=(1ll<<22)", "-DSPF_DRAIN_CYCLES=(1ll<<8)", "-I" + HERE, "-I" + GEN, "-Wno-unused-value"]
    if asan:
        flags += ["-fsanitize=address", "-fno-omit-frame-pointer"]
    objs, procs = [], []
    for f in [os.path.join(GEN, s.replace(".cu", ".cpp")) for s in SOURCES] + [os.path.join(GEN, os.path.basename(e).replace(".cu", ".cpp")) for e in EXTRA] + [os.path.join(HERE, "emu_runtime.cpp")]:
        o = os.path.join(GEN, os.path.basename(f) + (".asan.o" if asan else ".o"))
        objs.append(o)
        procs.append((f, subprocess.Popen(["g++", *flags, "-c", f, "-o", o], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    bad = False
    for f, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            bad = True
            print("---- g++ %s ----\n%s" % (f, out[-6000:]))
    if bad:
        raise RuntimeError("emulator build failed")
    subprocess.run(["g++", "-shared", *(["-fsanitize=address"] if asan else []), "-o", LIB + ".tmp", *objs], check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build_emu(force="--force" in sys.argv))
