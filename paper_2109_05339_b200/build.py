"""Build paper_2109_05339_b200/libspf.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libspf.so")
SOURCES = ["spf_api.cu", "spf_prepare.cu", "spf_slice.cu", "spf_match.cu", "spf_selftest.cu", "spf_microbench.cu"]
HEADERS = ["spf_internal.cuh", "ptx_sm100.cuh", "spf_slice_math.cuh", "spf_match_math.cuh", os.path.join("..", "..", "include", "spf.h")]
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fvisibility=hidden", "--expt-relaxed-constexpr"]


if os.environ.get("SPF_DEBUG", "0") == "1":
    # device-side asserts on the invariants the TMA / tcgen05 kernels rely on; objects of a
    # debug build are kept apart so that switching the flag never links a mix
    NVCC_FLAGS += ["-DSPF_DEBUG"]
    LIB = os.path.join(_HERE, "libspf_debug.so")
_OBJ_SUFFIX = ".debug.o" if "-DSPF_DEBUG" in NVCC_FLAGS else ".o"


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu to an object (only the stale ones) and link libspf.so; return its path."""
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    hdr_time = _newest([os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)])
    objs, procs = [], []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", _OBJ_SUFFIX))
        objs.append(o)
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr_time):
            cmd = [nvcc, *NVCC_FLAGS, "-c", s, "-o", o] + (["-Xptxas", "-v"] if verbose else [])
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write("---- nvcc %s ----\n%s\n" % (src, out))
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if procs or force or not os.path.exists(LIB):
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp", *objs, "-L" + os.path.join(CUDA_HOME, "lib64"), "-lcufft",
               "-Xlinker", "-rpath," + os.path.join(CUDA_HOME, "lib64")]
        subprocess.run(cmd, check=True)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv))
