"""Third-party pins for the instruction-level facts the kernels and the emulator rely on.

No B200 has been available to this repository, so the tcgen05 / TMA / mma.sync kernels have only ever executed under the
functional emulator of tests/emu/.  That evidence is worth what the emulator's reading of each instruction is worth.  The
CUTLASS / CuTe header tree vendored in this image states those readings as data -- descriptor bit-field unions, swizzle
atoms, fragment layouts -- and tests/cutlass_pin/cutlass_tables.cu (a HOST program; nothing is launched) prints them.
Here they are compared with
  * csrc/ptx_sm100.cuh's own descriptor builders (umma_desc_sw128, umma_idesc_f16), compiled unchanged;
  * the emulator's models, exercised through one-instruction probe kernels written against the same wrappers the library's
    kernels use (tests/emu/selftest/emu_probes.cu): where TMA puts element (row, k) of a 128-byte-swizzled tile, where
    tcgen05.mma reads it from (start address, SBO, swizzle, the +32-byte K step), tcgen05.ld's lane / column mapping,
    the fragment layouts of mma.sync.m16n8k16 and ldmatrix.x4.
A wrong bit position, a transposed fragment or a mis-stepped K advance in either fails here.  CUTLASS is a reference for
the TESTS only; the product neither includes nor links it.  Skipped when the header tree or nvcc is not there.
"""
import ctypes as C
import json
import os
import shutil
import subprocess
import sys
import sysconfig

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "emu"))
import emu_binding as eb  # noqa: E402

PIN = os.path.join(HERE, "cutlass_pin")


def _cutlass_include():
    roots = {sysconfig.get_paths()["purelib"], sysconfig.get_paths()["platlib"]}
    for root in roots:
        for sub in ("flashinfer/data/cutlass/include", "tilelang/3rdparty/cutlass/include"):
            p = os.path.join(root, sub)
            if os.path.exists(os.path.join(p, "cute", "arch", "mma_sm100_desc.hpp")):
                return p
    return None


@pytest.fixture(scope="module")
def tables():
    inc, nvcc = _cutlass_include(), shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if inc is None or not os.path.exists(nvcc):
        pytest.skip("no CUTLASS header tree / nvcc in this image")
    src, gen = os.path.join(PIN, "cutlass_tables.cu"), os.path.join(PIN, "gen")
    exe = os.path.join(gen, "cutlass_tables")
    os.makedirs(gen, exist_ok=True)
    if not os.path.exists(exe) or os.path.getmtime(exe) < os.path.getmtime(src):
        subprocess.run([nvcc, "-std=c++17", "-w", "-I" + inc, "-gencode", "arch=compute_100a,code=sm_100a", src, "-o", exe], check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    # on the host CuTe's smem-pointer cast prints one "ERROR: cast_smem_ptr_to_uint not supported" line and returns 0:
    # the start-address field is the only thing it feeds, and that field is checked below from our own builder
    return json.loads("".join(l for l in out.splitlines(True) if not l.startswith("ERROR")))


@pytest.fixture(scope="module")
def L():
    lib = eb.lib()
    lib.emu_probe_smem_desc.restype = C.c_ulonglong
    lib.emu_probe_smem_desc.argtypes = [C.c_uint]
    lib.emu_probe_idesc.restype = C.c_uint
    lib.emu_probe_idesc.argtypes = [C.c_int, C.c_int]
    for f in ("emu_probe_mma", "emu_probe_ldsm", "emu_probe_tma"):
        getattr(lib, f).restype = C.c_int
    for f in ("emu_probe_umma", "emu_probe_umma_pair"):
        getattr(lib, f).restype = C.c_int
        getattr(lib, f).argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
    lib.spf_emu_clear_fault()
    return lib


def _no_fault(lib):
    fault = (lib.spf_emu_last_fault() or b"").decode()
    lib.spf_emu_clear_fault()
    assert fault == "", fault


def test_instruction_descriptor_bits_are_cutlass_bits(tables, L):
    """umma_idesc_f16(M, N) == UMMA::make_instr_desc<half, half, float, M, N, K-major, K-major>() for every tile shape
    k_match_gemm instantiates (single CTA: M 128; CTA pair: M 256)."""
    for key, want in tables["idesc"].items():
        M, N = (int(x) for x in key.split("x"))
        assert L.emu_probe_idesc(M, N) == want, key


def test_shared_memory_descriptor_fields_are_cutlass_fields(tables, L):
    """umma_desc_sw128(addr): LBO, SBO, version, layout type, base offset and LBO mode as UMMA::make_umma_desc<Major::K>
    computes them for tile_to_shape(Layout_K_SW128_Atom<half>, (128, 64)); start address = (addr mod 2^18) >> 4, the
    CTA-rank bits of a cluster-window address dropped."""
    sd = tables["smem_desc"]
    for addr in (0, 0x400, 0x1C400, 0x8000 | (1 << 24)):
        d = L.emu_probe_smem_desc(addr)
        assert d & 0x3FFF == (addr & 0x3FFFF) >> 4
        assert (d >> 14) & 3 == 0 and (d >> 30) & 3 == 0
        assert (d >> 16) & 0x3FFF == sd["lbo"]
        assert (d >> 32) & 0x3FFF == sd["sbo"]
        assert (d >> 46) & 3 == sd["version"]
        assert (d >> 49) & 7 == sd["base_offset"] and (d >> 52) & 1 == sd["lbo_mode"]
        assert (d >> 61) & 7 == sd["layout_type"]
        assert d >> 32 == sd["hi"]                                  # nothing else set in the upper word


def test_tma_writes_the_swizzled_tile_where_cutlass_says(tables, L):
    """cp.async.bulk.tensor.2d through a SWIZZLE_128B map, box {64 fp16, 16 rows}: element (row, k) lands at CuTe's byte
    offset for the K-major SW128 atom (the emulator's TMA model; the same positions k_match_gemm's operands rely on)."""
    off = np.array(tables["sw128_byte_offset"])
    t = (np.arange(16 * 64, dtype=np.uint16) + 1000).reshape(16, 64)
    out = np.zeros(2048, np.uint8)
    assert L.emu_probe_tma(t.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p)) == 0
    _no_fault(L)
    got = out.view(np.uint16)
    assert np.array_equal(got[off[:16] // 2], t)
    assert sorted(off[:16].ravel().tolist()) == list(range(0, 2048, 2))     # the atom tiles the 16 rows exactly


def _image(mat, off):
    """byte image of a K-major SW128 tile holding fp16 matrix `mat` [rows][64], element (r, k) at CuTe's offset"""
    img = np.zeros(mat.shape[0] * 128, np.uint8)
    img.view(np.float16)[off[:mat.shape[0]] // 2] = mat
    return img


@pytest.mark.parametrize("kk", [0, 1, 2, 3])
def test_tcgen05_mma_reads_operands_where_cutlass_puts_them(tables, L, kk):
    """One tcgen05.mma (M 128, N 64, K 16) issued exactly as k_match_gemm issues it -- descriptors from umma_desc_sw128,
    K step kk as +2 kk in the address field -- on operand tiles laid out by CuTe's table: D = A[:, 16kk:16kk+16] .
    B[:, 16kk:16kk+16]^T, read back with tcgen05.ld 32x32b.x16 (thread = TMEM lane = row, register = column)."""
    off = np.array(tables["sw128_byte_offset"])
    rng = np.random.default_rng(10 + kk)
    A = rng.integers(-8, 9, (128, 64)).astype(np.float16)
    B = rng.integers(-8, 9, (64, 64)).astype(np.float16)
    imgA, imgB = _image(A, off), _image(B, off)
    out = np.zeros((128, 64), np.float32)
    assert L.emu_probe_umma(imgA.ctypes.data, imgB.ctypes.data, kk, out.ctypes.data) == 0
    _no_fault(L)
    ks = slice(16 * kk, 16 * kk + 16)
    want = A[:, ks].astype(np.float32) @ B[:, ks].astype(np.float32).T
    assert np.array_equal(out, want)
    t = tables
    assert t["tmem_ld_dst_bit"] == [0, 512, 511] and t["tmem_dp_bits"] == 32 << 16     # lane field at address bit 16, 16 x 32-bit columns per thread


@pytest.mark.parametrize("kk", [0, 3])
def test_tcgen05_mma_on_a_cta_pair_splits_rows_as_cutlass_says(tables, L, kk):
    """cta_group::2, M 256 x N 64, one instruction from the leader: CTA v supplies the rows of A and B, and receives the
    rows of D, that MMA_Traits<SM100_MMA_F16BF16_2x1SM_SS<..., 256, 64, ...>> assigns it (A and D: 128 v ... 128 v + 127;
    B: 32 v ... 32 v + 31), every tile at the same shared-memory offset in both CTAs."""
    pr = tables["pair_256x64"]
    assert pr["A_row"] == [[0, 127], [128, 255]] and pr["B_row"] == [[0, 31], [32, 63]] and pr["D_row"] == [[0, 127], [128, 255]]
    off = np.array(tables["sw128_byte_offset"])
    rng = np.random.default_rng(20 + kk)
    A = rng.integers(-8, 9, (256, 64)).astype(np.float16)
    B = rng.integers(-8, 9, (64, 64)).astype(np.float16)
    imgA = np.concatenate([_image(A[pr["A_row"][v][0]:pr["A_row"][v][1] + 1], off) for v in (0, 1)])
    imgB = np.concatenate([_image(B[pr["B_row"][v][0]:pr["B_row"][v][1] + 1], off) for v in (0, 1)])
    out = np.zeros((256, 64), np.float32)                           # CTA v writes rows D_row[v]
    assert L.emu_probe_umma_pair(imgA.ctypes.data, imgB.ctypes.data, kk, out.ctypes.data) == 0
    _no_fault(L)
    ks = slice(16 * kk, 16 * kk + 16)
    assert np.array_equal(out, A[:, ks].astype(np.float32) @ B[:, ks].astype(np.float32).T)


def test_mma_sync_fragments_are_cutlass_fragments(tables, L):
    """mma.sync.m16n8k16 (f16 x f16 -> f32): registers filled and read by MMA_Traits<SM80_16x8x16_F32F16F16F32_TN>'s
    A / B / C layouts give A . B (the emulator's fragment model; k_match_mma's operand feeding depends on it)."""
    rng = np.random.default_rng(3)
    A = rng.integers(-8, 9, (16, 16)).astype(np.float16)            # [m][k]
    B = rng.integers(-8, 9, (8, 16)).astype(np.float16)             # [n][k] ("TN": both K-contiguous)
    regs = np.zeros((32, 6), np.uint32)
    halves = regs.view(np.uint16).reshape(32, 12)                    # little endian: half 0 of a register is its low 16 bits
    for t in range(32):
        for v, (m, k) in enumerate(tables["mma_A"][t]):
            halves[t, v] = A[m, k].view(np.uint16)
        for v, (n, k) in enumerate(tables["mma_B"][t]):
            halves[t, 8 + v] = B[n, k].view(np.uint16)
    out = np.zeros((32, 4), np.float32)
    assert L.emu_probe_mma(regs.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p)) == 0
    _no_fault(L)
    got = np.full((16, 8), np.nan, np.float32)
    for t in range(32):
        for v, (m, n) in enumerate(tables["mma_C"][t]):
            got[m, n] = out[t, v]
    assert np.array_equal(got, A.astype(np.float32) @ B.astype(np.float32).T)


def test_ldmatrix_x4_is_cutlass_ldsm(tables, L):
    """ldmatrix.sync.aligned.m8n8.x4.shared.b16: register j of thread t holds the 32 bits Copy_Traits<SM75_U32x4_LDSM_N>
    assigns it, source thread s supplying the row whose address it passed (any permutation of rows)."""
    rng = np.random.default_rng(4)
    rows = rng.integers(0, 256, (32, 16)).astype(np.uint8)
    perm = rng.permutation(32).astype(np.int32)
    out = np.zeros((32, 4), np.uint32)
    assert L.emu_probe_ldsm(rows.ctypes.data_as(C.c_void_p), perm.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p)) == 0
    _no_fault(L)
    assert tables["ldsm_src_bit"] == [128 * s for s in range(32)]
    for t in range(32):
        for j in range(4):
            bit = tables["ldsm_dst_bit"][t][j]
            s, byte = bit // 128, (bit % 128) // 8
            assert out[t, j] == rows[perm[s], byte:byte + 4].view(np.uint32)[0], (t, j)
