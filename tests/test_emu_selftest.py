"""The emulator's own self-test: deliberately broken kernels (tests/emu/selftest/emu_faults.cu), written against the
wrappers of csrc/ptx_sm100.cuh, must be NOTICED -- a test suite that executes the kernels under an emulator is only worth
what the emulator can detect.  Each case runs one tiny kernel; the correct form passes, each broken form either faults
or produces poison (NaN), or -- for a wait that can never complete -- makes the kernels' own watchdog give up."""
import ctypes as C
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))
import emu_binding as eb  # noqa: E402


def _run(family, mode):
    L = eb.lib()
    L.emu_fault_case.argtypes = [C.c_char_p, C.c_int, C.c_void_p]
    L.spf_emu_clear_fault()
    out = np.full(128, np.nan, np.float32)
    assert L.emu_fault_case(family.encode(), mode, out.ctypes.data) == 0
    fault = (L.spf_emu_last_fault() or b"").decode()
    L.spf_emu_clear_fault()
    return out, fault


def test_a_correct_tma_load_passes():
    out, fault = _run("tma", 0)
    assert fault == ""
    want = np.array([y * 16 + x for y in range(8) for x in range(8)], np.float32)       # the (8 x 8 x 1) box at the origin
    assert np.array_equal(out[:64], want)


def test_reading_a_tile_without_waiting_for_its_barrier_reads_poison():
    out, fault = _run("tma", 1)
    assert np.isnan(out[:64]).all()                     # the copy is deferred: the tile still holds the 0xFF poison


def test_a_misaligned_bulk_copy_destination_faults():
    _, fault = _run("tma", 2)
    assert "alignment" in fault


def test_a_barrier_used_before_init_faults():
    _, fault = _run("tma", 3)
    assert "never initialised" in fault


def test_a_wait_that_cannot_complete_trips_the_watchdog():
    out, fault = _run("tma", 4)
    assert fault == "" and np.all(out[:64] == -777.0)   # the bounded wait of ptx_sm100.cuh gave up and said so


def test_tmem_cases():
    out, fault = _run("tmem", 0)
    assert fault == "" and np.isnan(out).all()          # TMEM holds NaN until an MMA writes it: reading it is legal, the value is poison
    assert "quadrant" in _run("tmem", 1)[1]             # a warp may only read its own 32 lanes
    assert "still allocated" in _run("tmem", 2)[1]      # leaving the block without tcgen05.dealloc
    assert "outside the" in _run("tmem", 3)[1]          # columns beyond the allocation
