"""The host emulation's own semantics (tests/emu/emu_rt.h, emu_ptx.h), pinned by small scenarios: if the emulation is the
evidence for kernels that have not run on a GPU, what it takes an mbarrier, a TMA box or a tensor-memory access to mean
must itself be checkable.  Expected values come from the PTX rules, written out here, not from the emulation."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
EMU = os.path.join(HERE, "emu")
CSRC = os.path.join(os.path.dirname(HERE), "paper_2606_00746_b200", "csrc")
LIB = os.path.join(EMU, "libemu_selftest.so")


@pytest.fixture(scope="module")
def st():
    deps = [os.path.join(EMU, f) for f in ("emu_selftest.cpp", "emu_rt.h", "emu_ptx.h", "shim/cuda_runtime.h", "shim/cuda_bf16.h", "shim/cuda.h")]
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-fPIC", "-w", "-I", EMU, "-I", os.path.join(EMU, "shim"), "-I", CSRC,
                        "-shared", "-o", LIB + ".tmp", deps[0]], check=True)
        os.replace(LIB + ".tmp", LIB)
    L = ctypes.CDLL(LIB)
    L.emu_err.restype = ctypes.c_char_p
    L.emu_out.restype = ctypes.POINTER(ctypes.c_int)
    L.st_tma_clip.argtypes = [ctypes.c_void_p]
    L.st_tma_swizzle.argtypes = [ctypes.c_void_p]
    L.st_tmem.argtypes = [ctypes.c_int]
    return L


def aligned(a: np.ndarray) -> np.ndarray:
    """A copy of `a` whose first byte is 16-byte aligned (TMA's rule for the global address)."""
    raw = np.empty(a.nbytes + 16, dtype=np.uint8)
    off = (-raw.ctypes.data) % 16
    out = raw[off:off + a.nbytes].view(a.dtype).reshape(a.shape)
    out[...] = a
    return out


def test_mbarrier_wait_by_parity(st):
    """A fresh mbarrier: waiting for parity 1 succeeds at once (the phase before the first counts as complete), parity 0
    needs `count` arrivals; once phase 0 is complete a wait for parity 0 keeps succeeding while phase 1 is open -- which is
    why a waiter must not skip a phase (csrc/gspn_line_fwd.cu, the per-direction full barriers)."""
    assert st.st_mbar_parity() == 0, st.emu_err()
    assert list(st.emu_out()[0:3]) == [1, 1, 1]


def test_mbarrier_transaction_bytes(st):
    assert st.st_mbar_tx() == 0, st.emu_err()
    assert st.emu_out()[1] == 63                     # the waiter saw the last of the 256 bytes


def test_mbarrier_over_arrival_is_an_error(st):
    assert st.st_mbar_overarrive() == 1 and b"more arrivals" in st.emu_err()


def test_a_wait_nobody_completes_is_reported(st):
    assert st.st_deadlock() == 1
    msg = st.emu_err()
    assert b"deadlock" in msg and b"1 of 2 arrivals pending" in msg


def test_tma_box_clipping_and_zero_fill(st):
    t = aligned(np.arange(2 * 5 * 8, dtype=np.float32).reshape(2, 5, 8))
    ref = t.copy()
    assert st.st_tma_clip(t.ctypes.data_as(ctypes.c_void_p)) == 0, st.emu_err()
    o = st.emu_out()
    # rows 3 and 4 of plane 1 arrive, rows 5 and 6 (outside the tensor) are zeros
    assert o[0] == 1 and o[1] == int(ref[1, 3, 0]) and o[2] == int(ref[1, 4, 7]) and o[3] == 0 and o[4] == 0
    # the store wrote the two rows inside the tensor and nothing else
    want = ref.copy()
    want[1, 3] = 1000 + np.arange(8); want[1, 4] = 1008 + np.arange(8)
    np.testing.assert_array_equal(t, want)


def test_tma_swizzle_32b(st):
    """CU_TENSOR_MAP_SWIZZLE_32B: the 16-byte half of a 32-byte row is exchanged where address bit 7 is set, i.e. in rows
    4..7 and 12..15 of a 1024-aligned stage (csrc/gspn_line_fwd.cu line_hoff)."""
    t = aligned(np.arange(16 * 16, dtype=np.uint16).reshape(16, 16))
    assert st.st_tma_swizzle(t.ctypes.data_as(ctypes.c_void_p)) == 0, st.emu_err()
    o = st.emu_out()
    first = [o[1 + r] for r in range(16)]
    want = [int(t[r, 8 if (r >> 2) & 1 else 0]) for r in range(16)]
    assert o[0] == 1 and first == want


def test_tensor_memory_rules(st):
    assert st.st_tmem(0) == 0, st.emu_err()
    assert st.emu_out()[0] == 37                     # thread 37 = warp 1, lane 5 reads back what it stored in its own lane
    assert st.st_tmem(1) == 1 and b"its own quarter" in st.emu_err()
    assert st.st_tmem(2) == 1 and b"beyond the 32 allocated" in st.emu_err()
