"""The group backward (csrc/gspn_group_bwd.cu, kernel and launcher) run on the host under tests/emu against the oracle.

It sits in GSPN_IMPL_AUTO's fall-back chain but no round-1 GPU test forced it; the GPU test that does
(tests/test_r2_gpu.py::test_group_backward_forced) was written after GPU access had closed.  The kernel is plain CUDA
(threads, __syncthreads, shared memory), so the host emulation runs it as it is: direction masks, h0, optional outputs,
lines shorter and longer than a warp.  See tests/test_line_emulated_cpu.py for what the emulation is.
"""
import ctypes
import os
import subprocess

import numpy as np
import pytest

import gspn_inputs as gi
import parity_util as pu
from test_line_emulated_cpu import to_dev, from_dev, ptr, heavy

HERE = os.path.dirname(os.path.abspath(__file__))
EMU = os.path.join(HERE, "emu")
CSRC = os.path.join(os.path.dirname(HERE), "paper_2606_00746_b200", "csrc")
LIB = os.path.join(EMU, "libgroup_emu.so")


@pytest.fixture(scope="module")
def emu():
    deps = [os.path.join(EMU, f) for f in ("group_emu.cpp", "emu_rt.h", "shim/cuda_runtime.h", "shim/cuda_bf16.h")]
    deps += [os.path.join(CSRC, f) for f in ("gspn_group_bwd.cu", "gspn_common.cuh", "gspn_kernels.h")]
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps):
        subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-fPIC", "-ffp-contract=off", "-w", "-I", EMU, "-I", os.path.join(EMU, "shim"),
                        "-I", CSRC, "-shared", "-o", LIB + ".tmp", deps[0]], check=True)
        os.replace(LIB + ".tmp", LIB)
    L = ctypes.CDLL(LIB)
    vp, ci, cu = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint
    L.emu_group_bwd.argtypes = [vp] * 11 + [ci] * 5 + [cu, ci, ctypes.c_double]
    L.emu_last_error.restype = ctypes.c_char_p
    return L


def run_bwd(L, cfg, dtype, t, need=("dx", "dlambda", "du", "dw3", "dh0")):
    d = {k: to_dev(v) for k, v in t.items()}
    st = d["x"].dtype
    fill = 0x7fc1 if dtype == "bf16" else np.nan
    shapes = {"dx": d["x"].shape, "dlambda": d["lam"].shape, "du": d["u"].shape, "dw3": d["w3"].shape,
              "dh0": (cfg.D, cfg.B, cfg.C, max(cfg.H, cfg.W))}
    out = {k: np.full(shapes[k], fill, dtype=st) for k in need}
    g = lambda k: ptr(out.get(k))
    rc = L.emu_group_bwd(ptr(d["x"]), ptr(d["w3"]), ptr(d["lam"]), ptr(d["u"]), ptr(d.get("h0")), ptr(d["dy"]), g("dx"), g("dlambda"),
                         g("du"), g("dw3"), g("dh0"), cfg.B, cfg.C, cfg.H, cfg.W, cfg.G, cfg.dir_mask, 0 if dtype == "f32" else 1, 60.0)
    return rc, {k: from_dev(v, dtype) for k, v in out.items()}


GROUP_SHAPES = [(1, 4, 27, 27, 1), (2, 4, 8, 8, 2), (1, 2, 40, 44, 2), (1, 4, 33, 35, 1), (1, 2, 100, 36, 1)]      # as the GPU test


@pytest.mark.parametrize("dtype", ["f32", pytest.param("bf16", marks=heavy)])
@pytest.mark.parametrize("shape", [pytest.param(s, marks=heavy) if max(s[2], s[3]) > 64 else s for s in GROUP_SHAPES],
                         ids=["x".join(map(str, s)) for s in GROUP_SHAPES])
def test_group_backward_emulated(emu, shape, dtype):
    ran = 0
    for mask in (15, 6, 9):
        cfg = gi.small_config("grp", *shape, dir_mask=mask, seed=95 + mask, backward=True)      # the GPU test's seeds
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
        rc, g = run_bwd(emu, cfg, dtype, t)
        if rc == 2:
            continue
        assert rc == 0, emu.emu_last_error().decode()
        go, Ag = pu.oracle_bwd(t, cfg)
        for k in go:
            r = pu.gate(g[k], go[k], Ag[k], dtype)
            assert r["ok"], (mask, k, r)
        ran += 1
    if not ran:
        pytest.skip("shape not held by the group kernel: " + emu.emu_last_error().decode())


def test_group_backward_optional_outputs_emulated(emu):
    for shape in [(1, 4, 8, 8, 2), (1, 4, 40, 44, 2)]:          # the shapes of tests/test_r2_gpu.py::test_optional_outputs_per_kernel
        cfg = gi.small_config("opt2", *shape, seed=91, backward=True)
        t = gi.make_inputs(cfg, "f32", device="cpu", with_dy=True)
        rc, full = run_bwd(emu, cfg, "f32", t)
        if rc == 2:
            continue
        assert rc == 0, emu.emu_last_error().decode()
        for need in (("dx",), ("dw3",), ("du", "dh0"), ("dlambda", "dw3"), ("dh0",)):
            rc, part = run_bwd(emu, cfg, "f32", t, need=need)
            assert rc == 0, emu.emu_last_error().decode()
            for k in need:
                np.testing.assert_array_equal(part[k], full[k], err_msg=f"{shape} {need} {k}")
