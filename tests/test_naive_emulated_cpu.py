"""The DEVICE code of the naive kernels (csrc/gspn_naive.cuh), run on the host by tests/emu/naive_emu.cpp, against the
oracle -- on a machine without a GPU.

Why: GPU access for this repository closed in round 2 before the shared-slab (`dir_stride_* = 0`) and chunked-scan
(`k_chunk`) options of the naive kernels could run on hardware.  The naive kernels use nothing but threadIdx,
__syncthreads and shared memory, so the very file nvcc compiles can be compiled by g++ against a small shim and run one
thread block at a time with host threads.  What this checks is the kernels' index arithmetic and control flow (the same
source); what it cannot check is anything specific to the GPU (launch configuration limits, fma contraction by nvcc is
not at play: the kernels call fmaf explicitly, which the host evaluates with the same single rounding).
The GPU parity tests (tests/test_parity_gpu.py, tests/test_r2_gpu.py) remain the parity evidence; this is the
CPU-side safety net under them.
"""
import ctypes
import os
import subprocess

import numpy as np
import pytest
import torch

import gspn_inputs as gi
import parity_util as pu
from oracle import gspn_oracle as orc

# the default run keeps one storage type / one chunk count per option; GSPN_EMU_FULL=1 runs the full grid
heavy = pytest.mark.skipif(os.environ.get("GSPN_EMU_FULL") != "1", reason="set GSPN_EMU_FULL=1 for the full grid of emulated cases")

HERE = os.path.dirname(os.path.abspath(__file__))
EMU = os.path.join(HERE, "emu")
CSRC = os.path.join(os.path.dirname(HERE), "paper_2606_00746_b200", "csrc")
LIB = os.path.join(EMU, "libnaive_emu.so")
SHARED_BITS = {"w3": 1, "lam": 2, "u": 4}


@pytest.fixture(scope="module")
def emu():
    srcs = [os.path.join(EMU, "naive_emu.cpp"), os.path.join(EMU, "shim", "cuda_runtime.h"), os.path.join(EMU, "shim", "cuda_bf16.h"), os.path.join(EMU, "emu_rt.h"),
            os.path.join(CSRC, "gspn_naive.cuh"), os.path.join(CSRC, "gspn_common.cuh")]
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(s) for s in srcs):
        cmd = ["g++", "-std=c++20", "-O1", "-pthread", "-fPIC", "-shared", "-ffp-contract=off", "-I", EMU, "-I", os.path.join(EMU, "shim"),
               "-I", CSRC, "-o", LIB + ".tmp", srcs[0]]
        subprocess.run(cmd, check=True)
        os.replace(LIB + ".tmp", LIB)
    L = ctypes.CDLL(LIB)
    vp, ci, cu = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint
    L.emu_naive_fwd.argtypes = [vp] * 6 + [ci] * 5 + [cu, cu, ci, cu, ci, vp]
    L.emu_naive_bwd.argtypes = [vp] * 11 + [ci] * 5 + [cu, cu, ci, cu, ci, vp]
    return L


def to_dev(t: torch.Tensor) -> np.ndarray:
    """Storage bytes of a tensor as the kernels see them (bf16 as uint16)."""
    t = t.contiguous()
    return t.view(torch.int16).numpy().view(np.uint16).copy() if t.dtype == torch.bfloat16 else t.numpy().copy()


def from_dev(a: np.ndarray, dtype: str) -> np.ndarray:
    if dtype == "bf16":
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


def ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def scratch(cfg, planes_per_cta, ctas):
    """The large-plane mode's global scratch (csrc/gspn_naive.cu naive_workspace_bytes), NaN-filled; None = shared memory."""
    return np.full(ctas * planes_per_cta * cfg.H * cfg.W, np.nan, dtype=np.float32)


def run_fwd(L, cfg, dtype, t, shared=(), k_chunk=0, flags=0, ws=False):
    d = {k: to_dev(v[0] if k in shared else v) for k, v in t.items()}
    y = np.full_like(d["x"], 0x7fc1 if dtype == "bf16" else np.nan)
    w = scratch(cfg, 1, cfg.B * cfg.C) if ws else None
    rc = L.emu_naive_fwd(ptr(d["x"]), ptr(d["w3"]), ptr(d["lam"]), ptr(d["u"]), ptr(d.get("h0")), ptr(y), cfg.B, cfg.C, cfg.H,
                         cfg.W, cfg.G, cfg.dir_mask, sum(SHARED_BITS[k] for k in shared), k_chunk, flags, 0 if dtype == "f32" else 1, ptr(w))
    assert rc == 0
    return from_dev(y, dtype)


def run_bwd(L, cfg, dtype, t, shared=(), k_chunk=0, need=("dx", "dlambda", "du", "dw3", "dh0"), flags=0, ws=False):
    d = {k: to_dev(v[0] if k in shared else v) for k, v in t.items()}
    full = {k: to_dev(v) for k, v in t.items()}
    st = full["x"].dtype
    fill = 0x7fc1 if dtype == "bf16" else np.nan
    shapes = {"dx": full["x"].shape, "dlambda": full["lam"].shape, "du": full["u"].shape, "dw3": full["w3"].shape,
              "dh0": (cfg.D, cfg.B, cfg.C, max(cfg.H, cfg.W))}
    out = {k: np.full(shapes[k], fill, dtype=st) for k in need}
    g = lambda k: ptr(out.get(k))
    w = scratch(cfg, 4, max(cfg.B * cfg.C, cfg.D * cfg.B * cfg.G)) if ws else None      # one buffer for both launches, as the launcher
    rc = L.emu_naive_bwd(ptr(d["x"]), ptr(d["w3"]), ptr(d["lam"]), ptr(d["u"]), ptr(d.get("h0")), ptr(d["dy"]), g("dx"), g("dlambda"),
                         g("du"), g("dw3"), g("dh0"), cfg.B, cfg.C, cfg.H, cfg.W, cfg.G, cfg.dir_mask,
                         sum(SHARED_BITS[k] for k in shared), k_chunk, flags, 0 if dtype == "f32" else 1, ptr(w))
    assert rc == 0
    return {k: from_dev(v, dtype) for k, v in out.items()}


CASES = [((2, 4, 8, 8, 2), 15), ((1, 4, 13, 17, 2), 15), ((1, 2, 33, 9, 1), 6), ((2, 2, 5, 40, 2), 9), ((1, 1, 1, 6, 1), 15),
         ((1, 2, 7, 1, 1), 15)]


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape,mask", CASES, ids=["x".join(map(str, s)) + f"-m{m}" for s, m in CASES])
def test_naive_kernels_emulated_match_the_oracle(emu, shape, mask, dtype):
    """The plain operator (what round 1 measured on hardware): forward and every gradient, with h0."""
    cfg = gi.small_config("emu", *shape, dir_mask=mask, seed=123, backward=True)
    t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
    yo, A = pu.oracle_fwd(t, cfg)
    r = pu.gate(run_fwd(emu, cfg, dtype, t), yo, A, dtype)
    assert r["ok"], r
    go, Ag = pu.oracle_bwd(t, cfg)
    g = run_bwd(emu, cfg, dtype, t)
    for k in go:
        r = pu.gate(g[k], go[k], Ag[k], dtype)
        assert r["ok"], (k, r)


SHARED_SETS = [("w3",), ("lam", "u"), ("w3", "lam", "u")]


@pytest.mark.parametrize("dtype", ["f32", pytest.param("bf16", marks=heavy)])
@pytest.mark.parametrize("shared", SHARED_SETS, ids=["+".join(s) for s in SHARED_SETS])
def test_shared_direction_slabs_emulated(emu, shared, dtype):
    """dir_stride_* = 0: one slab read by every direction == the dense operator on the slab replicated D times."""
    for shape, mask in [((2, 4, 9, 11, 2), 15), ((1, 2, 12, 7, 1), 6), ((1, 2, 6, 14, 2), 9)]:
        cfg = gi.small_config("emus", *shape, dir_mask=mask, seed=124, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
        rep = dict(t)
        for k in shared:
            rep[k] = t[k][:1].expand(cfg.D, *t[k].shape[1:]).contiguous()
        yo, A = pu.oracle_fwd(rep, cfg)
        y = run_fwd(emu, cfg, dtype, t, shared=shared)
        r = pu.gate(y, yo, A, dtype)
        assert r["ok"], (shape, mask, r)
        np.testing.assert_array_equal(y, run_fwd(emu, cfg, dtype, rep))          # same kernel, same arithmetic
        go, Ag = pu.oracle_bwd(rep, cfg)
        g = run_bwd(emu, cfg, dtype, t, shared=shared)
        gd = run_bwd(emu, cfg, dtype, rep)
        for k in go:
            r = pu.gate(g[k], go[k], Ag[k], dtype)
            assert r["ok"], (shape, mask, k, r)
            np.testing.assert_array_equal(g[k], gd[k], err_msg=k)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("k_chunk", [pytest.param(2, marks=heavy), 3, pytest.param(7, marks=heavy)])
def test_chunked_scan_emulated(emu, k_chunk, dtype):
    """k_chunk > 1 against oracle fwd_chunked / bwd_chunked, with h0, ragged bands and direction subsets."""
    for shape, mask in [((2, 4, 8, 8, 2), 15), ((1, 2, 13, 17, 1), 15), ((1, 2, 10, 9, 2), 6), ((1, 2, 11, 20, 1), 9)]:
        cfg = gi.small_config("emuc", *shape, dir_mask=mask, seed=125, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
        n = {k: pu.np64(v) for k, v in t.items()}
        yo = orc.fwd_chunked(n["x"], n["w3"], n["lam"], n["u"], cfg.G, mask, k_chunk, h0=n["h0"])
        A = orc.fwd_chunked_magnitude(n["x"], n["w3"], n["lam"], n["u"], cfg.G, mask, k_chunk, h0=n["h0"])
        y = run_fwd(emu, cfg, dtype, t, k_chunk=k_chunk)
        r = pu.gate(y, yo, A, dtype)
        assert r["ok"], (shape, mask, r)
        go = orc.bwd_chunked(n["x"], n["w3"], n["lam"], n["u"], n["dy"], cfg.G, mask, k_chunk, h0=n["h0"])
        Ag = orc.bwd_chunked_magnitude(n["x"], n["w3"], n["lam"], n["u"], n["dy"], cfg.G, mask, k_chunk, h0=n["h0"])
        g = run_bwd(emu, cfg, dtype, t, k_chunk=k_chunk)
        for k in go:
            r = pu.gate(g[k], go[k], Ag[k], dtype)
            assert r["ok"], (shape, mask, k, r)
        np.testing.assert_array_equal(run_fwd(emu, cfg, dtype, t, k_chunk=1), run_fwd(emu, cfg, dtype, t))


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_logits_in_the_load_path_emulated(emu, dtype):
    """GSPN_FLAG_W3_LOGITS: Eq. 3 where the taps are loaded, its adjoint where dw3 leaves; against the composition of the
    oracle's normalize / fwd / bwd / normalize_bwd.  Also with one shared logit slab and with k_chunk (flags compose)."""
    for shape, mask in [((2, 4, 8, 8, 2), 15), ((1, 2, 13, 17, 1), 15), ((1, 4, 10, 9, 2), 6), ((1, 2, 1, 12, 1), 15)]:
        cfg = gi.small_config("emul", *shape, dir_mask=mask, seed=127, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
        wt = gi.make_logits(cfg, dtype)["wt"]
        tl = dict(t, w3=wt)
        yo, A, go, Ag = pu.oracle_logits(t, wt, cfg)
        r = pu.gate(run_fwd(emu, cfg, dtype, tl, flags=1), yo, A, dtype)
        assert r["ok"], (shape, mask, r)
        g = run_bwd(emu, cfg, dtype, tl, flags=1)
        for k in go:
            r = pu.gate(g[k], go[k], Ag[k], dtype)
            assert r["ok"], (shape, mask, k, r)
    # one shared logit slab: the same slab normalised per direction (the in-grid taps differ between the axes)
    cfg = gi.small_config("emul2", 1, 4, 9, 11, 2, dir_mask=15, seed=128, backward=True)
    t = gi.make_inputs(cfg, "f32", device="cpu", with_dy=True)
    wt = gi.make_logits(cfg, "f32")["wt"]
    rep = wt[:1].expand(cfg.D, *wt.shape[1:]).contiguous()
    yo, A, go, Ag = pu.oracle_logits(t, rep, cfg)
    tl = dict(t, w3=wt)
    assert pu.gate(run_fwd(emu, cfg, "f32", tl, shared=("w3",), flags=1), yo, A, "f32")["ok"]
    g = run_bwd(emu, cfg, "f32", tl, shared=("w3",), flags=1)
    for k in go:
        assert pu.gate(g[k], go[k], Ag[k], "f32")["ok"], k
    # with bands: Eq. 3 then the chunked scan
    n = {k: pu.np64(v) for k, v in t.items()}
    w3 = orc.normalize(pu.np64(wt), 15)
    yo = orc.fwd_chunked(n["x"], w3, n["lam"], n["u"], cfg.G, 15, 3)
    A = orc.fwd_chunked_magnitude(n["x"], w3, n["lam"], n["u"], cfg.G, 15, 3)
    assert pu.gate(run_fwd(emu, cfg, "f32", tl, k_chunk=3, flags=1), yo, A, "f32")["ok"]


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_large_plane_mode_emulated(emu, dtype):
    """SURVEY 8(f) f2, first step: the plane-sized fp32 arrays (y; h, dx; h, dw3) in a global workspace instead of shared
    memory -- what the launchers switch to when a plane exceeds shared memory.  Forced here at small sizes (NaN-filled
    scratch): same bits as the shared-memory mode, and the oracle's values."""
    for shape, mask in [((2, 4, 9, 11, 2), 15), ((1, 2, 40, 7, 1), 6), ((1, 2, 6, 33, 2), 9)]:
        cfg = gi.small_config("emuw", *shape, dir_mask=mask, seed=129, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
        yo, A = pu.oracle_fwd(t, cfg)
        y = run_fwd(emu, cfg, dtype, t, ws=True)
        assert pu.gate(y, yo, A, dtype)["ok"], (shape, mask)
        np.testing.assert_array_equal(y, run_fwd(emu, cfg, dtype, t))
        go, Ag = pu.oracle_bwd(t, cfg)
        g, g0 = run_bwd(emu, cfg, dtype, t, ws=True), run_bwd(emu, cfg, dtype, t)
        for k in go:
            assert pu.gate(g[k], go[k], Ag[k], dtype)["ok"], (shape, mask, k)
            np.testing.assert_array_equal(g[k], g0[k], err_msg=k)


def test_optional_outputs_emulated(emu):
    cfg = gi.small_config("emuo", 1, 4, 9, 10, 2, seed=126, backward=True)
    t = gi.make_inputs(cfg, "f32", device="cpu", with_dy=True)
    full = run_bwd(emu, cfg, "f32", t)
    for need in (("dx",), ("dw3",), ("du", "dh0"), ("dlambda", "dw3")):
        part = run_bwd(emu, cfg, "f32", t, need=need)
        for k in need:
            np.testing.assert_array_equal(part[k], full[k])
