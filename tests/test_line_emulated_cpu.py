"""The line kernels (csrc/gspn_line_fwd.cu, csrc/gspn_line_bwd.cu: kernel AND launcher, the files nvcc compiles) run on the
host under tests/emu and compared with the oracle -- on a machine without a GPU.

GPU access for this repository closed in round 2 before the line backward had ever run and after the last three edits
of the line forward.  tests/emu gives the kernels what they are written against: the PTX wrappers of gspn_fused.cuh /
gspn_line.cuh become host stand-ins (tests/emu/emu_ptx.h: mbarriers with transaction counts, TMA tensor loads and stores
with box clipping / zero fill / SWIZZLE_32B, tensor memory with the 32x32b lane-quarter rule, named barriers, the bf16
FMA), a thread block runs as host threads with real warp shuffles and barriers (tests/emu/emu_rt.h), and the launchers'
launch statement becomes emu::launch.  The stand-ins also check what the hardware would fault on (TMA destination
alignment, tensor-map rules, shared- and tensor-memory bounds, mbarrier over-arrival) and every wait has a time limit, so
a protocol error is a test failure with a message, not a hang.

What this establishes: index arithmetic, stage / ring / checkpoint bookkeeping, barrier counts and phases, tensor-memory
layouts and the launchers' shared-memory layout and tensor maps reproduce the oracle within the GPU tolerances.  What it
cannot: memory-ordering between the generic and the async proxy or around tcgen05 (the fences are no-ops here), performance.
Asynchronous copies are run at both extremes: at once (default: a refill destroys a stage that is still being read) and
as late as the program allows (lazy mode: a load lands when somebody waits on its mbarrier, a store reads shared memory
when its bulk group is waited for).  The GPU parity tests remain the parity evidence.
"""
import ctypes
import os
import subprocess

import numpy as np
import pytest
import torch

import gspn_inputs as gi
import parity_util as pu

HERE = os.path.dirname(os.path.abspath(__file__))
EMU = os.path.join(HERE, "emu")
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(ROOT, "paper_2606_00746_b200", "csrc")
LIB = os.path.join(EMU, "libline_emu.so")
UNITS = ["line_fwd_emu.cpp", "line_bwd_emu.cpp", "line_emu_support.cpp"]


@pytest.fixture(scope="module")
def emu():
    deps = [os.path.join(EMU, f) for f in UNITS + ["emu_rt.h", "emu_ptx.h", "shim/cuda_runtime.h", "shim/cuda_bf16.h", "shim/cuda.h"]]
    deps += [os.path.join(CSRC, f) for f in ("gspn_line_fwd.cu", "gspn_line_bwd.cu", "gspn_line.cuh", "gspn_fused.cuh", "gspn_common.cuh",
                                             "gspn_kernels.h")] + [os.path.join(ROOT, "include", "gspn.h")]
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(d) for d in deps):
        objs, procs = [], []
        for u in UNITS:
            obj = os.path.join(EMU, u.replace(".cpp", ".emu.o"))
            objs.append(obj)
            procs.append(subprocess.Popen(["g++", "-std=c++20", "-O1", "-pthread", "-fPIC", "-ffp-contract=off", "-w", "-I", EMU,
                                           "-I", os.path.join(EMU, "shim"), "-I", CSRC, "-c", os.path.join(EMU, u), "-o", obj]))
        assert all(p.wait() == 0 for p in procs), "tests/emu does not compile"
        subprocess.run(["g++", "-shared", "-pthread", "-o", LIB + ".tmp"] + objs, check=True)
        os.replace(LIB + ".tmp", LIB)
    L = ctypes.CDLL(LIB)
    vp, ci, cu = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint
    L.emu_line_fwd.argtypes = [vp] * 6 + [ci] * 5 + [cu, ci, ctypes.c_double]
    L.emu_line_bwd.argtypes = [vp] * 11 + [ci] * 5 + [cu, ci, ctypes.c_double]
    L.emu_last_error.restype = ctypes.c_char_p
    L.emu_set_jitter.argtypes = [ci, cu]
    L.emu_set_lazy.argtypes = [ci]
    return L


def to_dev(t: torch.Tensor) -> np.ndarray:
    t = t.contiguous()
    return t.view(torch.int16).numpy().view(np.uint16).copy() if t.dtype == torch.bfloat16 else t.numpy().copy()


def from_dev(a: np.ndarray, dtype: str) -> np.ndarray:
    return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64) if dtype == "bf16" else a.astype(np.float64)


def ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


LIMIT_S = 60.0          # a wait inside the emulated kernel longer than this is reported as a deadlock
# A block of 160-320 threads on a few host cores is slow (a warp shuffle is two 32-thread barriers): the default run keeps the
# cases that take seconds; GSPN_EMU_FULL=1 adds the full-size units (128x128 C/G=4, 56x56 C/G=8) and more timing-noise
# and late-copy cases (about ten minutes more; all of them passed when this file was committed).
FULL = os.environ.get("GSPN_EMU_FULL") == "1"
heavy = pytest.mark.skipif(not FULL, reason="set GSPN_EMU_FULL=1 for the full-size emulated cases")


def run_fwd(L, cfg, dtype, t):
    d = {k: to_dev(v) for k, v in t.items()}
    y = np.full_like(d["x"], 0x7fc1 if dtype == "bf16" else np.nan)
    rc = L.emu_line_fwd(ptr(d["x"]), ptr(d["w3"]), ptr(d["lam"]), ptr(d["u"]), ptr(d.get("h0")), ptr(y), cfg.B, cfg.C, cfg.H, cfg.W,
                        cfg.G, cfg.dir_mask, 0 if dtype == "f32" else 1, LIMIT_S)
    return rc, from_dev(y, dtype)


def run_bwd(L, cfg, dtype, t):
    d = {k: to_dev(v) for k, v in t.items()}
    st = d["x"].dtype
    fill = 0x7fc1 if dtype == "bf16" else np.nan
    shapes = {"dx": d["x"].shape, "dlambda": d["lam"].shape, "du": d["u"].shape, "dw3": d["w3"].shape,
              "dh0": (cfg.D, cfg.B, cfg.C, max(cfg.H, cfg.W))}
    out = {k: np.full(s, fill, dtype=st) for k, s in shapes.items()}
    rc = L.emu_line_bwd(ptr(d["x"]), ptr(d["w3"]), ptr(d["lam"]), ptr(d["u"]), ptr(d.get("h0")), ptr(d["dy"]), ptr(out["dx"]),
                        ptr(out["dlambda"]), ptr(out["du"]), ptr(out["dw3"]), ptr(out["dh0"]), cfg.B, cfg.C, cfg.H, cfg.W, cfg.G,
                        cfg.dir_mask, 0 if dtype == "f32" else 1, LIMIT_S)
    return rc, {k: from_dev(v, dtype) for k, v in out.items()}


# shape (B, C, H, W, G), dir_mask, dtype, h0 -- one, two and four positions per lane (lines up to 32 / 64 / 128), C/G in
# {1, 2, 4, 8}, ragged last stages (H, W not multiples of 8 rows / 16 columns), single-plane and multi-plane TMA boxes,
# direction subsets, the full 128x128 unit of the 2K config and the 56x56 C/G = 8 unit of the classification config
FWD_CASES = [((1, 4, 8, 8, 1), 15, "f32", False), ((1, 4, 16, 16, 2), 15, "bf16", True), ((2, 8, 24, 40, 2), 15, "bf16", False),
             ((1, 4, 56, 56, 1), 15, "f32", True), ((1, 2, 40, 24, 1), 15, "bf16", False), ((1, 4, 72, 64, 1), 15, "bf16", True),
             ((1, 8, 128, 128, 2), 15, "bf16", False), ((1, 4, 16, 16, 1), 6, "f32", False), ((1, 4, 32, 48, 2), 9, "bf16", True),
             ((1, 4, 40, 40, 1), 1, "f32", False), ((1, 4, 40, 40, 1), 8, "bf16", False), ((1, 4, 20, 28, 2), 15, "f32", True),
             ((1, 8, 56, 56, 1), 15, "bf16", False), ((1, 4, 60, 56, 1), 12, "bf16", False), ((1, 4, 4, 4, 4), 3, "f32", False)]


def _id(c):
    return "x".join(map(str, c[0])) + f"-m{c[1]}-{c[2]}" + ("-h0" if c[3] else "")


@pytest.mark.parametrize("case", [pytest.param(c, marks=heavy) if max(c[0][2], c[0][3]) > 64 else c for c in FWD_CASES], ids=[_id(c) for c in FWD_CASES])
def test_line_forward_emulated(emu, case):
    shape, mask, dtype, h0 = case
    cfg = gi.small_config("lfe", *shape, dir_mask=mask, seed=7)
    t = gi.make_inputs(cfg, dtype, device="cpu", with_h0=h0)
    rc, y = run_fwd(emu, cfg, dtype, t)
    if rc == 2:
        pytest.skip("shape not held by the line forward: " + emu.emu_last_error().decode())
    assert rc == 0, emu.emu_last_error().decode()
    yo, A = pu.oracle_fwd(t, cfg)
    r = pu.gate(y, yo, A, dtype)
    assert r["ok"], r


BWD_CASES = [((1, 4, 8, 8, 1), 15, "f32", False), ((2, 4, 16, 16, 2), 15, "bf16", True), ((2, 4, 16, 16, 2), 15, "f32", True),
             ((1, 8, 56, 56, 1), 15, "bf16", True), ((1, 8, 40, 64, 2), 15, "bf16", True), ((1, 4, 128, 128, 1), 15, "bf16", True),
             ((1, 2, 128, 8, 1), 15, "bf16", True), ((1, 4, 24, 40, 2), 15, "f32", True), ((1, 8, 60, 56, 1), 15, "bf16", False),
             ((1, 2, 4, 4, 2), 15, "f32", True), ((1, 4, 20, 12, 2), 15, "f32", True), ((1, 4, 32, 48, 2), 6, "bf16", True),
             ((1, 4, 40, 40, 1), 9, "f32", False), ((1, 2, 36, 24, 1), 4, "bf16", True), ((1, 2, 36, 24, 1), 2, "f32", True)]


HEAVY_BWD = {(1, 8, 56, 56, 1), (1, 8, 40, 64, 2), (1, 4, 128, 128, 1), (1, 8, 60, 56, 1), (1, 2, 128, 8, 1)}


@pytest.mark.parametrize("case", [pytest.param(c, marks=heavy) if c[0] in HEAVY_BWD else c for c in BWD_CASES], ids=[_id(c) for c in BWD_CASES])
def test_line_backward_emulated(emu, case):
    """The line backward has never run on a GPU; here every gradient of every case is gated against the oracle."""
    shape, mask, dtype, h0 = case
    cfg = gi.small_config("lbe", *shape, dir_mask=mask, seed=8, backward=True)
    t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=h0)
    rc, g = run_bwd(emu, cfg, dtype, t)
    if rc == 2:
        pytest.skip("shape not held by the line backward: " + emu.emu_last_error().decode())
    assert rc == 0, emu.emu_last_error().decode()
    go, Ag = pu.oracle_bwd(t, cfg)
    for k in go:
        r = pu.gate(g[k], go[k], Ag[k], dtype)
        assert r["ok"], (k, r)


@pytest.mark.parametrize("seed,shape", [(1, (1, 4, 16, 24, 2)), pytest.param(2, (2, 4, 24, 48, 2), marks=heavy),
                                        pytest.param(3, (2, 4, 24, 48, 2), marks=heavy)])
def test_line_kernels_emulated_under_timing_noise(emu, seed, shape):
    """Random sleeps at the synchronisation operations (another interleaving of producers and consumers per seed): same
    results, bit for bit, as without."""
    cfg = gi.small_config("lje", *shape, seed=9, backward=True)
    t = gi.make_inputs(cfg, "bf16", device="cpu", with_dy=True, with_h0=True)
    rc, y0 = run_fwd(emu, cfg, "bf16", t)
    assert rc == 0, emu.emu_last_error().decode()
    rc, g0 = run_bwd(emu, cfg, "bf16", t)
    assert rc == 0, emu.emu_last_error().decode()
    emu.emu_set_jitter(300, seed)
    try:
        rc, y1 = run_fwd(emu, cfg, "bf16", t)
        assert rc == 0, emu.emu_last_error().decode()
        rc, g1 = run_bwd(emu, cfg, "bf16", t)
        assert rc == 0, emu.emu_last_error().decode()
    finally:
        emu.emu_set_jitter(0, 1)
    np.testing.assert_array_equal(y1, y0)
    for k in g0:
        np.testing.assert_array_equal(g1[k], g0[k], err_msg=k)


LAZY_CASES = [("fwd", (1, 4, 32, 48, 2), 15, "bf16", True), ("bwd", (1, 4, 16, 16, 2), 15, "bf16", True),
              ("bwd", (1, 4, 24, 40, 2), 15, "f32", True), ("bwd", (1, 4, 128, 128, 1), 15, "bf16", True),
              ("fwd", (1, 8, 128, 128, 2), 15, "bf16", False)]


@pytest.mark.parametrize("case", [pytest.param(c, marks=heavy) if i >= 2 else c for i, c in enumerate(LAZY_CASES)],
                         ids=[c[0] + "-" + _id(c[1:]) for c in LAZY_CASES])
def test_line_kernels_emulated_with_copies_as_late_as_allowed(emu, case):
    """The other extreme of the asynchronous copies (tests/emu/emu_rt.h, lazy mode): a TMA load lands only when a thread waits
    on its mbarrier, a TMA store reads shared memory only when its thread waits for the bulk group.  A consumer that read
    a stage without waiting, or an output stage rewritten before its store was waited for, would miss parity here."""
    which, shape, mask, dtype, h0 = case
    cfg = gi.small_config("lze", *shape, dir_mask=mask, seed=10, backward=True)
    t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=h0)
    emu.emu_set_lazy(1)
    try:
        if which == "fwd":
            tf = {k: v for k, v in t.items() if k != "dy"}
            rc, y = run_fwd(emu, cfg, dtype, tf)
            assert rc == 0, emu.emu_last_error().decode()
            yo, A = pu.oracle_fwd(tf, cfg)
            assert pu.gate(y, yo, A, dtype)["ok"]
        else:
            rc, g = run_bwd(emu, cfg, dtype, t)
            assert rc == 0, emu.emu_last_error().decode()
            go, Ag = pu.oracle_bwd(t, cfg)
            for k in go:
                assert pu.gate(g[k], go[k], Ag[k], dtype)["ok"], k
    finally:
        emu.emu_set_lazy(0)


def _poison_taps(w3: torch.Tensor, cfg) -> torch.Tensor:
    """NaN in every tap whose neighbour lies outside the grid (include/gspn.h: such a tap is never used)."""
    w = w3.clone()
    for q, d in enumerate(gi.dir_list(cfg.dir_mask)):
        if d < 2:
            w[q, :, :, 0, :, 0] = float("nan"); w[q, :, :, 2, :, cfg.W - 1] = float("nan")
        else:
            w[q, :, :, 0, 0, :] = float("nan"); w[q, :, :, 2, cfg.H - 1, :] = float("nan")
    return w


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_line_kernels_never_use_out_of_grid_taps_emulated(emu, dtype):
    """DESIGN.md reading 3 for the line kernels: NaN stored in the out-of-grid taps changes no output bit, forward or
    backward (the dw3 entries of those taps are written 0 either way)."""
    for shape in [(1, 4, 16, 16, 2), (1, 2, 40, 24, 1)]:
        cfg = gi.small_config("lpe", *shape, seed=11, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True)
        bad = dict(t, w3=_poison_taps(t["w3"], cfg))
        tf, bf = ({k: v for k, v in d.items() if k != "dy"} for d in (t, bad))
        rc0, y0 = run_fwd(emu, cfg, dtype, tf)
        rc1, y1 = run_fwd(emu, cfg, dtype, bf)
        assert rc0 == 0 and rc1 == 0, emu.emu_last_error().decode()
        np.testing.assert_array_equal(y1, y0)
        rc0, g0 = run_bwd(emu, cfg, dtype, t)
        rc1, g1 = run_bwd(emu, cfg, dtype, bad)
        assert rc0 == 0 and rc1 == 0, emu.emu_last_error().decode()
        for k in g0:
            np.testing.assert_array_equal(g1[k], g0[k], err_msg=f"{shape} {k}")


def test_line_backward_optional_outputs_emulated(emu):
    """Any subset of the gradients may be left out (NULL pointers): the others keep their bits."""
    cfg = gi.small_config("loe", 1, 4, 24, 32, 2, seed=12, backward=True)
    t = gi.make_inputs(cfg, "bf16", device="cpu", with_dy=True, with_h0=True)
    d = {k: to_dev(v) for k, v in t.items()}
    shapes = {"dx": d["x"].shape, "dlambda": d["lam"].shape, "du": d["u"].shape, "dw3": d["w3"].shape,
              "dh0": (cfg.D, cfg.B, cfg.C, max(cfg.H, cfg.W))}

    def run(need):
        out = {k: np.full(shapes[k], 0x7fc1, dtype=np.uint16) for k in need}
        g = lambda k: ptr(out.get(k))
        rc = emu.emu_line_bwd(ptr(d["x"]), ptr(d["w3"]), ptr(d["lam"]), ptr(d["u"]), ptr(d["h0"]), ptr(d["dy"]), g("dx"), g("dlambda"),
                              g("du"), g("dw3"), g("dh0"), cfg.B, cfg.C, cfg.H, cfg.W, cfg.G, cfg.dir_mask, 1, LIMIT_S)
        assert rc == 0, emu.emu_last_error().decode()
        return out

    full = run(("dx", "dlambda", "du", "dw3", "dh0"))
    for need in (("dx",), ("dw3",), ("du", "dh0"), ("dlambda", "dw3"), ("dh0",), ("dx", "dlambda", "du")):
        part = run(need)
        for k in need:
            np.testing.assert_array_equal(part[k], full[k], err_msg=f"{need} {k}")
