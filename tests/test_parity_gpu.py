"""GPU parity: libgspn (through the C ABI) against the fp64 CPU oracle on the same seeded inputs.

Small cases are compared element by element over whole tensors; BASELINE.json's full-size configs
are launched exactly as bench.py launches them and compared on sampled images (every (b,group)
unit is independent, so the oracle recomputes whole images).  Gates are in tests/parity_util.py.
"""
import os

import numpy as np
import pytest
import torch

import gspn_inputs as gi
import paper_2606_00746_b200 as gspn
import parity_util as pu

pytestmark = pytest.mark.gpu

IMPLS = [gspn.IMPL_NAIVE, gspn.IMPL_AUTO]
IMPL_IDS = ["naive", "auto"]
FWD_IMPLS = [gspn.IMPL_NAIVE, gspn.IMPL_AUTO, gspn.IMPL_FLAT, gspn.IMPL_CHAIN, gspn.IMPL_PLANE, gspn.IMPL_LINE]
FWD_IMPL_IDS = ["naive", "auto", "flat", "chain", "plane", "line"]

# (B, C, H, W, G): degenerate lines, W in {1,2,3}, H != W, beyond one warp, ragged tails, cg in {1,C}
SMALL_SHAPES = [
    (1, 1, 1, 1, 1), (1, 2, 1, 5, 1), (1, 2, 5, 1, 2), (2, 4, 4, 2, 2), (1, 3, 3, 3, 1),
    (2, 4, 5, 7, 2), (2, 4, 7, 5, 4), (1, 8, 16, 16, 8), (1, 4, 33, 35, 1), (2, 6, 40, 24, 3),
    (1, 4, 27, 27, 1), (1, 2, 73, 73, 2), (1, 8, 56, 56, 1), (1, 2, 128, 128, 1), (1, 2, 64, 130, 2),
    (1, 2, 100, 36, 1), (2, 8, 24, 40, 2), (1, 4, 8, 128, 1), (1, 4, 128, 8, 2), (2, 4, 12, 16, 4), (1, 4, 20, 12, 2),
    (1, 8, 60, 56, 1), (1, 4, 4, 4, 4), (1, 8, 128, 120, 2),
]


def _ids(shapes):
    return ["x".join(map(str, s)) for s in shapes]


def _unsupported_is_none(impl, fn):
    """As _fwd_or_skip inside a loop over shapes: None for a shape the forced kernel does not hold."""
    try:
        return fn()
    except gspn.GspnError as ex:
        if impl in (gspn.IMPL_PAIR, gspn.IMPL_PLANE, gspn.IMPL_LINE) and ex.status == 2:
            return None
        raise


def _fwd_or_skip(impl, fn):
    """The pair / plane kernels keep whole fp32 planes on chip: shapes they report as unsupported are skipped."""
    try:
        return fn()
    except gspn.GspnError as ex:
        if impl in (gspn.IMPL_PAIR, gspn.IMPL_PLANE, gspn.IMPL_LINE) and ex.status == 2:          # GSPN_EUNSUPPORTED
            pytest.skip(str(ex))
        raise


@pytest.mark.parametrize("impl", FWD_IMPLS, ids=FWD_IMPL_IDS)
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", SMALL_SHAPES, ids=_ids(SMALL_SHAPES))
def test_fwd_small_shapes(shape, dtype, impl):
    cfg = gi.small_config("s", *shape, seed=11)
    if impl in (gspn.IMPL_CHAIN, gspn.IMPL_PAIR, gspn.IMPL_PLANE) and max(shape[2], shape[3]) > 128:
        pytest.skip("chain kernels hold lines of at most 128 positions")
    r = _fwd_or_skip(impl, lambda: pu.check_fwd(cfg, dtype, impl=impl))
    assert r["ok"], r


@pytest.mark.parametrize("impl", FWD_IMPLS, ids=FWD_IMPL_IDS)
@pytest.mark.parametrize("mask", [1, 2, 4, 8, 3, 12, 5, 10, 7, 14])
def test_fwd_direction_masks(mask, impl):
    ran = 0
    for shape in [(2, 4, 9, 12, 2), (2, 4, 8, 16, 2), (1, 2, 40, 64, 1)]:
        for dtype in ("f32", "bf16"):
            cfg = gi.small_config("m", *shape, dir_mask=mask, seed=5 + mask)
            r = _unsupported_is_none(impl, lambda: pu.check_fwd(cfg, dtype, impl=impl))
            if r is not None:
                ran += 1
                assert r["ok"], (shape, dtype, r)
    assert ran >= 2


@pytest.mark.parametrize("impl", FWD_IMPLS, ids=FWD_IMPL_IDS)
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_fwd_with_initial_state(dtype, impl):
    ran = 0
    for shape in [(2, 4, 6, 9, 2), (1, 2, 20, 40, 1), (2, 4, 16, 8, 2), (1, 4, 128, 64, 4)]:
        cfg = gi.small_config("h0", *shape, seed=21)
        r = _unsupported_is_none(impl, lambda: pu.check_fwd(cfg, dtype, impl=impl, with_h0=True))
        if r is not None:
            ran += 1
            assert r["ok"], (shape, r)
    assert ran >= 2


@pytest.mark.parametrize("impl", FWD_IMPLS, ids=FWD_IMPL_IDS)
def test_cfg1_tiny_forward(impl):
    """BASELINE.json config 1: B=1, C=8, H=W=16, G=8, fp32, T->B, seed 0."""
    cfg = gi.CONFIGS["cfg1_tiny"]
    r = pu.check_fwd(cfg, "f32", impl=impl)
    assert r["ok"], r
    # fp32 on the tiny grid also meets BASELINE.json's literal wording on |y| above the floor
    assert r["max_err_over_A"] <= 1e-6


BWD_SHAPES = [
    (1, 1, 1, 1, 1), (1, 2, 1, 5, 1), (1, 2, 5, 1, 2), (1, 4, 8, 8, 2), (2, 4, 5, 7, 2),
    (2, 4, 7, 5, 4), (1, 4, 33, 35, 1), (1, 4, 27, 27, 2), (1, 4, 73, 73, 1), (1, 8, 56, 56, 1),
    (1, 2, 64, 40, 2),
]


@pytest.mark.parametrize("impl", IMPLS, ids=IMPL_IDS)
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", BWD_SHAPES, ids=_ids(BWD_SHAPES))
def test_bwd_small_shapes(shape, dtype, impl):
    cfg = gi.small_config("b", *shape, seed=13, backward=True)
    r = pu.check_bwd(cfg, dtype, impl=impl)
    assert r["ok"], r


@pytest.mark.parametrize("impl", IMPLS, ids=IMPL_IDS)
@pytest.mark.parametrize("mask", [1, 2, 4, 8, 6, 9, 13])
def test_bwd_direction_masks_and_h0(mask, impl):
    cfg = gi.small_config("bm", 2, 4, 9, 12, 2, dir_mask=mask, seed=40 + mask, backward=True)
    for dtype in ("f32", "bf16"):
        r = pu.check_bwd(cfg, dtype, impl=impl, with_h0=True)
        assert r["ok"], (dtype, r)


def _chain_or_skip(fn):
    """Run a check with the chain kernels forced; shapes they do not hold on chip are skipped."""
    try:
        return fn()
    except gspn.GspnError as ex:
        if ex.status == 2:          # GSPN_EUNSUPPORTED
            pytest.skip(str(ex))
        raise


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", BWD_SHAPES + [(1, 8, 73, 73, 2), (1, 2, 128, 128, 2), (1, 2, 100, 36, 1)],
                         ids=_ids(BWD_SHAPES + [(1, 8, 73, 73, 2), (1, 2, 128, 128, 2), (1, 2, 100, 36, 1)]))
def test_bwd_chain_small_shapes(shape, dtype):
    cfg = gi.small_config("bc", *shape, seed=17, backward=True)
    r = _chain_or_skip(lambda: pu.check_bwd(cfg, dtype, impl=gspn.IMPL_CHAIN))
    assert r["ok"] and r["variant"] == "chain_bwd", r


@pytest.mark.parametrize("mask", [1, 2, 4, 8, 3, 12, 6, 9, 13, 15])
def test_bwd_chain_direction_masks_and_h0(mask):
    cfg = gi.small_config("bcm", 2, 4, 9, 12, 2, dir_mask=mask, seed=60 + mask, backward=True)
    for dtype in ("f32", "bf16"):
        r = _chain_or_skip(lambda: pu.check_bwd(cfg, dtype, impl=gspn.IMPL_CHAIN, with_h0=True))
        assert r["ok"], (dtype, r)
    cfg = gi.small_config("bcm2", 1, 8, 37, 41, 2, dir_mask=mask, seed=80 + mask, backward=True)
    r = _chain_or_skip(lambda: pu.check_bwd(cfg, "bf16", impl=gspn.IMPL_CHAIN, with_h0=True))
    assert r["ok"], r


PLANE_BWD_SHAPES = [(1, 1, 1, 1, 1), (1, 2, 1, 5, 1), (1, 2, 5, 1, 2), (1, 4, 8, 8, 2), (2, 4, 5, 7, 2), (2, 4, 7, 5, 4),
                    (1, 4, 27, 27, 1), (2, 8, 27, 27, 2), (1, 4, 32, 32, 2), (1, 2, 20, 31, 1), (1, 8, 16, 16, 8)]


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", PLANE_BWD_SHAPES, ids=_ids(PLANE_BWD_SHAPES))
def test_bwd_plane_small_shapes(shape, dtype):
    """Whole-plane backward kernel forced: lines of at most one warp, 1 / 2 / 4 channels per group, h0."""
    cfg = gi.small_config("pb", *shape, seed=23, backward=True)
    r = _chain_or_skip(lambda: pu.check_bwd(cfg, dtype, impl=gspn.IMPL_PLANE, with_h0=True))
    assert r["ok"], r
    assert r["variant"] == "plane_bwd"


@pytest.mark.parametrize("mask", [1, 2, 4, 8, 3, 12, 6, 9, 13, 15])
def test_bwd_plane_direction_masks(mask):
    cfg = gi.small_config("pbm", 2, 8, 11, 14, 2, dir_mask=mask, seed=70 + mask, backward=True)
    for dtype in ("f32", "bf16"):
        r = pu.check_bwd(cfg, dtype, impl=gspn.IMPL_PLANE, with_h0=(mask % 2 == 1))
        assert r["ok"], (dtype, r)


LINE_BWD_SHAPES = [
    (1, 4, 8, 8, 1), (2, 4, 16, 16, 2), (1, 8, 56, 56, 1), (1, 8, 40, 64, 2), (1, 4, 128, 128, 1), (2, 8, 128, 128, 2),
    (1, 2, 128, 8, 1), (1, 4, 8, 128, 4), (1, 4, 24, 40, 2), (1, 8, 60, 56, 1), (1, 4, 36, 100, 1), (1, 8, 128, 120, 2),
    (1, 2, 4, 4, 2), (1, 4, 20, 12, 2),
]


# The line backward was written after GPU access for this repository had been closed (round 2): it compiles for
# sm_100a but has never run.  Its tests are opt-in so that an unverified kernel cannot take the CUDA context of the
# whole suite down with it: GSPN_TEST_LINE_BWD=1 python -m pytest tests -m gpu -k bwd_line
_line_bwd = pytest.mark.skipif(os.environ.get("GSPN_TEST_LINE_BWD", "0") != "1",
                               reason="line_bwd has not been run on hardware yet (set GSPN_TEST_LINE_BWD=1)")


@_line_bwd
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", LINE_BWD_SHAPES, ids=_ids(LINE_BWD_SHAPES))
def test_bwd_line_small_shapes(shape, dtype):
    """The line backward (16-byte-aligned rows, dx in tensor memory, C/G in {1, 2, 4, 8})."""
    cfg = gi.small_config("lb", *shape, seed=31, backward=True)
    r = _unsupported_is_none(gspn.IMPL_LINE, lambda: pu.check_bwd(cfg, dtype, impl=gspn.IMPL_LINE, with_h0=True))
    if r is None:
        pytest.skip("shape not held by the line backward in this storage type")
    assert r["ok"] and r["variant"] == "line_bwd", r


@_line_bwd
@pytest.mark.parametrize("mask", [1, 2, 4, 8, 3, 12, 6, 9, 13, 15])
def test_bwd_line_direction_masks(mask):
    for shape in [(2, 4, 8, 16, 2), (1, 8, 40, 64, 1)]:
        for dtype in ("f32", "bf16"):
            cfg = gi.small_config("lbm", *shape, dir_mask=mask, seed=40 + mask, backward=True)
            r = _unsupported_is_none(gspn.IMPL_LINE, lambda: pu.check_bwd(cfg, dtype, impl=gspn.IMPL_LINE, with_h0=(mask % 2 == 1)))
            if r is not None:
                assert r["ok"] and r["variant"] == "line_bwd", (shape, dtype, r)


def test_bwd_optional_outputs():
    cfg = gi.small_config("opt", 1, 4, 8, 8, 2, seed=3, backward=True)
    t = {k: v.cuda() for k, v in gi.make_inputs(cfg, "f32").items()}
    full = gspn.gspn_scan_bwd(t["x"], t["w3"], t["lam"], t["u"], t["dy"], cfg.G, cfg.dir_mask)
    for need in (("dx",), ("dw3",), ("du", "dh0"), ("dlambda", "dw3")):
        part = gspn.gspn_scan_bwd(t["x"], t["w3"], t["lam"], t["u"], t["dy"], cfg.G, cfg.dir_mask, need=need)
        assert set(part) == set(need)
        for k in need:
            assert torch.equal(part[k], full[k]), k


def test_fd_slice_of_cfg5():
    """BASELINE.json config 5: gradients against central finite differences of the GPU forward
    itself on a B=1, C=4, H=W=8 slice (fp32 storage, so the differences resolve)."""
    cfg = gi.small_config("fd", 1, 4, 8, 8, 1, seed=4, backward=True)
    t = gi.make_inputs(cfg, "f32")
    d = {k: v.cuda() for k, v in t.items()}
    g = gspn.gspn_scan_bwd(d["x"], d["w3"], d["lam"], d["u"], d["dy"], cfg.G, cfg.dir_mask)
    rng = np.random.default_rng(0)
    eps = 1e-2      # the scan is linear in each operand taken alone: central differences are exact up to rounding
    for name, key in (("dx", "x"), ("dlambda", "lam"), ("du", "u"), ("dw3", "w3")):
        base = d[key]
        for idx in rng.choice(base.numel(), size=12, replace=False):
            vals = []
            for sgn in (+1, -1):
                pert = base.clone()
                pert.view(-1)[idx] += sgn * eps
                args = dict(d)
                args[key] = pert
                y = gspn.gspn_scan_fwd(args["x"], args["w3"], args["lam"], args["u"], cfg.G, cfg.dir_mask)
                vals.append(float((y.double() * d["dy"].double()).sum()))
            fd = (vals[0] - vals[1]) / (2 * eps)
            got = float(g[name].view(-1)[idx])
            assert got == pytest.approx(fd, rel=2e-3, abs=2e-3), (name, idx)


def test_merge_parity():
    rng = torch.Generator().manual_seed(7)
    for dtype, st in (("f32", torch.float32), ("bf16", torch.bfloat16)):
        for shape, mask in (((4, 2, 6, 8, 8), 15), ((3, 1, 5, 7, 9), 7), ((2, 2, 3, 27, 27), 6), ((1, 1, 1, 1, 1), 8)):
            D, B, C, H, W = shape
            yd = torch.randn(shape, generator=rng).to(st)
            m = torch.randn((D, C), generator=rng)
            from oracle import gspn_oracle as orc
            for mm in (None, m):
                got = gspn.gspn_merge(yd.cuda(), None if mm is None else mm.cuda(), dir_mask=mask)
                ref = orc.merge(pu.np64(yd), None if mm is None else pu.np64(mm))
                A = orc.merge(np.abs(pu.np64(yd)), None if mm is None else np.abs(pu.np64(mm)))
                r = pu.gate(pu.np64(got), ref, A, dtype)
                assert r["ok"], (shape, dtype, r)


FULL = [("cfg2_cls56", "f32"), ("cfg2_cls56", "bf16"), ("cfg3_enc378", "bf16"), ("cfg4_2k", "bf16"),
        ("cfg5_1k", "bf16")]


@pytest.mark.parametrize("name,dtype", FULL, ids=[f"{n}-{d}" for n, d in FULL])
def test_fwd_full_size_configs(name, dtype):
    """BASELINE.json configs 2-5 at full size, launched as bench.py launches them."""
    cfg = gi.CONFIGS[name]
    t = gi.make_inputs(cfg, dtype, device="cuda:0", with_dy=False)
    y = gspn.gspn_scan_fwd(t["x"], t["w3"], t["lam"], t["u"], cfg.G, cfg.dir_mask)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(y.float()).all())
    r = pu.check_fwd_sampled(cfg, dtype, t, y)
    assert r["ok"], r


def test_bwd_full_size_cfg5():
    """BASELINE.json config 5 (1K forward + backward, bf16) at full size, sampled images."""
    cfg = gi.CONFIGS["cfg5_1k"]
    t = gi.make_inputs(cfg, "bf16", device="cuda:0", with_dy=True)
    g = gspn.gspn_scan_bwd(t["x"], t["w3"], t["lam"], t["u"], t["dy"], cfg.G, cfg.dir_mask)
    torch.cuda.synchronize()
    for k, v in g.items():
        assert bool(torch.isfinite(v.float()).all()), k
    r = pu.check_bwd_sampled(cfg, "bf16", t, g)
    assert r["ok"], r


def test_stability_property_at_full_size():
    """Property that holds at any size: with row-stochastic non-negative taps,
    lambda = u = 1 and x = 1 every direction's h equals the step count + 1, so
    y[i,j] = (i+1) + (H-i) + (j+1) + (W-j) = H + W + 2 (up to bf16 tap rounding, so fp32 here)."""
    B, C, H, W, G = 2, 8, 73, 73, 2
    cfg = gi.small_config("p", B, C, H, W, G, seed=77)
    t = gi.make_inputs(cfg, "f32", device="cuda:0")
    ones = torch.ones_like(t["lam"])
    y = gspn.gspn_scan_fwd(torch.ones_like(t["x"]), t["w3"], ones, ones, G, 15)
    assert torch.allclose(y, torch.full_like(y, H + W + 2), rtol=1e-5, atol=0)


def test_auto_selects_fused_kernels_where_supported():
    """GSPN_IMPL_AUTO must run the fused single-launch kernels on the benchmark shapes (no silent
    fallback to the naive path): 73x73 with 4 channels per group, forward and backward."""
    cfg = gi.small_config("sel", 1, 8, 73, 73, 2, seed=9, backward=True)
    r = pu.check_bwd(cfg, "bf16")
    assert r["ok"], r
    assert r["variant"] == "chain_bwd", r["variant"]
    assert gspn.gspn_last_launch_count() == 1
    r = pu.check_fwd(cfg, "bf16")
    assert r["ok"] and r["variant"] == "chain_fwd", r
    # 378-px kind of shape (27x27, rows not 16-byte aligned, lines of one warp): the whole-plane kernel
    cfg = gi.small_config("sel27", 2, 8, 27, 27, 2, seed=10, backward=True)
    r = pu.check_fwd(cfg, "bf16")
    assert r["ok"] and r["variant"] == "plane_fwd", r
    r = pu.check_bwd(cfg, "bf16")
    assert r["ok"] and r["variant"] == "plane_bwd", r
    assert gspn.gspn_last_launch_count() == 1


def test_chain_kernels_random_shapes():
    """Seeded sweep of the chain kernels and the whole-plane forward kernel (forced) over random shapes, masks, dtypes, group sizes and
    initial states: ragged tails, lines of 1..128 positions, 1/2/4 channels per group."""
    import random
    rnd = random.Random(2024)
    ran = 0
    for it in range(40):
        cg = rnd.choice([1, 2, 4]); G = rnd.choice([1, 2, 3]); C = cg * G; B = rnd.choice([1, 2])
        H = rnd.choice([1, 2, 3, 5, 13, 27, 32, 33, 40, 64, 65, 73, 97, 128])
        W = rnd.choice([1, 2, 3, 4, 7, 16, 27, 33, 35, 56, 65, 73, 96, 128])
        if rnd.random() < 0.6:
            H, W = min(H, 40), min(W, 40)
        mask = rnd.randint(1, 15); dt = rnd.choice(["f32", "bf16"]); h0 = rnd.random() < 0.4
        cfg = gi.small_config("rz", B, C, H, W, G, dir_mask=mask, seed=3000 + it, backward=True)
        for check, impl in ((pu.check_fwd, gspn.IMPL_CHAIN), (pu.check_bwd, gspn.IMPL_CHAIN), (pu.check_fwd, gspn.IMPL_PLANE)):
            try:
                r = check(cfg, dt, impl=impl, with_h0=h0)
            except gspn.GspnError as ex:
                if ex.status == 2:
                    continue
                raise
            ran += 1
            assert r["ok"], (check.__name__, impl, (B, C, H, W, G), mask, dt, h0, r)
    assert ran >= 70


# ---- Eq. (3) normalisation ------------------------------------------------------------
NORM_SHAPES = [(1, 1, 1, 1, 1), (1, 2, 1, 5, 2), (2, 2, 5, 1, 1), (2, 4, 5, 7, 2), (1, 8, 16, 16, 8), (2, 4, 27, 27, 2),
               (1, 4, 73, 73, 1), (2, 8, 56, 56, 4), (1, 2, 128, 128, 2), (1, 2, 64, 130, 1), (1, 3, 300, 37, 3)]


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", NORM_SHAPES, ids=_ids(NORM_SHAPES))
def test_normalize_small_shapes(shape, dtype):
    """gspn_normalize_fwd / _bwd against the fp64 oracle: vector path (16-byte-aligned planes) and scalar
    path (odd H*W in bf16), lines of one, ragged tails, every direction's edge mask."""
    cfg = gi.small_config("nz", *shape, seed=41)
    r = pu.check_norm(cfg, dtype)
    assert r["ok"], r


@pytest.mark.parametrize("mask", [1, 2, 4, 8, 5, 10, 14])
def test_normalize_direction_masks_and_sharp_logits(mask):
    """Each direction slab masks its own cross axis; logit std 6 drives sigmoids to both tails."""
    import dataclasses
    for dtype in ("f32", "bf16"):
        cfg = dataclasses.replace(gi.small_config("nm", 2, 4, 9, 12, 2, dir_mask=mask, seed=50 + mask), logit_std=6.0)
        r = pu.check_norm(cfg, dtype)
        assert r["ok"], (dtype, r)


def test_normalize_clamp_branch_on_gpu():
    """All logits near -40: S < GSPN_NORM_EPS, the clamp is active in forward and backward."""
    wt = torch.full((1, 1, 2, 3, 6, 8), -40.0, device="cuda:0") + 0.25 * torch.randn(
        (1, 1, 2, 3, 6, 8), generator=torch.Generator().manual_seed(3)).cuda()
    dw = torch.randn(wt.shape, generator=torch.Generator().manual_seed(4)).cuda()
    w3 = gspn.gspn_normalize_fwd(wt, 1)
    dwt = gspn.gspn_normalize_bwd(wt, dw, 1)
    ref = pu.orc.normalize(pu.np64(wt), 1)
    gref = pu.orc.normalize_bwd(pu.np64(wt), pu.np64(dw), 1)
    assert np.all(np.abs(pu.np64(w3) - ref) <= 1e-5 * np.abs(ref) + 1e-30)
    assert np.all(np.abs(pu.np64(dwt) - gref) <= 2e-5 * np.abs(gref) + 1e-30)


@pytest.mark.parametrize("name,dtype", [("cfg5_1k", "bf16"), ("cfg4_2k", "bf16"), ("cfg2_cls56", "f32")])
def test_normalize_full_size_configs(name, dtype):
    """The launch bench.py times (whole batch), checked on the first / middle / last images."""
    cfg = gi.CONFIGS[name]
    t = gi.make_logits(cfg, dtype, device="cuda:0", with_dw=True)
    w3 = gspn.gspn_normalize_fwd(t["wt"], cfg.dir_mask)
    dwt = gspn.gspn_normalize_bwd(t["wt"], t["dw3"], cfg.dir_mask)
    for b in (0, cfg.B // 2, cfg.B - 1):
        wt64, dw64 = pu.np64(t["wt"][:, b:b + 1]), pu.np64(t["dw3"][:, b:b + 1])
        ref = pu.orc.normalize(wt64, cfg.dir_mask)
        r = pu.gate(pu.np64(w3[:, b:b + 1]), ref, np.abs(ref), dtype)
        assert r["ok"], (b, r)
        gref = pu.orc.normalize_bwd(wt64, dw64, cfg.dir_mask)
        r = pu.gate(pu.np64(dwt[:, b:b + 1]), gref, pu.norm_bwd_magnitude(wt64, dw64, cfg.dir_mask), dtype)
        assert r["ok"], (b, r)
    # rows of the normalised taps sum to one up to the storage rounding: a property that holds at any size
    s = w3.float().sum(dim=3)
    assert float((s - 1).abs().max()) <= (1.2e-2 if dtype == "bf16" else 1e-5)
