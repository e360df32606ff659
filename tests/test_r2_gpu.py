"""Round-2 GPU parity additions ("Parity holes"): the host entry points, every image of the full-size
configs, the out-of-grid taps (reading 3), run-to-run bit identity, the backward of the aligned benchmark
shapes through GSPN_IMPL_AUTO with the variant reported, optional outputs per kernel.

Collected after test_parity_gpu.py on purpose: these cases were written while GPU access was closed for this
repository, so a failure here must not hide the results of the suite that had already run on hardware.
"""
import numpy as np
import pytest
import torch

import gspn_inputs as gi
import paper_2606_00746_b200 as gspn
import parity_util as pu

pytestmark = pytest.mark.gpu


def _try(fn):
    """None when the forced kernel reports the shape as unsupported."""
    try:
        return fn()
    except gspn.GspnError as ex:
        if ex.status == 2:
            return None
        raise


# ---------------------------------------------------------------------------------- host entry points (hole a)
@pytest.mark.parametrize("pinned", [True, False], ids=["pinned", "pageable"])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_host_entry_points_match_the_oracle(dtype, pinned):
    """gspn_scan_fwd_host / gspn_scan_bwd_host (the calls bench.py's e2e leg times) on an odd shape, every output
    gated against the oracle."""
    cfg = gi.small_config("host", 2, 4, 37, 41, 2, seed=51, backward=True)
    t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True)
    host = {k: (v.contiguous().pin_memory() if pinned else v.contiguous().clone()) for k, v in t.items()}
    L = max(cfg.H, cfg.W)
    st = host["x"].dtype
    mk = (lambda *s: torch.empty(*s, dtype=st).pin_memory()) if pinned else (lambda *s: torch.empty(*s, dtype=st))
    y = mk(*host["x"].shape)
    gspn.gspn_scan_fwd_host(host["x"], host["w3"], host["lam"], host["u"], y, cfg.G, cfg.dir_mask)
    yo, A = pu.oracle_fwd(t, cfg)
    r = pu.gate(pu.np64(y), yo, A, dtype)
    assert r["ok"], r
    outs = {"dx": mk(*host["x"].shape), "dlambda": mk(*host["lam"].shape), "du": mk(*host["u"].shape),
            "dw3": mk(*host["w3"].shape), "dh0": mk(cfg.D, cfg.B, cfg.C, L)}
    gspn.gspn_scan_bwd_host(host["x"], host["w3"], host["lam"], host["u"], host["dy"], outs["dx"], outs["dlambda"],
                            outs["du"], outs["dw3"], outs["dh0"], cfg.G, cfg.dir_mask)
    go, Ag = pu.oracle_bwd(t, cfg)
    for k in ("dx", "dlambda", "du", "dw3", "dh0"):
        r = pu.gate(pu.np64(outs[k]), go[k], Ag[k], dtype)
        assert r["ok"], (k, r)


# ---------------------------------------------------------------------------------- every image (hole b, c)
def _all_images_fwd(cfg, dtype, t, y, chunk):
    for b0 in range(0, cfg.B, chunk):
        b1 = min(cfg.B, b0 + chunk)
        sub = gi.with_batch(cfg, b1 - b0)
        yo, A = pu.oracle_fwd(pu._slice(t, b0, b1), sub)
        r = pu.gate(pu.np64(y[b0:b1]), yo, A, dtype)
        assert r["ok"], ((b0, b1), r)


def _all_images_bwd(cfg, dtype, t, g, chunk):
    for b0 in range(0, cfg.B, chunk):
        b1 = min(cfg.B, b0 + chunk)
        sub = gi.with_batch(cfg, b1 - b0)
        go, A = pu.oracle_bwd(pu._slice(t, b0, b1), sub)
        for k in ("dx", "dlambda", "du", "dw3", "dh0"):
            gk = g[k][b0:b1] if k == "dx" else g[k][:, b0:b1]
            r = pu.gate(pu.np64(gk), go[k], A[k], dtype)
            assert r["ok"], (k, (b0, b1), r)


@pytest.mark.parametrize("name,chunk", [("cfg5_1k", 4), ("cfg3_enc378", 32), ("cfg4_2k", 1)])
def test_every_image_of_the_full_size_forward(name, chunk):
    """Full size, launched as bench.py launches it, and EVERY image compared (a tail-wave or CTA-scheduling fault in
    an image the sampled check skips would pass there)."""
    cfg = gi.CONFIGS[name]
    t = gi.make_inputs(cfg, "bf16", device="cuda:0", with_dy=False)
    y = gspn.gspn_scan_fwd(t["x"], t["w3"], t["lam"], t["u"], cfg.G, cfg.dir_mask)
    torch.cuda.synchronize()
    _all_images_fwd(cfg, "bf16", t, y, chunk)


@pytest.mark.parametrize("name,chunk", [("cfg5_1k", 4), ("cfg3_enc378", 32)])
def test_every_image_of_the_full_size_backward(name, chunk):
    cfg = gi.CONFIGS[name]
    t = gi.make_inputs(cfg, "bf16", device="cuda:0", with_dy=True)
    g = gspn.gspn_scan_bwd(t["x"], t["w3"], t["lam"], t["u"], t["dy"], cfg.G, cfg.dir_mask)
    torch.cuda.synchronize()
    _all_images_bwd(cfg, "bf16", t, g, chunk)


# ---------------------------------------------------------------------------------- aligned benchmark shapes, backward (hole e)
@pytest.mark.parametrize("shape,dtype", [((1, 8, 128, 128, 2), "bf16"), ((2, 16, 56, 56, 2), "bf16"), ((1, 8, 56, 56, 1), "f32")],
                         ids=["128x128-cg4-bf16", "56x56-cg8-bf16", "56x56-cg8-f32"])
def test_auto_backward_on_the_aligned_benchmark_shapes(shape, dtype, record_property):
    """GSPN_IMPL_AUTO backward at the 2K shape (C/G = 4) and the classification shape (C/G = 8): parity, and the
    variant that ran is reported; a fall-through to the naive kernel is an expected failure, not a silent pass."""
    cfg = gi.small_config("ab", *shape, seed=61, backward=True)
    r = _try(lambda: pu.check_bwd(cfg, dtype))
    if r is None:
        record_property("variant", "none (GSPN_EUNSUPPORTED)")
        pytest.xfail("no backward kernel under GSPN_IMPL_AUTO holds this shape yet (naive_bwd needs 16*H*W bytes of shared "
                     "memory; line_bwd holds it but is opt-in until it has run on hardware)")
    assert r["ok"], r
    record_property("variant", r["variant"])
    if r["variant"].startswith("naive_bwd"):
        pytest.xfail("GSPN_IMPL_AUTO has no fused backward for this shape yet: it lands on " + r["variant"] +
                     " (line_bwd holds the shape but stays out of AUTO until it has run on hardware)")


# ---------------------------------------------------------------------------------- out-of-grid taps (hole f, reading 3)
def _poison(t, cfg):
    """NaN in every tap whose neighbour lies outside the grid (the generator stores 0 there)."""
    w = t["w3"].clone()
    for q, d in enumerate(gi.dir_list(cfg.dir_mask)):
        if d < 2:
            w[q, :, :, 0, :, 0] = float("nan")
            w[q, :, :, 2, :, cfg.W - 1] = float("nan")
        else:
            w[q, :, :, 0, 0, :] = float("nan")
            w[q, :, :, 2, cfg.H - 1, :] = float("nan")
    return w


STRICT = ("naive", "line")        # strict where the kernel has been read for it; the r1 kernels (also behind AUTO) report a leak as xfail


FWD_IMPLS = [("auto", gspn.IMPL_AUTO), ("naive", gspn.IMPL_NAIVE), ("tile", gspn.IMPL_FUSED), ("flat", gspn.IMPL_FLAT),
             ("chain", gspn.IMPL_CHAIN), ("plane", gspn.IMPL_PLANE), ("line", gspn.IMPL_LINE)]


@pytest.mark.parametrize("name,impl", FWD_IMPLS, ids=[n for n, _ in FWD_IMPLS])
def test_out_of_grid_taps_are_never_read_forward(name, impl):
    """include/gspn.h: the tap of a neighbour outside the grid is never used, so a NaN stored there cannot leak."""
    ran = 0
    for shape in [(1, 4, 16, 16, 2), (2, 4, 27, 27, 1), (1, 2, 40, 24, 1)]:
        for dtype in ("f32", "bf16"):
            cfg = gi.small_config("nan", *shape, seed=71)
            d = {k: v.cuda() for k, v in gi.make_inputs(cfg, dtype).items()}
            y0 = _try(lambda: gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, cfg.dir_mask, impl=impl))
            if y0 is None:
                continue
            y1 = gspn.gspn_scan_fwd(d["x"], _poison(d, cfg), d["lam"], d["u"], cfg.G, cfg.dir_mask, impl=impl)
            if not torch.equal(y0, y1) and name not in STRICT:
                pytest.xfail(f"{name}: a NaN in an out-of-grid tap reaches y at {shape} {dtype} (kernel not selected by AUTO here)")
            assert torch.equal(y0, y1), (shape, dtype)
            ran += 1
    assert ran >= 1


BWD_IMPLS = [("auto", gspn.IMPL_AUTO), ("naive", gspn.IMPL_NAIVE), ("group", gspn.IMPL_FUSED), ("chain", gspn.IMPL_CHAIN),
             ("plane", gspn.IMPL_PLANE)]


@pytest.mark.parametrize("name,impl", BWD_IMPLS, ids=[n for n, _ in BWD_IMPLS])
def test_out_of_grid_taps_are_never_read_backward(name, impl):
    """Every gradient but the dw3 entries of the poisoned taps themselves is unchanged (those entries multiply h
    outside the grid, which is 0: the kernels write 0 there whatever the tap holds)."""
    ran = 0
    for shape in [(1, 4, 16, 16, 2), (2, 4, 27, 27, 1), (1, 2, 40, 24, 1)]:
        for dtype in ("f32", "bf16"):
            cfg = gi.small_config("nanb", *shape, seed=72, backward=True)
            d = {k: v.cuda() for k, v in gi.make_inputs(cfg, dtype, with_dy=True).items()}
            g0 = _try(lambda: gspn.gspn_scan_bwd(d["x"], d["w3"], d["lam"], d["u"], d["dy"], cfg.G, cfg.dir_mask, impl=impl))
            if g0 is None:
                continue
            g1 = gspn.gspn_scan_bwd(d["x"], _poison(d, cfg), d["lam"], d["u"], d["dy"], cfg.G, cfg.dir_mask, impl=impl)
            for k in g0:
                if not torch.equal(g0[k], g1[k]) and name not in STRICT:
                    pytest.xfail(f"{name}: a NaN in an out-of-grid tap reaches {k} at {shape} {dtype}")
                assert torch.equal(g0[k], g1[k]), (shape, dtype, k)
            ran += 1
    assert ran >= 1


# ---------------------------------------------------------------------------------- run-to-run bit identity (hole g)
@pytest.mark.parametrize("name,impl", FWD_IMPLS, ids=[n for n, _ in FWD_IMPLS])
def test_forward_is_bit_identical_run_to_run(name, impl):
    """compute-sanitizer is closed on this pool; the named-barrier half swaps and the mbarrier hand-offs are checked
    by repetition instead: five runs on the same operands give the same bits."""
    ran = 0
    for shape, dtype in [((4, 8, 73, 73, 2), "bf16"), ((2, 8, 56, 56, 2), "bf16"), ((2, 8, 128, 128, 2), "bf16"),
                         ((8, 8, 27, 27, 2), "bf16"), ((2, 4, 56, 56, 1), "f32")]:
        cfg = gi.small_config("rep", *shape, seed=81)
        d = {k: v.cuda() for k, v in gi.make_inputs(cfg, dtype).items()}
        y0 = _try(lambda: gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, cfg.dir_mask, impl=impl))
        if y0 is None:
            continue
        for _ in range(4):
            y = gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, cfg.dir_mask, impl=impl)
            assert torch.equal(y, y0), (shape, dtype)
        ran += 1
    assert ran >= 1


@pytest.mark.parametrize("name,impl", BWD_IMPLS, ids=[n for n, _ in BWD_IMPLS])
def test_backward_is_bit_identical_run_to_run(name, impl):
    ran = 0
    for shape, dtype in [((4, 8, 73, 73, 2), "bf16"), ((8, 8, 27, 27, 2), "bf16"), ((2, 4, 56, 56, 1), "f32")]:
        cfg = gi.small_config("repb", *shape, seed=82, backward=True)
        d = {k: v.cuda() for k, v in gi.make_inputs(cfg, dtype, with_dy=True).items()}
        g0 = _try(lambda: gspn.gspn_scan_bwd(d["x"], d["w3"], d["lam"], d["u"], d["dy"], cfg.G, cfg.dir_mask, impl=impl))
        if g0 is None:
            continue
        for _ in range(4):
            g = gspn.gspn_scan_bwd(d["x"], d["w3"], d["lam"], d["u"], d["dy"], cfg.G, cfg.dir_mask, impl=impl)
            for k in g0:
                assert torch.equal(g[k], g0[k]), (shape, dtype, k)
        ran += 1
    assert ran >= 1


# ---------------------------------------------------------------------------------- optional outputs per kernel (ADVICE low)
@pytest.mark.parametrize("name,impl", BWD_IMPLS, ids=[n for n, _ in BWD_IMPLS])
@pytest.mark.parametrize("shape", [(1, 4, 8, 8, 2), (1, 4, 40, 44, 2)], ids=["8x8", "40x44"])
def test_optional_outputs_per_kernel(shape, name, impl):
    """NULL output pointers (any subset) leave the other outputs bit-identical, for every backward kernel and for
    lines longer than one warp."""
    cfg = gi.small_config("opt2", *shape, seed=91, backward=True)
    t = {k: v.cuda() for k, v in gi.make_inputs(cfg, "f32", with_dy=True).items()}
    full = _try(lambda: gspn.gspn_scan_bwd(t["x"], t["w3"], t["lam"], t["u"], t["dy"], cfg.G, cfg.dir_mask, impl=impl))
    if full is None:
        pytest.skip("shape not held by this kernel")
    for need in (("dx",), ("dw3",), ("du", "dh0"), ("dlambda", "dw3"), ("dh0",)):
        part = gspn.gspn_scan_bwd(t["x"], t["w3"], t["lam"], t["u"], t["dy"], cfg.G, cfg.dir_mask, need=need, impl=impl)
        assert set(part) == set(need)
        for k in need:
            assert torch.equal(part[k], full[k]), (need, k)


# ---------------------------------------------------------------------------------- the group backward
GROUP_SHAPES = [(1, 4, 27, 27, 1), (2, 4, 8, 8, 2), (1, 2, 40, 44, 2), (1, 4, 33, 35, 1), (1, 2, 100, 36, 1)]


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", GROUP_SHAPES, ids=["x".join(map(str, s)) for s in GROUP_SHAPES])
def test_group_backward_forced(shape, dtype):
    """fused_bwd_group sits in GSPN_IMPL_AUTO's fall-back chain but no round-1 test forced it: parity with masks and h0."""
    ran = 0
    for mask in (15, 6, 9):
        cfg = gi.small_config("grp", *shape, dir_mask=mask, seed=95 + mask, backward=True)
        r = _try(lambda: pu.check_bwd(cfg, dtype, impl=gspn.IMPL_FUSED, with_h0=True))
        if r is None:
            continue
        assert r["ok"] and r["variant"] == "fused_bwd_group", (mask, r)
        ran += 1
    if not ran:
        pytest.skip("shape not held by the group kernel")


@pytest.mark.parametrize("shape,dtype", [((1, 4, 27, 27, 1), "f32"), ((1, 2, 144, 144, 2), "bf16")], ids=["27x27-cg4-f32", "144x144-cg1-bf16"])
def test_auto_backward_fallback_shapes(shape, dtype, record_property):
    """Shapes the preferred backward kernels refuse (plane: fp32 planes beyond shared memory; chain: lines beyond 128):
    AUTO must still return oracle-exact gradients, whatever it lands on; the variant is recorded."""
    cfg = gi.small_config("fb", *shape, seed=97, backward=True)
    r = _try(lambda: pu.check_bwd(cfg, dtype, with_h0=True))
    if r is None:
        pytest.xfail("no backward kernel under GSPN_IMPL_AUTO holds this shape")
    record_property("variant", r["variant"])
    assert r["ok"], r


# ---------------------------------------------------------------------------------- the fused, pipelined host call
@pytest.mark.parametrize("shape", [(1, 4, 16, 16, 2), (5, 4, 37, 41, 2), (9, 8, 27, 27, 2)], ids=["B1", "B5", "B9"])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_fused_host_call_matches_the_oracle(dtype, shape):
    """gspn_scan_fwd_bwd_host: operands uploaded once, up to four batch chunks on three streams (ragged last chunk at
    B = 5 and 9); y and every gradient against the oracle, then with some outputs left out."""
    cfg = gi.small_config("fh", *shape, seed=53, backward=True)
    t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True)
    host = {k: v.contiguous().pin_memory() for k, v in t.items()}
    st = host["x"].dtype
    mk = lambda *s: torch.full(s, float("nan"), dtype=st).pin_memory()
    L = max(cfg.H, cfg.W)
    y = mk(*host["x"].shape)
    outs = {"dx": mk(*host["x"].shape), "dlambda": mk(*host["lam"].shape), "du": mk(*host["u"].shape),
            "dw3": mk(*host["w3"].shape), "dh0": mk(cfg.D, cfg.B, cfg.C, L)}
    gspn.gspn_scan_fwd_bwd_host(host["x"], host["w3"], host["lam"], host["u"], host["dy"], y, outs["dx"], outs["dlambda"],
                                outs["du"], outs["dw3"], outs["dh0"], cfg.G, cfg.dir_mask)
    yo, A = pu.oracle_fwd(t, cfg)
    r = pu.gate(pu.np64(y), yo, A, dtype)
    assert r["ok"], r
    go, Ag = pu.oracle_bwd(t, cfg)
    for k in ("dx", "dlambda", "du", "dw3"):
        r = pu.gate(pu.np64(outs[k]), go[k], Ag[k], dtype)
        assert r["ok"], (k, r)
    # dh0: entries past a direction's line are not written (they keep the NaN fill); compare the lines
    for q, d in enumerate(gi.dir_list(cfg.dir_mask)):
        n = cfg.W if d < 2 else cfg.H
        r = pu.gate(pu.np64(outs["dh0"][q, ..., :n]), go["dh0"][q, ..., :n], Ag["dh0"][q, ..., :n], dtype)
        assert r["ok"], ("dh0", q, r)
    # forward only / a subset of the gradients
    y2, dw2 = mk(*host["x"].shape), mk(*host["w3"].shape)
    gspn.gspn_scan_fwd_bwd_host(host["x"], host["w3"], host["lam"], host["u"], host["dy"], y2, None, None, None, None, None,
                                cfg.G, cfg.dir_mask)
    assert torch.equal(y2, y)
    gspn.gspn_scan_fwd_bwd_host(host["x"], host["w3"], host["lam"], host["u"], host["dy"], None, None, None, None, dw2, None,
                                cfg.G, cfg.dir_mask)
    assert torch.equal(dw2, outs["dw3"])


# ---------------------------------------------------------------------------------- shared direction slabs
SHARED_SETS = [("w3",), ("lam", "u"), ("w3", "lam", "u")]


@pytest.mark.parametrize("shared", SHARED_SETS, ids=["+".join(s) for s in SHARED_SETS])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_shared_direction_slabs(dtype, shared):
    """gspn_args_t.dir_stride_* = 0 (reading 6): ONE slab of w3 / lambda / u read by every
    direction.  Oracle: the same slab replicated over the D directions (what "shared" means); the gradients stay per
    direction.  Also bit-identical to the dense call on the replicated operands (same kernel, same arithmetic), and
    refused by every kernel but the naive one."""
    for shape, mask in [((2, 4, 16, 16, 2), 15), ((1, 4, 37, 41, 2), 15), ((2, 2, 27, 27, 1), 6), ((1, 2, 70, 33, 1), 9)]:
        cfg = gi.small_config("shr", *shape, dir_mask=mask, seed=88, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True)
        rep = dict(t)
        for k in shared:
            rep[k] = t[k][:1].expand(cfg.D, *t[k].shape[1:]).contiguous()
        d = {k: v.cuda() for k, v in rep.items()}
        one = {k: (t[k][0].contiguous().cuda() if k in shared else d[k]) for k in ("w3", "lam", "u")}
        y = gspn.gspn_scan_fwd(d["x"], one["w3"], one["lam"], one["u"], cfg.G, mask, shared=shared)
        assert gspn.gspn_last_variant() == "naive_fwd"
        yo, A = pu.oracle_fwd(rep, cfg)
        r = pu.gate(pu.np64(y), yo, A, dtype)
        assert r["ok"], (shape, mask, r)
        assert torch.equal(y, gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, mask, impl=gspn.IMPL_NAIVE))
        g = gspn.gspn_scan_bwd(d["x"], one["w3"], one["lam"], one["u"], d["dy"], cfg.G, mask, shared=shared)
        assert gspn.gspn_last_variant() == "naive_bwd"
        go, Ag = pu.oracle_bwd(rep, cfg)
        gd = gspn.gspn_scan_bwd(d["x"], d["w3"], d["lam"], d["u"], d["dy"], cfg.G, mask, impl=gspn.IMPL_NAIVE)
        for k in ("dx", "dlambda", "du", "dw3", "dh0"):
            assert tuple(g[k].shape) == tuple(gd[k].shape), k          # one slab per direction, shared or not
            r = pu.gate(pu.np64(g[k]), go[k], Ag[k], dtype)
            assert r["ok"], (shape, mask, k, r)
            assert torch.equal(g[k], gd[k]), (shape, mask, k)
    with pytest.raises(gspn.GspnError) as ei:
        gspn.gspn_scan_fwd(d["x"], one["w3"], one["lam"], one["u"], cfg.G, mask, shared=shared, impl=gspn.IMPL_CHAIN)
    assert ei.value.status == 2


# ---------------------------------------------------------------------------------- chunked scan
@pytest.mark.parametrize("k_chunk", [2, 3, 7])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_chunked_scan_matches_the_oracle(dtype, k_chunk):
    """gspn_args_t.k_chunk (reading 10): bands of ceil(L / k_chunk) lines in image coordinates, independent
    scans with a zero initial state; forward and every gradient against oracle.fwd_chunked / bwd_chunked, with h0, ragged
    last bands (37 / 3, 41 / 7, 70 / 3) and direction subsets; k_chunk = 1 is bit-identical to the plain call."""
    from oracle import gspn_oracle as orc
    for shape, mask in [((2, 4, 16, 16, 2), 15), ((1, 4, 37, 41, 2), 15), ((2, 2, 27, 27, 1), 6), ((1, 2, 70, 33, 1), 9)]:
        cfg = gi.small_config("chk", *shape, dir_mask=mask, seed=99, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
        d = {k: v.cuda() for k, v in t.items()}
        n = {k: pu.np64(v) for k, v in t.items()}
        y = gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, mask, h0=d["h0"], k_chunk=k_chunk)
        assert gspn.gspn_last_variant() == "naive_fwd"
        yo = orc.fwd_chunked(n["x"], n["w3"], n["lam"], n["u"], cfg.G, mask, k_chunk, h0=n["h0"])
        A = orc.fwd_chunked_magnitude(n["x"], n["w3"], n["lam"], n["u"], cfg.G, mask, k_chunk, h0=n["h0"])
        r = pu.gate(pu.np64(y), yo, A, dtype)
        assert r["ok"], (shape, mask, r)
        g = gspn.gspn_scan_bwd(d["x"], d["w3"], d["lam"], d["u"], d["dy"], cfg.G, mask, h0=d["h0"], k_chunk=k_chunk)
        assert gspn.gspn_last_variant() == "naive_bwd"
        go = orc.bwd_chunked(n["x"], n["w3"], n["lam"], n["u"], n["dy"], cfg.G, mask, k_chunk, h0=n["h0"])
        Ag = orc.bwd_chunked_magnitude(n["x"], n["w3"], n["lam"], n["u"], n["dy"], cfg.G, mask, k_chunk, h0=n["h0"])
        for k in ("dx", "dlambda", "du", "dw3", "dh0"):
            r = pu.gate(pu.np64(g[k]), go[k], Ag[k], dtype)
            assert r["ok"], (shape, mask, k, r)
        y1 = gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, mask, h0=d["h0"], k_chunk=1, impl=gspn.IMPL_NAIVE)
        assert torch.equal(y1, gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, mask, h0=d["h0"], impl=gspn.IMPL_NAIVE))
        assert not torch.equal(y1, y)                     # the bands matter
    with pytest.raises(gspn.GspnError) as ei:
        gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, mask, k_chunk=2, impl=gspn.IMPL_CHAIN)
    assert ei.value.status == 2


# ---------------------------------------------------------------------------------- logits in the load path (second half)
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_logits_in_the_load_path(dtype):
    """GSPN_FLAG_W3_LOGITS: `w3` holds raw logits, Eq. 3 is applied where the taps are loaded (normalised taps never written
    to memory), and the backward writes the gradient of the logits.  Oracle: normalize -> fwd, bwd -> normalize_bwd in fp64
    (tests/parity_util.oracle_logits).  Also against the two-kernel route (gspn_normalize_fwd, then the scan) in fp32,
    where both keep full-precision taps."""
    for shape, mask in [((2, 4, 16, 16, 2), 15), ((1, 4, 37, 41, 2), 15), ((2, 2, 27, 27, 1), 6), ((1, 2, 70, 33, 1), 9)]:
        cfg = gi.small_config("lgt", *shape, dir_mask=mask, seed=131, backward=True)
        t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=True)
        wt = gi.make_logits(cfg, dtype)["wt"]
        d = {k: v.cuda() for k, v in t.items()}
        wd = wt.cuda()
        yo, A, go, Ag = pu.oracle_logits(t, wt, cfg)
        y = gspn.gspn_scan_fwd(d["x"], wd, d["lam"], d["u"], cfg.G, mask, h0=d["h0"], w3_logits=True)
        assert gspn.gspn_last_variant() == "naive_fwd"
        r = pu.gate(pu.np64(y), yo, A, dtype)
        assert r["ok"], (shape, mask, r)
        g = gspn.gspn_scan_bwd(d["x"], wd, d["lam"], d["u"], d["dy"], cfg.G, mask, h0=d["h0"], w3_logits=True)
        for k in ("dx", "dlambda", "du", "dw3", "dh0"):
            r = pu.gate(pu.np64(g[k]), go[k], Ag[k], dtype)
            assert r["ok"], (shape, mask, k, r)
        if dtype == "f32":      # two-kernel route: normalise into fp32 taps, then the same naive scan
            w3 = gspn.gspn_normalize_fwd(wd, mask)
            y2 = gspn.gspn_scan_fwd(d["x"], w3, d["lam"], d["u"], cfg.G, mask, h0=d["h0"], impl=gspn.IMPL_NAIVE)
            assert pu.gate(pu.np64(y2), yo, A, dtype)["ok"]
    with pytest.raises(gspn.GspnError) as ei:
        gspn.gspn_scan_fwd(d["x"], wd, d["lam"], d["u"], cfg.G, mask, w3_logits=True, impl=gspn.IMPL_CHAIN)
    assert ei.value.status == 2


# ---------------------------------------------------------------------------------- large planes (first step)
@pytest.mark.parametrize("shape,dtype", [((1, 2, 256, 256, 1), "bf16"), ((1, 2, 300, 260, 2), "f32"), ((1, 2, 1024, 1024, 1), "bf16"),
                                         ((2, 2, 512, 64, 1), "f32")], ids=["256x256-bf16", "300x260-f32", "1024x1024-bf16", "512x64-f32"])
def test_large_plane_forward(shape, dtype, record_property):
    """Planes beyond shared memory (the paper's 256^2 .. 1024^2 shapes): served through the caller
    workspace (gspn_args_t.workspace, allocated by the binding from gspn_workspace_bytes).  Whole tensor against the oracle."""
    cfg = gi.small_config("big", *shape, seed=141)
    B, C, H, W, G = shape
    need = gspn.lib().gspn_workspace_bytes(B, C, H, W, G, 15, 0 if dtype == "f32" else 1, 0)
    r = pu.check_fwd(cfg, dtype)
    record_property("variant", r["variant"])
    assert r["ok"], r
    if 4 * H * W + 8 * (max(H, W) + 2) > 227 * 1024:
        assert need == 4 * B * C * H * W
        assert r["variant"] != "naive_fwd"                 # the shared-memory mode cannot hold it (flat_fwd takes lines up to 256)
        if max(H, W) > 256:
            assert r["variant"] == "naive_fwd_ws", r["variant"]
    else:
        assert need == 0


@pytest.mark.parametrize("shape,dtype", [((1, 2, 160, 160, 1), "bf16"), ((1, 4, 128, 128, 1), "bf16"), ((1, 2, 256, 256, 2), "f32"),
                                         ((1, 1, 600, 40, 1), "bf16")], ids=["160x160-bf16", "128x128-cg4-bf16", "256x256-f32", "600x40-bf16"])
def test_large_plane_backward(shape, dtype, record_property):
    """The backward of planes no kernel holds on chip (from about 120 x 120): every gradient against the oracle; the
    variant that ran is recorded."""
    cfg = gi.small_config("bigb", *shape, seed=142, backward=True)
    r = pu.check_bwd(cfg, dtype, with_h0=True)
    record_property("variant", r["variant"])
    assert r["ok"], r


def test_workspace_errors():
    """Without a workspace the large-plane shapes report GSPN_EWORKSPACE (status 4) through the plain C call; a forced
    fused kernel still reports GSPN_EUNSUPPORTED."""
    import ctypes
    cfg = gi.small_config("bige", 1, 2, 256, 256, 1, seed=143)
    d = {k: v.cuda() for k, v in gi.make_inputs(cfg, "f32").items()}
    y = torch.empty_like(d["x"])
    p = lambda t: ctypes.c_void_p(t.data_ptr())
    rc = gspn.lib().gspn_scan_fwd(p(d["x"]), p(d["w3"]), p(d["lam"]), p(d["u"]), p(y), 1, 2, 256, 256, 1, 15, 0, None)
    assert rc == 4 and b"workspace" in gspn.lib().gspn_last_error()
    with pytest.raises(gspn.GspnError) as ei:
        gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, 15, impl=gspn.IMPL_CHAIN)
    assert ei.value.status == 2
