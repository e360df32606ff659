"""Pins of the chunked-scan oracle (oracle/gspn_oracle.py fwd_chunked / bwd_chunked, DESIGN.md
reading 10: bands of ceil(L / k_chunk) lines in image coordinates, each an independent scan with a zero initial state).

Nothing here calls the chunked oracle to produce its own expected values: a step-by-step recurrence with the reset rule
written out independently (pure Python loops, tiny sizes), scipy's lfilter / numpy's cumsum per band, the plain oracle at
k_chunk = 1, locality of a perturbation, and central finite differences for the adjoint.  CPU only.
"""
import numpy as np
import pytest
from scipy.signal import lfilter

from oracle import gspn_oracle as orc


def rand_problem(rng, B, C, H, W, G, mask, with_h0=True):
    D = orc.popcount(mask)
    x = rng.standard_normal((B, C, H, W))
    lam = rng.uniform(0.1, 1.0, (D, B, C, H, W))
    u = rng.standard_normal((D, B, C, H, W))
    w3 = rng.uniform(0.05, 1.0, (D, B, G, 3, H, W))
    w3 /= w3.sum(axis=3, keepdims=True)
    h0 = rng.standard_normal((D, B, C, max(H, W))) if with_h0 else None
    return x, w3, lam, u, h0


def pixel(d, s, p, H, W):
    """Image (i, j) of scan step s, cross position p (ascending rows / columns for d = 0 / 2, descending for 1 / 3)."""
    return [(s, p), (H - 1 - s, p), (p, s), (p, W - 1 - s)][d]


def loops_fwd(x, w3, lam, u, G, mask, k_chunk, h0):
    """The recurrence of Eq. (1)-(2) one step at a time; at the first line of a band (image coordinates) the state of the
    line before counts as zero.  Independent of the oracle's slicing: one pass over the whole axis with a reset test."""
    B, C, H, W = x.shape
    cg = C // G
    y = np.zeros_like(x)
    for q, d in enumerate(dd for dd in range(4) if mask >> dd & 1):
        Ls, Lp = (H, W) if d < 2 else (W, H)
        Lc = -(-Ls // k_chunk)
        for b in range(B):
            for c in range(C):
                prev = np.zeros(Lp) if h0 is None else h0[q, b, c, :Lp].copy()
                for s in range(Ls):
                    line = (Ls - 1 - s) if d in (1, 3) else s                    # image coordinate along the scan axis
                    band_entry = (line % Lc == Lc - 1 or line == Ls - 1) if d in (1, 3) else (line % Lc == 0)
                    if s > 0 and band_entry:
                        prev = np.zeros(Lp)
                    cur = np.zeros(Lp)
                    for p in range(Lp):
                        i, j = pixel(d, s, p, H, W)
                        acc = lam[q, b, c, i, j] * x[b, c, i, j]
                        for k in range(3):
                            pn = p + k - 1
                            if 0 <= pn < Lp:
                                acc += w3[q, b, c // cg, k, i, j] * prev[pn]
                        cur[p] = acc
                        y[b, c, i, j] += u[q, b, c, i, j] * acc
                    prev = cur
    return y


@pytest.mark.parametrize("mask", [15, 1, 2, 4, 8, 6])
@pytest.mark.parametrize("k_chunk", [2, 3, 5])
def test_chunked_forward_matches_the_step_by_step_recurrence_with_resets(mask, k_chunk):
    rng = np.random.default_rng(100 + mask + k_chunk)
    B, C, H, W, G = 1, 2, 7, 5, 1
    x, w3, lam, u, h0 = rand_problem(rng, B, C, H, W, G, mask)
    want = loops_fwd(x, w3, lam, u, G, mask, k_chunk, h0)
    got = orc.fwd_chunked(x, w3, lam, u, G, mask, k_chunk, h0=h0)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)
    # and it is not the global scan (the reset matters)
    assert np.abs(got - orc.fwd(x, w3, lam, u, G, mask, h0=h0)).max() > 1e-3


def test_one_chunk_is_the_plain_scan():
    rng = np.random.default_rng(5)
    x, w3, lam, u, h0 = rand_problem(rng, 2, 4, 9, 6, 2, 15)
    dy = rng.standard_normal(x.shape)
    np.testing.assert_array_equal(orc.fwd_chunked(x, w3, lam, u, 2, 15, 1, h0=h0), orc.fwd(x, w3, lam, u, 2, 15, h0=h0))
    g1, g0 = orc.bwd_chunked(x, w3, lam, u, dy, 2, 15, 1, h0=h0), orc.bwd(x, w3, lam, u, dy, 2, 15, h0=h0)
    for k in g0:
        np.testing.assert_array_equal(g1[k], g0[k], err_msg=k)


def test_bands_cover_the_axis_once():
    for L in (1, 5, 7, 73, 128):
        for k in (1, 2, 3, 4, 8, 200):
            bands = orc.chunk_bands(L, k)
            assert bands[0][0] == 0 and bands[-1][1] == L and len(bands) <= k
            assert all(b0[1] == b1[0] for b0, b1 in zip(bands, bands[1:]))
            Lc = -(-L // k)
            assert all(b - a == Lc for a, b in bands[:-1]) and 0 < bands[-1][1] - bands[-1][0] <= Lc


@pytest.mark.parametrize("d", [0, 1, 2, 3])
def test_centre_tap_only_is_a_first_order_filter_per_band(d):
    """Taps (0, a, 0), lambda = u = 1: every line of the cross axis is h[s] = a h[s-1] + x[s] restarted in every band:
    scipy.signal.lfilter per band (a = 1: numpy cumsum)."""
    rng = np.random.default_rng(31 + d)
    B, C, H, W, G, k_chunk = 1, 2, 11, 9, 1, 3
    x = rng.standard_normal((B, C, H, W))
    for a in (1.0, 0.6):
        w3 = np.zeros((1, B, G, 3, H, W)); w3[:, :, :, 1] = a
        lam = np.ones((1, B, C, H, W)); u = np.ones((1, B, C, H, W))
        got = orc.fwd_chunked(x, w3, lam, u, G, 1 << d, k_chunk)
        axis = 2 if d < 2 else 3
        want = np.zeros_like(x)
        for lo, hi in orc.chunk_bands(x.shape[axis], k_chunk):
            sl = [slice(None)] * 4; sl[axis] = slice(lo, hi)
            band = x[tuple(sl)]
            if d in (1, 3):
                band = np.flip(band, axis)
            f = np.cumsum(band, axis=axis) if a == 1.0 else lfilter([1.0], [1.0, -a], band, axis=axis)
            want[tuple(sl)] = np.flip(f, axis) if d in (1, 3) else f
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)


@pytest.mark.parametrize("d", [0, 1, 2, 3])
def test_a_perturbation_stays_inside_its_band(d):
    rng = np.random.default_rng(41 + d)
    B, C, H, W, G, k_chunk = 1, 2, 10, 12, 2, 4
    x, w3, lam, u, _ = rand_problem(rng, B, C, H, W, G, 1 << d, with_h0=False)
    y0 = orc.fwd_chunked(x, w3, lam, u, G, 1 << d, k_chunk)
    axis = 2 if d < 2 else 3
    bands = orc.chunk_bands(x.shape[axis], k_chunk)
    lo, hi = bands[1]
    x2 = x.copy()
    sl = [slice(None)] * 4; sl[axis] = slice(lo, hi)
    x2[tuple(sl)] += 1.0
    diff = orc.fwd_chunked(x2, w3, lam, u, G, 1 << d, k_chunk) - y0
    inside = np.zeros(x.shape, bool); inside[tuple(sl)] = True
    assert np.all(diff[~inside] == 0.0) and np.abs(diff[inside]).max() > 0.1


def _loss(x, w3, lam, u, h0, dy, G, mask, k):
    return float((orc.fwd_chunked(x, w3, lam, u, G, mask, k, h0=h0) * dy).sum())


@pytest.mark.parametrize("shape,k_chunk", [((1, 4, 8, 8, 2), 2), ((2, 2, 5, 7, 1), 3), ((1, 2, 6, 4, 2), 4)])
def test_chunked_backward_matches_central_finite_differences(shape, k_chunk):
    B, C, H, W, G = shape
    mask = 15
    rng = np.random.default_rng(19)
    x, w3, lam, u, h0 = rand_problem(rng, B, C, H, W, G, mask)
    w3 = rng.uniform(0.05, 1.0, w3.shape)                 # no row-sum constraint: every tap is a free variable
    dy = rng.standard_normal(x.shape)
    g = orc.bwd_chunked(x, w3, lam, u, dy, G, mask, k_chunk, h0=h0)
    eps = 1e-6
    for name, arr in {"dx": x, "dw3": w3, "dlambda": lam, "du": u, "dh0": h0}.items():
        flat, gflat = arr.reshape(-1), g[name].reshape(-1)
        for idx in rng.choice(flat.size, size=min(60, flat.size), replace=False):
            old = flat[idx]
            flat[idx] = old + eps; lp = _loss(x, w3, lam, u, h0, dy, G, mask, k_chunk)
            flat[idx] = old - eps; lm = _loss(x, w3, lam, u, h0, dy, G, mask, k_chunk)
            flat[idx] = old
            fd = (lp - lm) / (2 * eps)
            assert abs(fd - gflat[idx]) <= 1e-6 * max(1.0, abs(fd)), (name, idx, fd, gflat[idx])
    # the taps that multiply the (zero) state before a band's first line get no gradient; h0 reaches only the first band
    q_tb = 0
    for lo, hi in orc.chunk_bands(H, k_chunk)[1:]:
        assert np.all(g["dw3"][q_tb, :, :, :, lo, :] == 0.0)
