"""ctypes front end of the CPU oracle (oracle/gspn_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg.  Nothing under
paper_2606_00746_b200/ imports this module and this module imports nothing
from there.

All functions take and return C-contiguous numpy arrays in the layouts of
include/gspn.h (x [B,C,H,W]; w3 [D,B,G,3,H,W]; lambda,u [D,B,C,H,W];
h0/dh0 [D,B,C,max(H,W)]).  dtype float64 selects the truth build, float32 the
pinned-order diagnostic build.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gspn_oracle.c")
_HDR = os.path.join(_HERE, "gspn_oracle_impl.h")
_LIB = os.path.join(_HERE, "libgspn_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, OpenMP over planes, no FMA contraction)."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", _LIB + ".tmp", _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
        os.replace(_LIB + ".tmp", _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
    return _lib


def threads() -> int:
    return int(_load().gspn_oracle_threads())


def set_threads(n: int) -> None:
    _load().gspn_oracle_set_threads(int(n))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _prep(a, dt):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=dt)
    return a


def popcount(mask: int) -> int:
    return bin(mask & 15).count("1")


def _check(x, w3, lam, u, G, mask, h0=None):
    B, C, H, W = x.shape
    D = popcount(mask)
    assert w3.shape == (D, B, G, 3, H, W), (w3.shape, (D, B, G, 3, H, W))
    assert lam.shape == (D, B, C, H, W) and u.shape == (D, B, C, H, W)
    if h0 is not None:
        assert h0.shape == (D, B, C, max(H, W))
    return B, C, H, W, D


def fwd(x, w3, lam, u, G: int, mask: int, h0=None, return_h: bool = False):
    """y = sum_d u_d * scan_d(x)  (Eq. 1, 2, 5, 9).  Returns y or (y, h[D,B,C,H,W])."""
    dt = np.float32 if x.dtype == np.float32 else np.float64
    x, w3, lam, u, h0 = (_prep(a, dt) for a in (x, w3, lam, u, h0))
    B, C, H, W, D = _check(x, w3, lam, u, G, mask, h0)
    y = np.empty_like(x)
    hs = np.empty((D, B, C, H, W), dtype=dt) if return_h else None
    fn = _load().gspn_oracle_fwd_f32 if dt == np.float32 else _load().gspn_oracle_fwd_f64
    rc = fn(_ptr(x), _ptr(w3), _ptr(lam), _ptr(u), _ptr(h0), _ptr(y), _ptr(hs),
            B, C, H, W, int(G), ctypes.c_uint(mask))
    if rc != 0:
        raise ValueError("gspn_oracle_fwd: invalid arguments")
    return (y, hs) if return_h else y


def bwd(x, w3, lam, u, dy, G: int, mask: int, h0=None):
    """Adjoint of fwd.  Returns dict(dx, dlambda, du, dw3, dh0)."""
    dt = np.float32 if x.dtype == np.float32 else np.float64
    x, w3, lam, u, dy, h0 = (_prep(a, dt) for a in (x, w3, lam, u, dy, h0))
    B, C, H, W, D = _check(x, w3, lam, u, G, mask, h0)
    assert dy.shape == x.shape
    out = dict(dx=np.empty_like(x), dlambda=np.empty_like(lam), du=np.empty_like(u),
               dw3=np.empty_like(w3), dh0=np.empty((D, B, C, max(H, W)), dtype=dt))
    fn = _load().gspn_oracle_bwd_f32 if dt == np.float32 else _load().gspn_oracle_bwd_f64
    rc = fn(_ptr(x), _ptr(w3), _ptr(lam), _ptr(u), _ptr(h0), _ptr(dy), _ptr(out["dx"]),
            _ptr(out["dlambda"]), _ptr(out["du"]), _ptr(out["dw3"]), _ptr(out["dh0"]),
            B, C, H, W, int(G), ctypes.c_uint(mask))
    if rc != 0:
        raise ValueError("gspn_oracle_bwd: invalid arguments")
    return out


def merge(y_dirs, m=None):
    """y = sum_q m[q,c] * y_dirs[q]  (m None = ones)."""
    y_dirs = _prep(y_dirs, np.float64)
    m = _prep(m, np.float64)
    D, B, C, H, W = y_dirs.shape
    y = np.empty((B, C, H, W), dtype=np.float64)
    rc = _load().gspn_oracle_merge_f64(_ptr(y_dirs), _ptr(m), _ptr(y), D, B, C, H, W)
    if rc != 0:
        raise ValueError("gspn_oracle_merge: invalid arguments")
    return y


NORM_EPS = 1e-6      # clamp bound of Eq. (3)'s denominator (reading R17; the paper gives none)


def normalize(wt, mask: int, eps: float = NORM_EPS):
    """w3 = Eq. (3) of the logits wt [D,B,G,3,H,W] (fp64): sigmoid, sum over the in-grid taps, clamp, divide."""
    wt = _prep(wt, np.float64)
    D, B, G, three, H, W = wt.shape
    assert three == 3 and D == popcount(mask)
    w3 = np.empty_like(wt)
    rc = _load().gspn_oracle_normalize_f64(_ptr(wt), _ptr(w3), B, G, H, W, ctypes.c_uint(mask),
                                           ctypes.c_double(eps))
    if rc != 0:
        raise ValueError("gspn_oracle_normalize: invalid arguments")
    return w3


def normalize_bwd(wt, dw3, mask: int, eps: float = NORM_EPS, magnitude: bool = False):
    """dwt = adjoint of normalize at wt applied to dw3 (fp64); magnitude=True: sum of |terms| instead."""
    wt = _prep(wt, np.float64)
    dw3 = _prep(dw3, np.float64)
    D, B, G, three, H, W = wt.shape
    assert three == 3 and D == popcount(mask) and dw3.shape == wt.shape
    dwt = np.empty_like(wt)
    rc = _load().gspn_oracle_normalize_bwd_f64(_ptr(wt), _ptr(dw3), _ptr(dwt), B, G, H, W,
                                               ctypes.c_uint(mask), ctypes.c_double(eps), int(magnitude))
    if rc != 0:
        raise ValueError("gspn_oracle_normalize_bwd: invalid arguments")
    return dwt


def fwd_magnitude(x, w3, lam, u, G: int, mask: int, h0=None):
    """A >= |y| elementwise: the same recurrence on |x|, |lambda|, |u|, |w3|, |h0|.

    A_i is the sum of the absolute values of the terms behind y_i, i.e. the
    natural scale of its rounding error (tolerance section)."""
    a = [np.abs(np.asarray(t, dtype=np.float64)) for t in (x, w3, lam, u)]
    return fwd(a[0], a[1], a[2], a[3], G, mask,
               None if h0 is None else np.abs(np.asarray(h0, dtype=np.float64)))


def bwd_magnitude(x, w3, lam, u, dy, G: int, mask: int, h0=None):
    a = [np.abs(np.asarray(t, dtype=np.float64)) for t in (x, w3, lam, u, dy)]
    return bwd(a[0], a[1], a[2], a[3], a[4], G, mask,
               None if h0 is None else np.abs(np.asarray(h0, dtype=np.float64)))


# ---------------------------------------------------------------------------------------------------------------------
# Chunked scan (PAPER.md:125,129 use `k_chunk` in the launch grid `(chunk, b, c)` and never define it).
# Reading (reading 10): the scan axis is cut, in IMAGE coordinates, into k_chunk bands of Lc = ceil(L / k_chunk)
# lines (the last band may be shorter, and fewer than k_chunk bands exist when Lc * (k_chunk - 1) >= L); every band is an
# independent scan on its sub-grid with a zero initial state.  Both directions of an axis share the bands.  h0 / dh0 belong
# to the band that holds scan step 0 of the direction.  The definition is written out as such: slice, call the plain
# oracle above (one direction at a time) on the sub-grid, put the pieces back.  y sums the directions in ascending order.
def chunk_bands(L: int, k_chunk: int):
    """[(first line, one past the last line)] of the bands of a scan axis of L lines."""
    assert k_chunk >= 1
    Lc = -(-L // k_chunk)
    return [(a, min(a + Lc, L)) for a in range(0, L, Lc)]


def _band_views(d, a, b):
    """Index tuples of band [a, b) of direction d for [B,C,H,W] and for one direction slab [1,B,*,...,H,W]."""
    img = (slice(None), slice(None), slice(a, b), slice(None)) if d < 2 else (slice(None), slice(None), slice(None), slice(a, b))
    return img, (Ellipsis,) + img[2:]


def _band_h0(h0, q, d, a, b, H, W, shape_bc):
    """h0 of the sub-problem: the direction's h0 for the band holding scan step 0, else None."""
    L = H if d < 2 else W
    holds_step0 = (a == 0) if d in (0, 2) else (b == L)
    if h0 is None or not holds_step0:
        return None, holds_step0
    Lp = W if d < 2 else H
    Hb, Wb = (b - a, W) if d < 2 else (H, b - a)
    sub = np.zeros((1,) + shape_bc + (max(Hb, Wb),), dtype=h0.dtype)
    sub[0, ..., :Lp] = h0[q, ..., :Lp]
    return sub, holds_step0


def fwd_chunked(x, w3, lam, u, G: int, mask: int, k_chunk: int, h0=None):
    """y of the chunked scan: per direction and band, the plain forward on the sub-grid."""
    dt = np.float32 if x.dtype == np.float32 else np.float64
    x, w3, lam, u, h0 = (_prep(a, dt) for a in (x, w3, lam, u, h0))
    B, C, H, W, D = _check(x, w3, lam, u, G, mask, h0)
    y = np.zeros_like(x)
    for q, d in enumerate(dd for dd in range(4) if mask >> dd & 1):
        for a, b in chunk_bands(H if d < 2 else W, k_chunk):
            img, slab = _band_views(d, a, b)
            h0b, _ = _band_h0(h0, q, d, a, b, H, W, (B, C))
            y[img] += fwd(x[img], w3[q:q + 1][slab], lam[q:q + 1][slab], u[q:q + 1][slab], G, 1 << d, h0=h0b)
    return y


def bwd_chunked(x, w3, lam, u, dy, G: int, mask: int, k_chunk: int, h0=None):
    """Adjoint of fwd_chunked: per direction and band, the plain backward on the sub-grid; dx sums the directions in
    ascending order; dh0 comes from the band that holds scan step 0 (entries past the line are 0)."""
    dt = np.float32 if x.dtype == np.float32 else np.float64
    x, w3, lam, u, dy, h0 = (_prep(a, dt) for a in (x, w3, lam, u, dy, h0))
    B, C, H, W, D = _check(x, w3, lam, u, G, mask, h0)
    out = dict(dx=np.zeros_like(x), dlambda=np.zeros_like(lam), du=np.zeros_like(u), dw3=np.zeros_like(w3),
               dh0=np.zeros((D, B, C, max(H, W)), dtype=dt))
    for q, d in enumerate(dd for dd in range(4) if mask >> dd & 1):
        Lp = W if d < 2 else H
        for a, b in chunk_bands(H if d < 2 else W, k_chunk):
            img, slab = _band_views(d, a, b)
            h0b, holds_step0 = _band_h0(h0, q, d, a, b, H, W, (B, C))
            g = bwd(x[img], w3[q:q + 1][slab], lam[q:q + 1][slab], u[q:q + 1][slab], dy[img], G, 1 << d, h0=h0b)
            out["dx"][img] += g["dx"]
            out["dlambda"][q:q + 1][slab] = g["dlambda"]
            out["du"][q:q + 1][slab] = g["du"]
            out["dw3"][q:q + 1][slab] = g["dw3"]
            if holds_step0:
                out["dh0"][q, ..., :Lp] = g["dh0"][0, ..., :Lp]
    return out


def fwd_chunked_magnitude(x, w3, lam, u, G: int, mask: int, k_chunk: int, h0=None):
    a = [np.abs(np.asarray(t, dtype=np.float64)) for t in (x, w3, lam, u)]
    return fwd_chunked(a[0], a[1], a[2], a[3], G, mask, k_chunk, None if h0 is None else np.abs(np.asarray(h0, dtype=np.float64)))


def bwd_chunked_magnitude(x, w3, lam, u, dy, G: int, mask: int, k_chunk: int, h0=None):
    a = [np.abs(np.asarray(t, dtype=np.float64)) for t in (x, w3, lam, u, dy)]
    return bwd_chunked(a[0], a[1], a[2], a[3], a[4], G, mask, k_chunk, None if h0 is None else np.abs(np.asarray(h0, dtype=np.float64)))
