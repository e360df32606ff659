"""Pins of the CPU oracle against what the paper and the mathematics fix.

Nothing here compares the oracle with itself re-typed: every expected value is a
closed form, a library routine (numpy cumsum / matmul / polynomial, scipy lfilter),
a dense-matrix brute force of Eq. (4), an invariant or a
finite difference.  Runs on CPU only.
"""
import math
import os

import numpy as np
import pytest
from scipy.signal import lfilter

from oracle import gspn_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")
DIRS = {0: 1, 1: 2, 2: 4, 3: 8}     # dir id -> mask bit


# ----------------------------------------------------------------------------- helpers
def img_index(d, s, p, H, W):
    """Image (i,j) of scan step s, cross position p -- written independently of the oracle."""
    if d == 0:
        return s, p
    if d == 1:
        return H - 1 - s, p
    if d == 2:
        return p, s
    return p, W - 1 - s


def dims(d, H, W):
    return (H, W) if d < 2 else (W, H)     # (Ls, Lp)


def rand_problem(rng, B, C, H, W, G, mask, stochastic=True):
    D = orc.popcount(mask)
    x = rng.standard_normal((B, C, H, W))
    lam = rng.uniform(0.1, 1.0, (D, B, C, H, W))
    u = rng.standard_normal((D, B, C, H, W))
    w3 = rng.uniform(0.05, 1.0, (D, B, G, 3, H, W))
    if stochastic:
        q = 0
        for d in range(4):
            if not mask >> d & 1:
                continue
            if d < 2:
                w3[q, :, :, 0, :, 0] = 0
                w3[q, :, :, 2, :, W - 1] = 0
            else:
                w3[q, :, :, 0, 0, :] = 0
                w3[q, :, :, 2, H - 1, :] = 0
            q += 1
        w3 /= w3.sum(axis=3, keepdims=True)
    return x, w3, lam, u


def single_dir(d, H, W, B=1, C=1, G=1):
    """Zero-initialised single-direction operand set with lambda = u = 1."""
    x = np.zeros((B, C, H, W))
    lam = np.ones((1, B, C, H, W))
    u = np.ones((1, B, C, H, W))
    w3 = np.zeros((1, B, G, 3, H, W))
    return x, w3, lam, u


def dense_G(d, w3p, lamp, H, W):
    """Eq. (4): G_{s,t} = (prod_{tau=t+1..s} w_tau) Lambda_t as a dense
    (Ls*Lp) x (Ls*Lp) matrix acting on the scan-ordered vector of one plane."""
    Ls, Lp = dims(d, H, W)
    ws, Lams = [], []
    for s in range(Ls):
        m = np.zeros((Lp, Lp))
        lam_s = np.zeros(Lp)
        for p in range(Lp):
            i, j = img_index(d, s, p, H, W)
            lam_s[p] = lamp[i, j]
            for k in range(3):
                pn = p + k - 1
                if 0 <= pn < Lp:
                    m[p, pn] = w3p[k, i, j]
        ws.append(m)
        Lams.append(np.diag(lam_s))
    Gm = np.zeros((Ls * Lp, Ls * Lp))
    for s in range(Ls):
        for t in range(s + 1):
            prod = np.eye(Lp)
            for tau in range(t + 1, s + 1):
                prod = ws[tau] @ prod
            Gm[s * Lp:(s + 1) * Lp, t * Lp:(t + 1) * Lp] = prod @ Lams[t]
    return Gm, ws


def to_scan_vec(d, a, H, W):
    Ls, Lp = dims(d, H, W)
    v = np.zeros(Ls * Lp)
    for s in range(Ls):
        for p in range(Lp):
            v[s * Lp + p] = a[img_index(d, s, p, H, W)]
    return v


def from_scan_vec(d, v, H, W):
    Ls, Lp = dims(d, H, W)
    a = np.zeros((H, W))
    for s in range(Ls):
        for p in range(Lp):
            a[img_index(d, s, p, H, W)] = v[s * Lp + p]
    return a


# ----------------------------------------------------------------------------- forward pins
def read_trinomial():
    rows = []
    with open(os.path.join(GOLD, "trinomial_triangle.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            rows.append([int(t) for t in line.split()])
    return rows


def test_golden_trinomial_matches_polynomial_expansion():
    rows = read_trinomial()
    for t, row in enumerate(rows):
        coef = np.polynomial.polynomial.polypow([1, 1, 1], t)
        assert [int(round(c)) for c in coef] == row


@pytest.mark.parametrize("d", [0, 1, 2, 3])
def test_delta_response_is_trinomial(d):
    """lambda=u=1, x=delta on the first scan line, taps 1/3: h[t, p0+s] = T(t,s)/3^t."""
    rows = read_trinomial()
    steps = len(rows)
    H, W = (steps, 2 * steps + 3) if d < 2 else (2 * steps + 3, steps)
    Ls, Lp = dims(d, H, W)
    p0 = Lp // 2
    x, w3, lam, u = single_dir(d, H, W)
    w3[:] = 1.0 / 3.0
    x[0, 0][img_index(d, 0, p0, H, W)] = 1.0
    y = orc.fwd(x, w3, lam, u, 1, DIRS[d])
    for t, row in enumerate(rows):
        half = len(row) // 2
        for s_off, coef in zip(range(-half, half + 1), row):
            got = y[0, 0][img_index(d, t, p0 + s_off, H, W)]
            assert got == pytest.approx(coef / 3.0 ** t, rel=1e-14, abs=0)
        # outside the cone the response is exactly zero
        for p in range(Lp):
            if abs(p - p0) > half:
                assert y[0, 0][img_index(d, t, p, H, W)] == 0.0


@pytest.mark.parametrize("d", [0, 1, 2, 3])
def test_constant_lines_accumulate(d):
    """Row-stochastic taps (edges renormalised) and lambda*x constant along each scan
    line s (= c_s) give h[s,:] = sum_{s'<=s} c_s' for ANY taps."""
    rng = np.random.default_rng(7)
    H, W = 6, 9
    x, w3, lam, u = rand_problem(rng, 1, 2, H, W, 1, DIRS[d])
    Ls, Lp = dims(d, H, W)
    c = rng.uniform(-1, 1, Ls)
    lam[:] = 0.25
    u[:] = 1.0
    for s in range(Ls):
        for p in range(Lp):
            x[0, :, *img_index(d, s, p, H, W)] = c[s] / 0.25
    y = orc.fwd(x, w3, lam, u, 1, DIRS[d])
    for s in range(Ls):
        for p in range(Lp):
            assert y[0, 1][img_index(d, s, p, H, W)] == pytest.approx(c[:s + 1].sum(), abs=1e-13)


@pytest.mark.parametrize("d", [0, 1, 2, 3])
def test_centre_tap_only_is_prefix_sum_and_iir(d):
    """w0=1: h = cumulative sum of lambda*x along the scan (numpy.cumsum);
    w0=a: first-order IIR (scipy.signal.lfilter)."""
    rng = np.random.default_rng(3)
    H, W = 7, 5
    x, w3, lam, u = single_dir(d, H, W, C=2)
    x[:] = rng.standard_normal(x.shape)
    lam[:] = rng.uniform(0.2, 1, lam.shape)
    for a in (1.0, 0.6):
        w3[:] = 0
        w3[:, :, :, 1] = a
        y = orc.fwd(x, w3, lam, u, 1, DIRS[d])
        lx = (lam[0] * x)[0]                       # [C,H,W]
        axis = 1 if d < 2 else 2
        if d in (1, 3):
            lx = np.flip(lx, axis=axis)
        ref = np.cumsum(lx, axis=axis) if a == 1.0 else lfilter([1.0], [1.0, -a], lx, axis=axis)
        if d in (1, 3):
            ref = np.flip(ref, axis=axis)
        np.testing.assert_allclose(y[0], ref, rtol=1e-13, atol=1e-13)


@pytest.mark.parametrize("d", [0, 1, 2, 3])
@pytest.mark.parametrize("k", [0, 2])
def test_single_side_tap_is_diagonal_sum(d, k):
    """Only tap k (weight 1): h[s,p] = sum_t (lambda x)[s-t, p + t*(k-1)] -- pins which
    of w-/w+ looks at p-1/p+1 and the orientation of every direction."""
    rng = np.random.default_rng(11)
    H, W = 5, 6
    x, w3, lam, u = single_dir(d, H, W)
    x[:] = rng.standard_normal(x.shape)
    w3[:, :, :, k] = 1.0
    y = orc.fwd(x, w3, lam, u, 1, DIRS[d])
    Ls, Lp = dims(d, H, W)
    for s in range(Ls):
        for p in range(Lp):
            ref = 0.0
            for t in range(s + 1):
                pp = p + t * (k - 1)
                if 0 <= pp < Lp:
                    ref += x[0, 0][img_index(d, s - t, pp, H, W)]
            assert y[0, 0][img_index(d, s, p, H, W)] == pytest.approx(ref, abs=1e-13)


@pytest.mark.parametrize("HW", [(4, 4), (3, 5), (5, 2), (1, 4), (4, 1)])
@pytest.mark.parametrize("d", [0, 1, 2, 3])
def test_dense_matrix_brute_force(d, HW):
    """h = G x with G of Eq. (4) built from dense Lp x Lp matrices."""
    H, W = HW
    rng = np.random.default_rng(100 + d)
    x, w3, lam, u = rand_problem(rng, 1, 2, H, W, 2, DIRS[d], stochastic=False)
    y, h = orc.fwd(x, w3, lam, u, 2, DIRS[d], return_h=True)
    for c in range(2):
        Gm, _ = dense_G(d, w3[0, 0, c], lam[0, 0, c], H, W)
        href = from_scan_vec(d, Gm @ to_scan_vec(d, x[0, c], H, W), H, W)
        np.testing.assert_allclose(h[0, 0, c], href, rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(y[0, c], u[0, 0, c] * href, rtol=1e-12, atol=1e-12)


def test_h0_enters_through_first_step_weights():
    """h_0 = w_0 h_{-1} + lambda_0 x_0 with h_{-1} = h0 (reading R1)."""
    rng = np.random.default_rng(5)
    H, W = 4, 6
    for d in range(4):
        x, w3, lam, u = rand_problem(rng, 1, 1, H, W, 1, DIRS[d])
        Ls, Lp = dims(d, H, W)
        h0 = np.zeros((1, 1, 1, max(H, W)))
        h0[0, 0, 0, :Lp] = rng.standard_normal(Lp)
        _, h = orc.fwd(x, w3, lam, u, 1, DIRS[d], h0=h0, return_h=True)
        _, ws = dense_G(d, w3[0, 0, 0], lam[0, 0, 0], H, W)
        for p in range(Lp):
            i, j = img_index(d, 0, p, H, W)
            ref = ws[0][p] @ h0[0, 0, 0, :Lp] + lam[0, 0, 0, i, j] * x[0, 0, i, j]
            assert h[0, 0, 0, i, j] == pytest.approx(ref, abs=1e-13)
        # and by linearity the rest of the response to h0 alone is prod(w) h0
        x0 = np.zeros_like(x)
        _, hh = orc.fwd(x0, w3, lam, u, 1, DIRS[d], h0=h0, return_h=True)
        v = h0[0, 0, 0, :Lp].copy()
        for s in range(Ls):
            v = ws[s] @ v
            for p in range(Lp):
                assert hh[0, 0, 0][img_index(d, s, p, H, W)] == pytest.approx(v[p], abs=1e-13)


def test_direction_symmetries():
    """scan_d = P_d^-1 o scan_TB o P_d with P_d a flip / transpose of every tensor."""
    rng = np.random.default_rng(9)
    B, C, H, W, G = 2, 4, 5, 7, 2

    def P(d, a):        # maps image-layout tensor of direction d onto the T->B problem
        if d == 0:
            return a
        if d == 1:
            return np.flip(a, axis=-2)
        if d == 2:
            return np.swapaxes(a, -1, -2)
        return np.flip(np.swapaxes(a, -1, -2), axis=-2)

    def Pinv(d, a):
        if d == 0:
            return a
        if d == 1:
            return np.flip(a, axis=-2)
        if d == 2:
            return np.swapaxes(a, -1, -2)
        return np.swapaxes(np.flip(a, axis=-2), -1, -2)

    for d in range(1, 4):
        x, w3, lam, u = rand_problem(rng, B, C, H, W, G, DIRS[d])
        y = orc.fwd(x, w3, lam, u, G, DIRS[d])
        yt = orc.fwd(np.ascontiguousarray(P(d, x)), np.ascontiguousarray(P(d, w3)),
                     np.ascontiguousarray(P(d, lam)), np.ascontiguousarray(P(d, u)), G, 1)
        np.testing.assert_allclose(y, Pinv(d, yt), rtol=0, atol=1e-13)


def test_four_direction_output_is_sum_of_single_directions():
    rng = np.random.default_rng(21)
    B, C, H, W, G = 2, 6, 5, 4, 3
    for mask in (15, 5, 10, 6, 9, 14):
        x, w3, lam, u = rand_problem(rng, B, C, H, W, G, mask)
        y = orc.fwd(x, w3, lam, u, G, mask)
        acc = np.zeros_like(y)
        q = 0
        for d in range(4):
            if mask >> d & 1:
                acc += orc.fwd(x, w3[q:q + 1], lam[q:q + 1], u[q:q + 1], G, DIRS[d])
                q += 1
        np.testing.assert_allclose(y, acc, rtol=0, atol=1e-13)


def test_group_sharing_equals_replicated_taps():
    """Eq. (5): G<C equals G=C with each group's taps replicated."""
    rng = np.random.default_rng(2)
    B, C, H, W, G = 2, 6, 4, 5, 2
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, 15)
    y = orc.fwd(x, w3, lam, u, G, 15)
    w3_full = np.repeat(w3, C // G, axis=2)
    y_full = orc.fwd(x, w3_full, lam, u, C, 15)
    np.testing.assert_array_equal(y, y_full)
    dy = rng.standard_normal(x.shape)
    g = orc.bwd(x, w3, lam, u, dy, G, 15)
    gf = orc.bwd(x, w3_full, lam, u, dy, C, 15)
    np.testing.assert_allclose(g["dx"], gf["dx"], atol=1e-13)
    D = 4
    dw_sum = gf["dw3"].reshape(D, B, G, C // G, 3, H, W).sum(axis=3)
    np.testing.assert_allclose(g["dw3"], dw_sum, atol=1e-12)


def test_stability_bound():
    """Row-stochastic non-negative taps, |x|<=M: |h[s,p]| <= M sum_{s'<=s} max_p lambda[s',p]
    (Stability-Context condition)."""
    rng = np.random.default_rng(4)
    B, C, H, W, G = 1, 3, 12, 9, 1
    for d in range(4):
        x, w3, lam, u = rand_problem(rng, B, C, H, W, G, DIRS[d])
        x = rng.uniform(-2.0, 2.0, x.shape)
        _, h = orc.fwd(x, w3, lam, u, G, DIRS[d], return_h=True)
        Ls, Lp = dims(d, H, W)
        for c in range(C):
            bound = 0.0
            for s in range(Ls):
                bound += max(lam[0, 0, c][img_index(d, s, p, H, W)] for p in range(Lp))
                for p in range(Lp):
                    assert abs(h[0, 0, c][img_index(d, s, p, H, W)]) <= 2.0 * bound + 1e-12


def test_linearity_in_x():
    rng = np.random.default_rng(6)
    x, w3, lam, u = rand_problem(rng, 1, 2, 6, 5, 1, 15)
    x2 = rng.standard_normal(x.shape)
    y1 = orc.fwd(x, w3, lam, u, 1, 15)
    y2 = orc.fwd(x2, w3, lam, u, 1, 15)
    y12 = orc.fwd(2.0 * x - 3.0 * x2, w3, lam, u, 1, 15)
    np.testing.assert_allclose(y12, 2.0 * y1 - 3.0 * y2, atol=1e-12)


def test_invalid_arguments_are_rejected():
    rng = np.random.default_rng(1)
    x, w3, lam, u = rand_problem(rng, 1, 4, 3, 3, 2, 1)
    with pytest.raises(ValueError):
        orc.fwd(x, np.zeros((1, 1, 3, 3, 3, 3)), lam, u, 3, 1)      # C % G != 0


# ----------------------------------------------------------------------------- backward pins
def _loss(x, w3, lam, u, h0, dy, G, mask):
    return float((orc.fwd(x, w3, lam, u, G, mask, h0=h0) * dy).sum())


@pytest.mark.parametrize("shape", [(1, 4, 8, 8, 2), (2, 2, 5, 7, 1), (1, 3, 3, 1, 3), (1, 2, 1, 4, 2)])
def test_backward_matches_central_finite_differences(shape):
    B, C, H, W, G = shape
    mask = 15
    rng = np.random.default_rng(17)
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, mask, stochastic=False)
    h0 = rng.standard_normal((4, B, C, max(H, W)))
    dy = rng.standard_normal(x.shape)
    g = orc.bwd(x, w3, lam, u, dy, G, mask, h0=h0)
    eps = 1e-6
    ops = {"dx": x, "dw3": w3, "dlambda": lam, "du": u, "dh0": h0}
    for name, arr in ops.items():
        flat = arr.reshape(-1)
        gflat = g[name].reshape(-1)
        idxs = rng.choice(flat.size, size=min(40, flat.size), replace=False)
        for idx in idxs:
            if name == "dh0":
                # entries past the direction's cross length are unused: gradient 0
                q, rem = divmod(idx, B * C * max(H, W))
                p = rem % max(H, W)
                d = [dd for dd in range(4) if mask >> dd & 1][q]
                if p >= dims(d, H, W)[1]:
                    assert gflat[idx] == 0.0
                    continue
            if name == "dw3":
                # out-of-grid taps are never read: gradient 0
                q, rem = divmod(idx, B * G * 3 * H * W)
                k = (rem // (H * W)) % 3
                i, j = divmod(rem % (H * W), W)
                d = [dd for dd in range(4) if mask >> dd & 1][q]
                p = j if d < 2 else i
                Lp = dims(d, H, W)[1]
                if (k == 0 and p == 0) or (k == 2 and p == Lp - 1):
                    assert gflat[idx] == 0.0
                    continue
            old = flat[idx]
            flat[idx] = old + eps
            lp = _loss(x, w3, lam, u, h0, dy, G, mask)
            flat[idx] = old - eps
            lm = _loss(x, w3, lam, u, h0, dy, G, mask)
            flat[idx] = old
            fd = (lp - lm) / (2 * eps)
            assert gflat[idx] == pytest.approx(fd, rel=2e-6, abs=2e-7), (name, idx)


def test_adjoint_identity():
    """<scan(v), dy> = <v, dx(dy)> to rounding (the scan is linear in x)."""
    rng = np.random.default_rng(23)
    B, C, H, W, G = 2, 4, 9, 6, 2
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, 15)
    dy = rng.standard_normal(x.shape)
    v = rng.standard_normal(x.shape)
    g = orc.bwd(x, w3, lam, u, dy, G, 15)
    lhs = float((orc.fwd(v, w3, lam, u, G, 15) * dy).sum())
    rhs = float((v * g["dx"]).sum())
    assert lhs == pytest.approx(rhs, rel=1e-13)


@pytest.mark.parametrize("d", [0, 1, 2, 3])
def test_backward_dense_transpose(d):
    """dx = G^T (u * dy), du = dy * (G x) with the dense G of Eq. (4)."""
    rng = np.random.default_rng(31 + d)
    H, W = 4, 3
    x, w3, lam, u = rand_problem(rng, 1, 1, H, W, 1, DIRS[d], stochastic=False)
    dy = rng.standard_normal(x.shape)
    g = orc.bwd(x, w3, lam, u, dy, 1, DIRS[d])
    Gm, _ = dense_G(d, w3[0, 0, 0], lam[0, 0, 0], H, W)
    gy = to_scan_vec(d, (u[0, 0, 0] * dy[0, 0]), H, W)
    np.testing.assert_allclose(g["dx"][0, 0], from_scan_vec(d, Gm.T @ gy, H, W), atol=1e-12)
    hv = Gm @ to_scan_vec(d, x[0, 0], H, W)
    np.testing.assert_allclose(g["du"][0, 0, 0], dy[0, 0] * from_scan_vec(d, hv, H, W), atol=1e-12)


def test_magnitude_run_dominates():
    rng = np.random.default_rng(8)
    x, w3, lam, u = rand_problem(rng, 1, 4, 6, 6, 2, 15)
    dy = rng.standard_normal(x.shape)
    y = orc.fwd(x, w3, lam, u, 2, 15)
    A = orc.fwd_magnitude(x, w3, lam, u, 2, 15)
    assert np.all(A >= np.abs(y) - 1e-12)
    g = orc.bwd(x, w3, lam, u, dy, 2, 15)
    Ag = orc.bwd_magnitude(x, w3, lam, u, dy, 2, 15)
    for k in g:
        assert np.all(Ag[k] >= np.abs(g[k]) - 1e-12)


# ----------------------------------------------------------------------------- merge, float build
def test_merge_matches_einsum():
    rng = np.random.default_rng(12)
    yd = rng.standard_normal((3, 2, 5, 4, 6))
    m = rng.standard_normal((3, 5))
    np.testing.assert_allclose(orc.merge(yd, m), np.einsum("qc,qbchw->bchw", m, yd), atol=1e-13)
    np.testing.assert_allclose(orc.merge(yd), yd.sum(axis=0), atol=1e-13)


def test_float_build_tracks_double_build():
    """The pinned-order float build stays within 1e-5 of the magnitude scale of the
    double build (the fp32 gate of DESIGN.md is attainable)."""
    rng = np.random.default_rng(13)
    B, C, H, W, G = 2, 8, 40, 33, 2
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, 15)
    xs, ws, ls, us = (a.astype(np.float32) for a in (x, w3, lam, u))
    y64 = orc.fwd(xs.astype(np.float64), ws.astype(np.float64), ls.astype(np.float64),
                  us.astype(np.float64), G, 15)
    A = orc.fwd_magnitude(xs, ws, ls, us, G, 15)
    y32 = orc.fwd(xs, ws, ls, us, G, 15)
    assert y32.dtype == np.float32
    assert np.all(np.abs(y32 - y64) <= np.maximum(1e-5 * A, 1e-6))


# ----------------------------------------------------------------------------- Eq. (3) normalisation
def _in_grid(d, k, i, j, H, W):
    """Tap k of pixel (i,j) has its neighbour inside the grid -- written independently of the oracle."""
    p, L = (j, W) if d < 2 else (i, H)
    return not ((k == 0 and p == 0) or (k == 2 and p == L - 1))


def test_normalize_rows_are_stochastic_and_edges_masked():
    """Eq. (3): nonnegative, rows sum to one over N(j), out-of-grid taps are exactly 0
    (vertical directions mask along j, horizontal ones along i)."""
    rng = np.random.default_rng(30)
    H, W = 5, 7
    wt = rng.normal(0, 2, (4, 2, 3, 3, H, W))
    w = orc.normalize(wt, 15)
    assert np.all(w >= 0)
    np.testing.assert_allclose(w.sum(axis=3), 1.0, atol=1e-14)
    for d in range(4):
        for k in range(3):
            for i in range(H):
                for j in range(W):
                    if not _in_grid(d, k, i, j, H, W):
                        assert np.all(w[d, :, :, k, i, j] == 0.0)
                    else:
                        assert np.all(w[d, :, :, k, i, j] > 0.0)


def test_normalize_equal_logits_closed_form():
    """Equal logits: every in-grid tap gets 1/|N(j)| (1/3 inside, 1/2 on an edge, 1 on a line of one)."""
    for H, W in ((4, 6), (1, 5), (5, 1), (1, 1)):
        for c in (-3.0, 0.0, 2.5):
            w = orc.normalize(np.full((4, 1, 1, 3, H, W), c), 15)
            for d in range(4):
                for i in range(H):
                    for j in range(W):
                        n = sum(_in_grid(d, k, i, j, H, W) for k in range(3))
                        for k in range(3):
                            exp = 1.0 / n if _in_grid(d, k, i, j, H, W) else 0.0
                            assert abs(w[d, 0, 0, k, i, j] - exp) < 1e-15


def test_normalize_ratio_identity_with_library_softplus():
    """log(w_k / w_k') = log sigmoid(a_k) - log sigmoid(a_k') = softplus(-a_k') - softplus(-a_k):
    numpy's logaddexp gives the right-hand side without forming a sigmoid or a sum."""
    rng = np.random.default_rng(31)
    wt = rng.normal(0, 3, (1, 2, 2, 3, 6, 6))
    w = orc.normalize(wt, 1)
    inner = (slice(None),) * 3
    lhs = np.log(w[inner + (0, slice(None), slice(1, 5))] / w[inner + (2, slice(None), slice(1, 5))])
    a0 = wt[inner + (0, slice(None), slice(1, 5))]
    a2 = wt[inner + (2, slice(None), slice(1, 5))]
    rhs = np.logaddexp(0.0, -a2) - np.logaddexp(0.0, -a0)
    np.testing.assert_allclose(lhs, rhs, atol=1e-12)


def test_normalize_two_tap_edge_is_a_logistic_of_softplus_difference():
    """On an edge N(j) has two taps: w_1 = 1 / (1 + sigmoid(a_2)/sigmoid(a_1)) = expit(softplus(-a_2) - softplus(-a_1))
    with scipy's expit as the library routine."""
    from scipy.special import expit
    rng = np.random.default_rng(32)
    wt = rng.normal(0, 2, (1, 1, 1, 3, 4, 5))
    w = orc.normalize(wt, 1)                      # T->B: column 0 has no k=0 neighbour
    a1, a2 = wt[0, 0, 0, 1, :, 0], wt[0, 0, 0, 2, :, 0]
    np.testing.assert_allclose(w[0, 0, 0, 1, :, 0], expit(np.logaddexp(0, -a2) - np.logaddexp(0, -a1)), atol=1e-14)


def test_normalize_clamp_branch_constant():
    """All logits -40: S = 3*sigmoid(-40) = 1.27e-17 < eps = 1e-6, so w_k = sigmoid(-40)/eps.
    sigmoid(-40) = e^-40/(1+e^-40) = 4.248354255291589e-18 (e^-40 to 16 digits)."""
    w = orc.normalize(np.full((1, 1, 1, 3, 3, 3), -40.0), 1)
    np.testing.assert_allclose(w[0, 0, 0, :, 1, 1], 4.248354255291589e-12, rtol=1e-12)
    assert w[0, 0, 0, 0, 1, 0] == 0.0             # masking still applies under the clamp


@pytest.mark.parametrize("mask", [1, 4, 15, 10])
def test_normalize_bwd_finite_differences(mask):
    """Central differences in fp64 of <dw3, normalize(wt)> against the adjoint, clamp inactive."""
    rng = np.random.default_rng(33 + mask)
    D = orc.popcount(mask)
    wt = rng.normal(0, 1.5, (D, 1, 2, 3, 4, 5))
    dw = rng.standard_normal(wt.shape)
    g = orc.normalize_bwd(wt, dw, mask)
    eps = 1e-6
    idx = [tuple(rng.integers(0, n) for n in wt.shape) for _ in range(60)]
    for ix in idx:
        p, m = wt.copy(), wt.copy()
        p[ix] += eps; m[ix] -= eps
        fd = float(np.sum(dw * (orc.normalize(p, mask) - orc.normalize(m, mask)))) / (2 * eps)
        assert abs(fd - g[ix]) <= 1e-8 + 1e-6 * abs(fd), (ix, fd, g[ix])


def test_normalize_bwd_clamp_branch_and_invariants():
    """(a) clamp active: the denominator is the constant eps, so dwt_k = s_k(1-s_k) dw_k / eps -- checked by
    finite differences; (b) clamp inactive: rows of w sum to one, so a constant added to dw over N(j) changes
    nothing; (c) out-of-grid taps get no gradient."""
    rng = np.random.default_rng(35)
    wt = np.full((1, 1, 1, 3, 3, 4), -40.0) + rng.normal(0, 0.1, (1, 1, 1, 3, 3, 4))
    dw = rng.standard_normal(wt.shape)
    g = orc.normalize_bwd(wt, dw, 1)
    for ix in [(0, 0, 0, 1, 1, 1), (0, 0, 0, 0, 2, 2), (0, 0, 0, 2, 0, 1)]:
        p, m = wt.copy(), wt.copy()
        p[ix] += 1e-4; m[ix] -= 1e-4
        fd = float(np.sum(dw * (orc.normalize(p, 1) - orc.normalize(m, 1)))) / 2e-4
        assert abs(fd - g[ix]) <= 1e-6 * abs(fd) + 1e-30
    wt = rng.normal(0, 1, (2, 1, 2, 3, 4, 5))
    dw = rng.standard_normal(wt.shape)
    g0 = orc.normalize_bwd(wt, dw, 5)
    g1 = orc.normalize_bwd(wt, dw + 3.25, 5)
    np.testing.assert_allclose(g0, g1, atol=1e-13)
    assert np.all(g0[0, :, :, 0, :, 0] == 0) and np.all(g0[0, :, :, 2, :, -1] == 0)      # T->B: along j
    assert np.all(g0[1, :, :, 0, 0, :] == 0) and np.all(g0[1, :, :, 2, -1, :] == 0)      # L->R: along i


def test_normalized_taps_feed_the_scan_stably():
    """Eq. (3) output used as w3: the stability bound of PAPER.md:94 holds (|h| <= M * sum of lambda maxima)."""
    rng = np.random.default_rng(36)
    B, C, H, W, G = 1, 4, 9, 8, 2
    w3 = orc.normalize(rng.normal(0, 2, (4, B, G, 3, H, W)), 15)
    x = rng.uniform(-1, 1, (B, C, H, W))
    lam = rng.uniform(0, 1, (4, B, C, H, W))
    y, h = orc.fwd(x, w3, lam, np.ones_like(lam), G, 15, return_h=True)
    for q in range(4):
        Ls = H if q < 2 else W
        bound = lam[q].max() * Ls
        assert np.all(np.abs(h[q]) <= bound + 1e-12)


def test_normalize_bwd_magnitude_closed_form_and_dominance():
    """Magnitude mode of the Eq. (3) adjoint (the scale A of the normalize_bwd gate, tests/parity_util.py).
    Closed form at an interior pixel with equal logits a and dw = (1, 0, 0): s = sigmoid(a), S = 3s, w_k = 1/3, so
    the plain adjoint is (1-s)*(1 - 1/3)/3 = (1-s)*2/9 for k = 0 and -(1-s)/9 for k = 1, 2, while the sum of the
    absolute values of the same terms is (1-s)*(1 + 1/3)/3 = (1-s)*4/9 and (1-s)/9."""
    for a in (-1.5, 0.0, 0.7):
        wt = np.full((1, 1, 1, 3, 3, 3), a)
        dw = np.zeros_like(wt)
        dw[0, 0, 0, 0, 1, 1] = 1.0
        s = 1.0 / (1.0 + math.exp(-a))
        g = orc.normalize_bwd(wt, dw, 1)[0, 0, 0, :, 1, 1]
        m = orc.normalize_bwd(wt, dw, 1, magnitude=True)[0, 0, 0, :, 1, 1]
        np.testing.assert_allclose(g, [(1 - s) * 2 / 9, -(1 - s) / 9, -(1 - s) / 9], rtol=1e-13)
        np.testing.assert_allclose(m, [(1 - s) * 4 / 9, (1 - s) / 9, (1 - s) / 9], rtol=1e-13)
    rng = np.random.default_rng(41)
    wt = rng.normal(0, 2, (4, 2, 2, 3, 5, 6))
    dw = rng.standard_normal(wt.shape)
    g = orc.normalize_bwd(wt, dw, 15)
    m = orc.normalize_bwd(wt, dw, 15, magnitude=True)
    assert np.all(m >= np.abs(g) - 1e-15) and np.all(m >= 0)
    # the sign of dw does not matter to the magnitude; it is linear under positive scaling
    np.testing.assert_allclose(orc.normalize_bwd(wt, -dw, 15, magnitude=True), m, rtol=1e-14)
    np.testing.assert_allclose(orc.normalize_bwd(wt, 2.5 * dw, 15, magnitude=True), 2.5 * m, rtol=1e-13)
    # one nonzero tap gradient per pixel: the in-bracket terms dw_k and -dw_k w_k have opposite signs for tap k (so the
    # magnitude is |dw_k|(1 + w_k) against |dw_k|(1 - w_k)) and a single term for the other taps (magnitude = |value|)
    one = np.zeros_like(dw)
    one[:, :, :, 1] = dw[:, :, :, 1]
    g1 = orc.normalize_bwd(wt, one, 15)
    m1 = orc.normalize_bwd(wt, one, 15, magnitude=True)
    w = orc.normalize(wt, 15)
    np.testing.assert_allclose(m1[:, :, :, 0], np.abs(g1[:, :, :, 0]), rtol=1e-12, atol=1e-300)
    np.testing.assert_allclose(m1[:, :, :, 2], np.abs(g1[:, :, :, 2]), rtol=1e-12, atol=1e-300)
    np.testing.assert_allclose(m1[:, :, :, 1] * (1 - w[:, :, :, 1]), np.abs(g1[:, :, :, 1]) * (1 + w[:, :, :, 1]),
                               rtol=1e-10, atol=1e-300)


def test_float_build_of_backward_tracks_double_build():
    """The pinned-order float build of the adjoint (the timed cpu_baseline) stays within 1e-5 of the magnitude
    scale of the double build on every gradient."""
    rng = np.random.default_rng(42)
    B, C, H, W, G = 2, 8, 31, 26, 2
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, 15)
    dy = rng.standard_normal(x.shape)
    h0 = rng.standard_normal((4, B, C, max(H, W)))
    s = [a.astype(np.float32) for a in (x, w3, lam, u, dy, h0)]
    d = [a.astype(np.float64) for a in s]
    g64 = orc.bwd(d[0], d[1], d[2], d[3], d[4], G, 15, h0=d[5])
    A = orc.bwd_magnitude(d[0], d[1], d[2], d[3], d[4], G, 15, h0=d[5])
    g32 = orc.bwd(s[0], s[1], s[2], s[3], s[4], G, 15, h0=s[5])
    for k in ("dx", "dlambda", "du", "dw3", "dh0"):
        assert g32[k].dtype == np.float32
        assert np.all(np.abs(g32[k] - g64[k]) <= np.maximum(1e-5 * A[k], 1e-6)), k


@pytest.mark.parametrize("mask", [15, 6, 9])
def test_out_of_grid_taps_are_never_read_by_the_oracle(mask):
    """DESIGN.md reading 3 / include/gspn.h: the tap of a neighbour outside the grid is never used.  What a slab
    SHARED by every direction (gspn_args_t.dir_stride_* = 0, reading 6) relies on: a tap that is in the grid for a
    vertical scan lies outside it for a horizontal one and must then count as absent, whatever it holds.  NaN in every
    out-of-grid tap changes no output; the dw3 entries of those taps are exactly 0."""
    rng = np.random.default_rng(77)
    B, C, H, W, G = 2, 4, 6, 9, 2
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, mask)
    dy = rng.standard_normal(x.shape)
    bad = w3.copy()
    out = np.zeros(w3.shape, bool)
    for q, d in enumerate(dd for dd in range(4) if mask >> dd & 1):
        if d < 2:
            out[q, :, :, 0, :, 0] = True; out[q, :, :, 2, :, W - 1] = True
        else:
            out[q, :, :, 0, 0, :] = True; out[q, :, :, 2, H - 1, :] = True
    bad[out] = np.nan
    np.testing.assert_array_equal(orc.fwd(x, bad, lam, u, G, mask), orc.fwd(x, w3, lam, u, G, mask))
    g0, g1 = orc.bwd(x, w3, lam, u, dy, G, mask), orc.bwd(x, bad, lam, u, dy, G, mask)
    for k in g0:
        np.testing.assert_array_equal(g1[k], g0[k], err_msg=k)
    assert np.all(g1["dw3"][out] == 0.0)
    # one slab replicated over the directions: its in-grid taps for one axis are out-of-grid taps for the other, so the
    # result equals the one with those taps zeroed per direction
    D = orc.popcount(mask)
    rep = np.repeat(w3[:1], D, axis=0)
    zeroed = rep.copy(); zeroed[out] = 0.0
    np.testing.assert_array_equal(orc.fwd(x, rep, lam, u, G, mask), orc.fwd(x, zeroed, lam, u, G, mask))
