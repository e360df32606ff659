"""Lane-level numpy model of the data flow of the line kernels (csrc/gspn_line_fwd.cu, gspn_line_bwd.cu) against the
oracle.  It is NOT the kernel: it restates, with 32 lanes as an array axis, the ownership maps, stage geometry, TMA
box clipping, tensor-memory layouts, the in-place turn between them, the checkpoint / recompute schedule, the
neighbour exchanges with their boundary rules and the fixed-order dw3 reduction the kernels rely on, so that an index or
boundary mistake in the DESIGN shows on a machine without a GPU.  (Written in round 2 after GPU access had closed.)
"""
import numpy as np
import pytest

from oracle import gspn_oracle as orc

S = 8          # scan steps per stage (kLineSteps)


def P_of(L):
    return 1 if L <= 32 else 2 if L <= 64 else 4


def box_rows(plane, s0):
    """TMA row box: rows s0 .. s0+S-1 of plane [H, W]; rows outside the tensor arrive as zeros."""
    H = plane.shape[0]
    out = np.zeros((S,) + plane.shape[1:], plane.dtype)
    lo, hi = max(s0, 0), min(s0 + S, H)
    if hi > lo:
        out[lo - s0:hi - s0] = plane[lo:hi]
    return out


def store_rows(plane, stage, s0):
    """TMA store of a row box: the part outside the tensor is not written."""
    H = plane.shape[0]
    lo, hi = max(s0, 0), min(s0 + S, H)
    if hi > lo:
        plane[lo:hi] = stage[lo - s0:hi - s0]


def shfl_up(v):        # lane a receives lane a-1 (lane 0 keeps its own value)
    o = v.copy(); o[1:] = v[:-1]; return o


def shfl_dn(v):
    o = v.copy(); o[:-1] = v[1:]; return o


def nbr_rows(v, H):
    """Row-owner layout (lane b owns rows b + 32k): v[lane, k] -> (value at row-1, value at row+1), 0 outside."""
    P = v.shape[1]
    lane = np.arange(32)
    up = np.zeros_like(v); dn = np.zeros_like(v)
    for k in range(P):
        su = v[:, k].copy()
        if k > 0:
            su[31] = v[31, k - 1]
        sd = v[:, k].copy()
        if k < P - 1:
            sd[0] = v[0, k + 1]
        up[:, k] = su[(lane + 31) % 32]
        dn[:, k] = sd[(lane + 1) % 32]
        if k == 0:
            up[0, k] = 0.0
        dn[lane + 32 * k >= H - 1, k] = 0.0
    return up, dn


class Tmem:
    """One channel's lane quarter: [32 lanes, columns]."""
    def __init__(self, cols):
        self.m = np.full((32, cols), np.nan)

    def transpose(self, H, W, P):
        """line_transpose: column-owner (pixel (i, P a + k) at lane a, column i P + k) -> row-owner (pixel (b + 32 t, j)
        at lane b, column t 32 P + j), 32 image rows at a time, in place."""
        WP = W // P
        for t in range((H + 31) // 32):
            tile = np.full((32, W), np.nan)
            for r8 in range(4):
                f = self.m[:, (32 * t + 8 * r8) * P:(32 * t + 8 * r8) * P + 8 * P].copy()      # [lane, r * P + k]
                for a in range(WP):
                    for r in range(8):
                        tile[8 * r8 + r, P * a:P * a + P] = f[a, r * P:r * P + P]
            for b in range(32):
                self.m[b, t * 32 * P:t * 32 * P + W] = tile[b]


# ------------------------------------------------------------------------------------------------ forward model
def model_fwd(x, w3, lam, u, G, mask):
    B, C, H, W = x.shape
    cg = C // G
    P = P_of(max(H, W))
    dirs = [d for d in range(4) if mask >> d & 1]
    y = np.zeros_like(x)
    for b in range(B):
        for c in range(C):
            g = c // cg
            tm = Tmem(((H + 31) // 32) * 32 * P)
            touched = False
            # ---- vertical pair: lane a owns columns P a + k
            hs = {0: np.zeros((32, P)), 1: np.zeros((32, P))}
            # the two directions of the pair meet at a barrier: first halves (stores), then second halves (adds)
            for phase, d in ((0, 0), (0, 1), (1, 0), (1, 1)):
                if d not in dirs:
                    continue
                q = dirs.index(d)
                both = 0 in dirs and 1 in dirs
                Hh = (H + 1) // 2
                first = (Hh if d == 0 else H - Hh) if both else H
                h = hs[d]
                WP = W // P
                for s in (range(0, first) if phase == 0 else range(first, H)):
                    blk, r = divmod(s, S)
                    s0 = H - (blk + 1) * S if d else blk * S
                    rl = S - 1 - r if d else r
                    i = H - 1 - s if d else s
                    st = {k: box_rows(w3[q, b, g, k], s0) for k in range(3)}
                    st[0][:, 0] = 0.0; st[2][:, W - 1] = 0.0                 # edge taps zeroed in the stage
                    sl, su_, sx = box_rows(lam[q, b, c], s0), box_rows(u[q, b, c], s0), box_rows(x[b, c], s0)

                    def own(a):          # [32, P] view of a stage row for the owning lanes (clamped beyond the line)
                        o = np.zeros((32, P))
                        for ln in range(32):
                            lp = ln if ln < WP else 0
                            o[ln] = a[rl, P * lp:P * lp + P]
                        return o
                    w0, w1, w2, la, uu, xx = own(st[0]), own(st[1]), own(st[2]), own(sl), own(su_), own(sx)
                    hl, hr = shfl_up(h[:, P - 1]), shfl_dn(h[:, 0])
                    hn = np.empty_like(h)
                    for k in range(P):
                        l = hl if k == 0 else h[:, k - 1]
                        rr = hr if k == P - 1 else h[:, k + 1]
                        hn[:, k] = w0[:, k] * l + w2[:, k] * rr + la[:, k] * xx[:, k] + w1[:, k] * h[:, k]
                    h = hn
                    acc = both and s >= first
                    col = slice(i * P, i * P + P)
                    tm.m[:, col] = (tm.m[:, col] if acc else 0.0) + uu * h
                hs[d] = h
                touched = True
            any_v = touched
            any_h = 2 in dirs or 3 in dirs
            if any_v and any_h:
                tm.transpose(H, W, P)
            # ---- horizontal pair: lane b owns rows b + 32k, stages of 2K columns (here: any stage width, column order only)
            hs = {0: np.zeros((32, P)), 1: np.zeros((32, P))}
            for phase, d in ((0, 0), (0, 1), (1, 0), (1, 1)):
                if 2 + d not in dirs:
                    continue
                q = dirs.index(2 + d)
                both = 2 in dirs and 3 in dirs
                Wh = (W // 2 + 3) // 4 * 4
                first = (Wh if d == 0 else W - Wh) if both else W
                h = hs[d]
                rows = np.arange(32)[:, None] + 32 * np.arange(P)[None, :]
                rc = np.where(rows < H, rows, 0)
                t0 = w3[q, b, g, 0].copy(); t0[0, :] = 0.0
                t2 = w3[q, b, g, 2].copy(); t2[H - 1, :] = 0.0
                for s in (range(0, first) if phase == 0 else range(first, W)):
                    j = W - 1 - s if d else s
                    up, dn = nbr_rows(h, H)
                    # the kernel's forward does not zero the neighbours (the taps are zeroed); the result is the same
                    h = t0[rc, j] * up + t2[rc, j] * dn + lam[q, b, c][rc, j] * x[b, c][rc, j] + w3[q, b, g, 1][rc, j] * h
                    acc = any_v or (both and s >= first)
                    for k in range(P):
                        if 32 * k >= H:
                            continue                     # slots past the plane own no tensor-memory columns
                        colk = k * 32 * P + j
                        tm.m[:, colk] = (tm.m[:, colk] if acc else 0.0) + u[q, b, c][rc[:, k], j] * h[:, k]
                hs[d] = h
            # ---- the plane leaves
            if any_h:
                for k in range(P):
                    for ln in range(32):
                        i = ln + 32 * k
                        if i < H:
                            y[b, c, i] = tm.m[ln, k * 32 * P:k * 32 * P + W]
            else:
                WP = W // P
                for i in range(H):
                    for a in range(WP):
                        y[b, c, i, P * a:P * a + P] = tm.m[a, i * P:i * P + P]
    return y


# ------------------------------------------------------------------------------------------------ backward model
def model_bwd(x, w3, lam, u, dy, G, mask, h0=None):
    B, C, H, W = x.shape
    cg = C // G
    L = max(H, W)
    P = P_of(L)
    dirs = [d for d in range(4) if mask >> d & 1]
    D = len(dirs)
    out = dict(dx=np.zeros_like(x), dlambda=np.zeros_like(lam), du=np.zeros_like(u), dw3=np.zeros_like(w3),
               dh0=np.zeros((D, B, C, L)))
    for b in range(B):
        for g in range(G):
            chans = list(range(g * cg, (g + 1) * cg))
            tms = [Tmem(((H + 31) // 32) * 32 * P) for _ in chans]
            acc = False
            any_v, any_h = bool(mask & 3), bool(mask & 12)
            for d in range(4):
                if d == 2 and any_v and any_h:
                    for tm in tms:
                        tm.transpose(H, W, P)
                if d not in dirs:
                    continue
                q = dirs.index(d)
                rev = d & 1
                if d < 2:
                    _bwd_dir_v(out, tms, x, w3, lam, u, dy, h0, b, g, chans, q, rev, acc, H, W, P)
                else:
                    _bwd_dir_h(out, tms, x, w3, lam, u, dy, h0, b, g, chans, q, rev, acc, H, W, P)
                acc = True
            for ci, c in enumerate(chans):
                tm = tms[ci]
                if any_h:
                    for k in range(P):
                        for ln in range(32):
                            i = ln + 32 * k
                            if i < H:
                                out["dx"][b, c, i] = tm.m[ln, k * 32 * P:k * 32 * P + W]
                else:
                    for i in range(H):
                        for a in range(W // P):
                            out["dx"][b, c, i, P * a:P * a + P] = tm.m[a, i * P:i * P + P]
    return out


def _bwd_dir_v(out, tms, x, w3, lam, u, dy, h0, b, g, chans, q, rev, acc, H, W, P):
    NC = len(chans)
    WP = W // P
    nblk = (H + S - 1) // S
    lanes = np.arange(32)
    active = lanes < WP
    first_lane, last_lane = lanes == 0, lanes == WP - 1

    def own(a, rl):
        o = np.zeros((32, P))
        for ln in range(32):
            lp = ln if ln < WP else 0
            o[ln] = a[rl, P * lp:P * lp + P]
        return o

    def stage(blk):
        s0 = H - (blk + 1) * S if rev else blk * S
        st = [box_rows(w3[q, b, g, k], s0) for k in range(3)]
        st[0][:, 0] = 0.0; st[2][:, W - 1] = 0.0
        return s0, st

    # pass 1: checkpoints
    ck = np.zeros((NC, nblk, 32, P))
    for ci, c in enumerate(chans):
        h = np.zeros((32, P))
        if h0 is not None:
            for ln in range(WP):
                h[ln] = h0[q, b, c, P * ln:P * ln + P]
        for blk in range(nblk):
            s0, st = stage(blk)
            sl, sx = box_rows(lam[q, b, c], s0), box_rows(x[b, c], s0)
            ck[ci, blk] = h
            nr = min(S, H - blk * S)
            for r in range(nr):
                rl = S - 1 - r if rev else r
                w0, w1, w2, la, xx = own(st[0], rl), own(st[1], rl), own(st[2], rl), own(sl, rl), own(sx, rl)
                hl, hr = shfl_up(h[:, P - 1]), shfl_dn(h[:, 0])
                hn = np.empty_like(h)
                for k in range(P):
                    l = hl if k == 0 else h[:, k - 1]
                    rr = hr if k == P - 1 else h[:, k + 1]
                    hn[:, k] = w0[:, k] * l + w2[:, k] * rr + la[:, k] * xx[:, k] + w1[:, k] * h[:, k]
                h = hn
    # pass 2
    carry = np.zeros((NC, 32, P))
    for blk in range(nblk - 1, -1, -1):
        s0, st = stage(blk)
        nr = min(S, H - blk * S)
        ops = []
        for ci, c in enumerate(chans):
            ops.append(dict(l=box_rows(lam[q, b, c], s0), x=box_rows(x[b, c], s0), u=box_rows(u[q, b, c], s0),
                            dy=box_rows(dy[b, c], s0)))
        hb = np.zeros((NC, S + 1, 32, P)); hls = np.zeros((NC, S, 32)); hrs = np.zeros((NC, S, 32))
        for ci in range(NC):
            hb[ci, 0] = ck[ci, blk]
            for r in range(nr):
                rl = S - 1 - r if rev else r
                w0, w1, w2 = own(st[0], rl), own(st[1], rl), own(st[2], rl)
                la, xx = own(ops[ci]["l"], rl), own(ops[ci]["x"], rl)
                hl, hr = shfl_up(hb[ci, r, :, P - 1]), shfl_dn(hb[ci, r, :, 0])
                hl[first_lane] = 0.0; hr[last_lane] = 0.0
                hls[ci, r], hrs[ci, r] = hl, hr
                for k in range(P):
                    l = hl if k == 0 else hb[ci, r, :, k - 1]
                    rr = hr if k == P - 1 else hb[ci, r, :, k + 1]
                    hb[ci, r + 1, :, k] = w0[:, k] * l + w2[:, k] * rr + la[:, k] * xx[:, k] + w1[:, k] * hb[ci, r, :, k]
        o_dl = np.full((NC, S, W), np.nan); o_du = np.full((NC, S, W), np.nan); o_dw = np.full((3, S, W), np.nan)
        for gq in (1, 0):
            if 4 * gq >= nr:
                continue
            part = np.full((NC, 4, 3, 32 * P), np.nan)
            for ci, c in enumerate(chans):
                tm = tms[ci]
                for t in (3, 2, 1, 0):
                    r = 4 * gq + t
                    if r >= nr:
                        continue
                    rs = S - 1 - r if rev else r
                    i = H - 1 - (blk * S + r) if rev else blk * S + r
                    w0, w1, w2 = own(st[0], rs), own(st[1], rs), own(st[2], rs)
                    lf, xf = own(ops[ci]["l"], rs), own(ops[ci]["x"], rs)
                    uu, dyf = own(ops[ci]["u"], rs), own(ops[ci]["dy"], rs)
                    gh = dyf * uu + carry[ci]
                    du_ = dyf * hb[ci, r + 1]
                    dl_ = xf * gh
                    p0 = np.empty((32, P)); p1 = np.empty((32, P)); p2 = np.empty((32, P))
                    for k in range(P):
                        p0[:, k] = gh[:, k] * (hls[ci, r] if k == 0 else hb[ci, r, :, k - 1])
                        p1[:, k] = gh[:, k] * hb[ci, r, :, k]
                        p2[:, k] = gh[:, k] * (hrs[ci, r] if k == P - 1 else hb[ci, r, :, k + 1])
                    t0, t1, t2 = w0 * gh, w1 * gh, w2 * gh
                    tl, tr = shfl_up(t2[:, P - 1]), shfl_dn(t0[:, 0])
                    tl[first_lane] = 0.0; tr[last_lane] = 0.0
                    for k in range(P):
                        carry[ci][:, k] = (tl if k == 0 else t2[:, k - 1]) + t1[:, k] + (tr if k == P - 1 else t0[:, k + 1])
                    col = slice(i * P, i * P + P)
                    tm.m[:, col] = (tm.m[:, col] if acc else 0.0) + lf * gh
                    for tap, pv in enumerate((p0, p1, p2)):
                        part[ci, t, tap] = pv.reshape(-1)                       # position P*lane + k
                    for ln in range(WP):
                        o_dl[ci, rs, P * ln:P * ln + P] = dl_[ln]
                        o_du[ci, rs, P * ln:P * ln + P] = du_[ln]
            # reduction after the barrier: warp w takes step 4 gq + w (+ NC ...), channels in ascending order
            for t in range(4):
                r = 4 * gq + t
                if r >= nr:
                    continue
                rs = S - 1 - r if rev else r
                for tap in range(3):
                    s = part[0, t, tap].copy()
                    for cc in range(1, NC):
                        s = s + part[cc, t, tap]
                    o_dw[tap, rs, :WP * P] = s[:WP * P]
        for ci, c in enumerate(chans):
            store_rows(out["dlambda"][q, b, c], o_dl[ci], s0)
            store_rows(out["du"][q, b, c], o_du[ci], s0)
        for tap in range(3):
            store_rows(out["dw3"][q, b, g, tap], o_dw[tap], s0)
    for ci, c in enumerate(chans):
        for ln in range(WP):
            out["dh0"][q, b, c, P * ln:P * ln + P] = carry[ci][ln]


def _bwd_dir_h(out, tms, x, w3, lam, u, dy, h0, b, g, chans, q, rev, acc, H, W, P):
    NC = len(chans)
    nblk = (W + S - 1) // S
    rows = np.arange(32)[:, None] + 32 * np.arange(P)[None, :]
    valid = rows < H
    rc = np.where(valid, rows, 0)

    def cols(plane, s0c):
        """column stage: columns s0c .. s0c+S-1 of plane [H, W] as [H, S], zeros outside"""
        o = np.zeros((H, S))
        lo, hi = max(s0c, 0), min(s0c + S, W)
        if hi > lo:
            o[:, lo - s0c:hi - s0c] = plane[:, lo:hi]
        return o

    def stage(blk):
        s0c = W - (blk + 1) * S if rev else blk * S
        st = [cols(w3[q, b, g, k], s0c) for k in range(3)]
        st[0][0, :] = 0.0; st[2][H - 1, :] = 0.0
        return s0c, st

    ck = np.zeros((NC, nblk, 32, P))
    for ci, c in enumerate(chans):
        h = np.zeros((32, P))
        if h0 is not None:
            h = np.where(valid, h0[q, b, c][rc], 0.0)
        for blk in range(nblk):
            s0c, st = stage(blk)
            sl, sx = cols(lam[q, b, c], s0c), cols(x[b, c], s0c)
            ck[ci, blk] = h
            nr = min(S, W - blk * S)
            for r in range(nr):
                co = S - 1 - r if rev else r
                up, dn = nbr_rows(h, H)
                h = st[0][rc, co] * up + st[2][rc, co] * dn + sl[rc, co] * sx[rc, co] + st[1][rc, co] * h
    carry = np.zeros((NC, 32, P))
    for blk in range(nblk - 1, -1, -1):
        s0c, st = stage(blk)
        nr = min(S, W - blk * S)
        ops = [dict(l=cols(lam[q, b, c], s0c), x=cols(x[b, c], s0c), u=cols(u[q, b, c], s0c), dy=cols(dy[b, c], s0c))
               for c in chans]
        hb = np.zeros((NC, S + 1, 32, P))
        for ci in range(NC):
            hb[ci, 0] = ck[ci, blk]
            for r in range(nr):
                co = S - 1 - r if rev else r
                up, dn = nbr_rows(hb[ci, r], H)
                hb[ci, r + 1] = (st[0][rc, co] * up + st[2][rc, co] * dn + ops[ci]["l"][rc, co] * ops[ci]["x"][rc, co]
                                 + st[1][rc, co] * hb[ci, r])
        o_dl = np.full((NC, H, S), np.nan); o_du = np.full((NC, H, S), np.nan); o_dw = np.full((3, H, S), np.nan)
        for gq in (1, 0):
            if 4 * gq >= nr:
                continue
            qm = 1 - gq if rev else gq                                    # four-column group in memory order
            part = np.full((NC, 4, 3, 32 * P), np.nan)
            for ci, c in enumerate(chans):
                tm = tms[ci]
                j0 = s0c + 4 * qm
                dxv = np.zeros((32, P, 4))
                if acc:
                    for k in range(P):
                        if 32 * k < H:
                            dxv[:, k, :] = tm.m[:, k * 32 * P + j0:k * 32 * P + j0 + 4]
                dlv = np.zeros((32, P, 4)); duv = np.zeros((32, P, 4))
                for t in (3, 2, 1, 0):
                    r = 4 * gq + t
                    e = 3 - t if rev else t
                    if r >= nr:
                        continue
                    co = 4 * qm + e
                    hu, hd = nbr_rows(hb[ci, r], H)
                    dyf = ops[ci]["dy"][rc, co]
                    gh = dyf * ops[ci]["u"][rc, co] + carry[ci]
                    duv[:, :, e] = dyf * hb[ci, r + 1]
                    dlv[:, :, e] = ops[ci]["x"][rc, co] * gh
                    lg = ops[ci]["l"][rc, co] * gh
                    dxv[:, :, e] = dxv[:, :, e] + lg if acc else lg
                    for k in range(P):
                        part[ci, t, 0, 32 * k:32 * k + 32] = (gh * hu)[:, k]
                        part[ci, t, 1, 32 * k:32 * k + 32] = (gh * hb[ci, r])[:, k]
                        part[ci, t, 2, 32 * k:32 * k + 32] = (gh * hd)[:, k]
                    t0, t1, t2 = st[0][rc, co] * gh, st[1][rc, co] * gh, st[2][rc, co] * gh
                    a2, _ = nbr_rows(t2, H)
                    _, a0 = nbr_rows(t0, H)
                    carry[ci] = a2 + t1 + a0
                for k in range(P):
                    if 32 * k < H:
                        tm.m[:, k * 32 * P + j0:k * 32 * P + j0 + 4] = dxv[:, k, :]
                    for ln in range(32):
                        if ln + 32 * k < H:
                            o_dl[ci, ln + 32 * k, 4 * qm:4 * qm + 4] = dlv[ln, k]
                            o_du[ci, ln + 32 * k, 4 * qm:4 * qm + 4] = duv[ln, k]
            for k in range(P):
                for ln in range(32):
                    if ln + 32 * k >= H:
                        continue
                    for tap in range(3):
                        sm = np.zeros(4)
                        for t in range(4):
                            e = 3 - t if rev else t
                            a = 0.0
                            if 4 * gq + t < nr:
                                a = part[0, t, tap, 32 * k + ln]
                                for cc in range(1, NC):
                                    a = a + part[cc, t, tap, 32 * k + ln]
                            sm[e] = a
                        o_dw[tap, ln + 32 * k, 4 * qm:4 * qm + 4] = sm
        # TMA store of the column stage: columns outside the tensor are clipped
        lo, hi = max(s0c, 0), min(s0c + S, W)
        for ci, c in enumerate(chans):
            out["dlambda"][q, b, c][:, lo:hi] = o_dl[ci][:, lo - s0c:hi - s0c]
            out["du"][q, b, c][:, lo:hi] = o_du[ci][:, lo - s0c:hi - s0c]
        for tap in range(3):
            out["dw3"][q, b, g, tap][:, lo:hi] = o_dw[tap][:, lo - s0c:hi - s0c]
    for ci, c in enumerate(chans):
        for k in range(P):
            for ln in range(32):
                if ln + 32 * k < H:
                    out["dh0"][q, b, c, ln + 32 * k] = carry[ci][ln, k]


# ------------------------------------------------------------------------------------------------ the checks
def rand_problem(rng, B, C, H, W, G, mask):
    D = bin(mask).count("1")
    x = rng.standard_normal((B, C, H, W))
    lam = rng.uniform(0.1, 1.0, (D, B, C, H, W))
    u = rng.standard_normal((D, B, C, H, W))
    w3 = rng.uniform(0.05, 1.0, (D, B, G, 3, H, W))
    w3 /= w3.sum(axis=3, keepdims=True)
    # out-of-grid taps hold garbage on purpose: nothing may read them (reading 3)
    qi = 0
    for d in range(4):
        if not mask >> d & 1:
            continue
        if d < 2:
            w3[qi, :, :, 0, :, 0] = 7.0; w3[qi, :, :, 2, :, W - 1] = -5.0
        else:
            w3[qi, :, :, 0, 0, :] = 7.0; w3[qi, :, :, 2, H - 1, :] = -5.0
        qi += 1
    return x, w3, lam, u


SHAPES = [(1, 2, 8, 8, 1, 15), (1, 4, 12, 16, 2, 15), (1, 2, 40, 36, 1, 15), (1, 2, 36, 40, 2, 15), (1, 2, 70, 72, 1, 15),
          (1, 4, 16, 8, 4, 3), (1, 2, 8, 24, 1, 12), (1, 2, 20, 12, 1, 6), (1, 2, 9, 8, 1, 9), (1, 1, 33, 4, 1, 15),
          (1, 2, 4, 68, 2, 15), (2, 2, 8, 8, 2, 1), (1, 2, 8, 8, 1, 2), (1, 2, 8, 8, 1, 4), (1, 2, 8, 8, 1, 8)]


@pytest.mark.parametrize("shape", SHAPES, ids=["x".join(map(str, s)) for s in SHAPES])
def test_forward_dataflow_matches_the_oracle(shape):
    B, C, H, W, G, mask = shape
    rng = np.random.default_rng(100 + H * W + mask)
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, mask)
    w3o = w3.copy()
    y = model_fwd(x, w3, lam, u, G, mask)
    ref = orc.fwd(x, w3o, lam, u, G, mask)
    np.testing.assert_allclose(y, ref, rtol=1e-11, atol=1e-11)


@pytest.mark.parametrize("shape", SHAPES, ids=["x".join(map(str, s)) for s in SHAPES])
def test_backward_dataflow_matches_the_oracle(shape):
    B, C, H, W, G, mask = shape
    rng = np.random.default_rng(200 + H * W + mask)
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, mask)
    dy = rng.standard_normal(x.shape)
    D = bin(mask).count("1")
    h0 = rng.standard_normal((D, B, C, max(H, W)))
    got = model_bwd(x, w3, lam, u, dy, G, mask, h0=h0)
    ref = orc.bwd(x, w3, lam, u, dy, G, mask, h0=h0)
    L = max(H, W)
    for k in ("dx", "dlambda", "du", "dh0"):
        a, r = got[k], ref[k]
        if k == "dh0":          # entries past a direction's line are not written by either side
            qi = 0
            for d in range(4):
                if mask >> d & 1:
                    n = W if d < 2 else H
                    np.testing.assert_allclose(a[qi, ..., :n], r[qi, ..., :n], rtol=1e-10, atol=1e-10, err_msg=k)
                    qi += 1
        else:
            np.testing.assert_allclose(a, r, rtol=1e-10, atol=1e-10, err_msg=k)
    # dw3: the oracle's value at an out-of-grid tap is 0 (h outside the grid is 0): the model writes 0 there too
    np.testing.assert_allclose(got["dw3"], ref["dw3"], rtol=1e-10, atol=1e-10, err_msg="dw3")
