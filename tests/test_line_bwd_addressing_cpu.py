"""Address-level numpy model of gspn_line_bwd.cu: every shared-memory access of the kernel (operand stages filled by
TMA boxes, output stages drained by TMA stores, fp32 partial buffers, checkpoints) goes through flat arrays with the
kernel's own offset formulas, for both storage widths (16-byte pieces of 8 bf16 or 4 fp32 columns), single- and
multi-plane boxes, and the ring / buffer rotation across directions.  Values are fp64; only the indexing is under test.
Companion of tests/test_line_dataflow_cpu.py (which models the arithmetic and the tensor-memory layouts).
"""
import numpy as np
import pytest

from oracle import gspn_oracle as orc
from test_line_dataflow_cpu import P_of, Tmem, nbr_rows, rand_problem, shfl_dn, shfl_up

S = 8
NS = 2          # kBwdStages


class Layout:
    """LineBwdParams of the host side (line_bwd_run)."""
    def __init__(self, H, W, NC, ES):
        self.H, self.W, self.NC, self.ES = H, W, NC, ES
        self.K = 16 // ES
        self.NCH = S // self.K
        L = max(H, W)
        self.P = P_of(L)
        self.pb = (S * L * ES + 127) // 128 * 128
        self.multi = H == W and S * L * ES == self.pb
        self.N1, self.N2, self.NOUT = 3 + 2 * NC, 3 + 4 * NC, 2 * NC + 3
        self.LAM, self.X, self.U, self.DY = 3, 3 + NC, 3 + 2 * NC, 3 + 3 * NC
        self.ODLAM, self.ODU, self.ODW = 0, NC, 2 * NC
        self.Lpad = 32 * self.P
        self.part_stride = 4 * 3 * self.Lpad
        self.stage_bytes = self.N2 * self.pb
        self.out_bytes = self.NOUT * self.pb
        self.nblk_max = (L + S - 1) // S


class Bytes:
    """Shared memory addressed in bytes, holding one value per storage element."""
    def __init__(self, nbytes, ES):
        self.ES = ES
        self.a = np.full(nbytes // ES, np.nan)

    def ix(self, byte):
        assert byte % self.ES == 0, byte
        return byte // self.ES


def tma_rows(sm, dst, tensor, s0, plane0, npl, W, H, load=True):
    """3-D box (W, S, npl) at (0, s0, plane0): planes land back to back; rows outside the tensor: zeros / not written."""
    for p in range(npl):
        for r in range(S):
            i = s0 + r
            o = sm.ix(dst) + (p * S + r) * W
            if load:
                sm.a[o:o + W] = tensor[plane0 + p, i] if 0 <= i < H else 0.0
            elif 0 <= i < H:
                tensor[plane0 + p, i] = sm.a[o:o + W]


def tma_cols(sm, dst, tensor, chunk0, plane0, npl, W, H, K, NCH, load=True):
    """4-D box (K, H, NCH, npl) over [16 B][row][chunk][plane]: shared layout [plane][chunk][row][16 B]."""
    for p in range(npl):
        for ch in range(NCH):
            c = chunk0 + ch
            for row in range(H):
                o = sm.ix(dst) + ((p * NCH + ch) * H + row) * K
                if load:
                    sm.a[o:o + K] = tensor[plane0 + p, row, c * K:c * K + K] if 0 <= c < W // K else 0.0
                elif 0 <= c < W // K:
                    tensor[plane0 + p, row, c * K:c * K + K] = sm.a[o:o + K]


def model(x, w3, lam, u, dy, G, mask, h0, ES):
    B, C, H, W = x.shape
    NC = C // G
    ly = Layout(H, W, NC, ES)
    P, K, NCH, pb = ly.P, ly.K, ly.NCH, ly.pb
    dirs = [d for d in range(4) if mask >> d & 1]
    D = len(dirs)
    L = max(H, W)
    out = dict(dx=np.zeros_like(x), dlambda=np.full_like(lam, np.nan), du=np.full_like(u, np.nan),
               dw3=np.full_like(w3, np.nan), dh0=np.zeros((D, B, C, L)))
    # flat plane views of the tensors, as the tensor maps see them
    X, DYt = x.reshape(B * C, H, W), dy.reshape(B * C, H, W)
    LAMt, Ut, W3t = lam.reshape(D * B * C, H, W), u.reshape(D * B * C, H, W), w3.reshape(D * B * G * 3, H, W)
    DL, DU, DW = out["dlambda"].reshape(D * B * C, H, W), out["du"].reshape(D * B * C, H, W), out["dw3"].reshape(D * B * G * 3, H, W)
    lanes = np.arange(32)
    for b in range(B):
        for g in range(G):
            c0 = g * NC
            ring = Bytes(NS * ly.stage_bytes, ES)
            outs = Bytes(2 * ly.out_bytes, ES)
            part = np.full(2 * NC * ly.part_stride, np.nan)
            ckpt = np.full(NC * ly.nblk_max * ly.Lpad, np.nan)
            tms = [Tmem(((H + 31) // 32) * 32 * P) for _ in range(NC)]
            it = ob = grp = 0
            acc = False
            any_v, any_h = bool(mask & 3), bool(mask & 12)

            def fill(stg, vert, rev, q, blk, npass2):
                """the producer's boxes for one stage"""
                Ls = H if vert else W
                s0 = Ls - (blk + 1) * S if rev else blk * S
                pw, pc, px = ((q * B + b) * G + g) * 3, (q * B + b) * C + c0, b * C + c0
                base = stg * ly.stage_bytes
                ring.a[ring.ix(base):ring.ix(base + ly.stage_bytes)] = np.nan          # stale data must not be relied on
                boxes = [(W3t, pw, 0, 3), (LAMt, pc, ly.LAM, NC), (X, px, ly.X, NC)]
                if npass2:
                    boxes += [(Ut, pc, ly.U, NC), (DYt, px, ly.DY, NC)]
                for ten, plane, slot, n in boxes:
                    for (pl0, sl0, npl) in ([(plane, slot, n)] if ly.multi else [(plane + i, slot + i, 1) for i in range(n)]):
                        if vert:
                            tma_rows(ring, base + sl0 * pb, ten, s0, pl0, npl, W, H)
                        else:
                            tma_cols(ring, base + sl0 * pb, ten, s0 // K, pl0, npl, W, H, K, NCH)
                return s0

            def issue_store(buf, s0, vert, q):
                pc, pw = (q * B + b) * C + c0, ((q * B + b) * G + g) * 3
                obase = buf * ly.out_bytes
                groups = [(DL, pc, ly.ODLAM, NC), (DU, pc, ly.ODU, NC), (DW, pw, ly.ODW, 3)]
                for ten, plane, slot, n in groups:
                    for (pl0, sl0, npl) in ([(plane, slot, n)] if ly.multi else [(plane + i, slot + i, 1) for i in range(n)]):
                        if vert:
                            tma_rows(outs, obase + sl0 * pb, ten, s0, pl0, npl, W, H, load=False)
                        else:
                            tma_cols(outs, obase + sl0 * pb, ten, s0 // K, pl0, npl, W, H, K, NCH, load=False)

            for d in range(4):
                if d == 2 and any_v and any_h:
                    for tm in tms:
                        tm.transpose(H, W, P)
                if d not in dirs:
                    continue
                q, rev, vert = dirs.index(d), d & 1, d < 2
                Ls = H if vert else W
                nblk = (Ls + S - 1) // S
                WP = W // P
                active = lanes < WP
                first_lane, last_lane = lanes == 0, lanes == WP - 1
                lp = np.where(active, lanes, 0)
                rows = lanes[:, None] + 32 * np.arange(P)[None, :]
                rowc = np.where(rows < H, rows, 0)

                def vld(sb, slot, rs):          # line_ld<ST, P>(base + rs * W + slot * pbe): [32, P]
                    o = ring.ix(sb + slot * pb) + rs * W
                    return np.stack([ring.a[o + P * lp + k] for k in range(P)], axis=1)

                def sub(sb, slot, qm):          # sub_ld at sub_off(rowc, qm): [32, P, 4]
                    o = np.empty((32, P, 4))
                    for k in range(P):
                        for ln in range(32):
                            off = (rowc[ln, k] * 16 + qm * 8) if ES == 2 else ((qm * H + rowc[ln, k]) * 16)
                            i0 = ring.ix(sb + slot * pb + off)
                            o[ln, k] = ring.a[i0:i0 + 4]
                    return o

                def zero_taps(sb):
                    if vert:
                        for ln in range(S):
                            ring.a[ring.ix(sb) + ln * W] = 0.0
                            ring.a[ring.ix(sb + 2 * pb) + ln * W + W - 1] = 0.0
                    else:
                        for ln in range(NCH):
                            i0 = ring.ix(sb + (ln * H) * 16); ring.a[i0:i0 + K] = 0.0
                            i0 = ring.ix(sb + 2 * pb + (ln * H + H - 1) * 16); ring.a[i0:i0 + K] = 0.0

                # ---------------- pass 1 (all channel warps; they share the stage, so blocks outer)
                hs = []
                for ci in range(NC):
                    hh = np.zeros((32, P))
                    line0 = h0[q, b, c0 + ci]
                    if vert:
                        for ln in range(WP):
                            hh[ln] = line0[P * ln:P * ln + P]
                    else:
                        hh = np.where(rows < H, line0[rowc], 0.0)
                    hs.append(hh)
                for blk in range(nblk):
                    stg = it % NS
                    fill(stg, vert, rev, q, blk, False)
                    sb = stg * ly.stage_bytes
                    zero_taps(sb)
                    nr = min(S, Ls - blk * S)
                    for ci in range(NC):
                        h = hs[ci]
                        ckb = ci * nblk * ly.Lpad + blk * ly.Lpad
                        for k in range(P):
                            if vert:
                                ckpt[ckb + P * lanes + k] = h[:, k]
                            else:
                                ckpt[ckb + 32 * k + lanes] = h[:, k]
                        for r in range(nr):
                            if vert:
                                rs = S - 1 - r if rev else r
                                w0, w1, w2 = vld(sb, 0, rs), vld(sb, 1, rs), vld(sb, 2, rs)
                                la, xx = vld(sb, ly.LAM + ci, rs), vld(sb, ly.X + ci, rs)
                                hl, hr = shfl_up(h[:, P - 1]), shfl_dn(h[:, 0])
                                hn = np.empty_like(h)
                                for k in range(P):
                                    l = hl if k == 0 else h[:, k - 1]
                                    rr = hr if k == P - 1 else h[:, k + 1]
                                    hn[:, k] = w0[:, k] * l + w2[:, k] * rr + la[:, k] * xx[:, k] + w1[:, k] * h[:, k]
                                h = hn
                            else:
                                qq, tt = divmod(r, 4)
                                qm = 1 - qq if rev else qq
                                e = 3 - tt if rev else tt
                                s0_, s1_, s2_ = sub(sb, 0, qm), sub(sb, 1, qm), sub(sb, 2, qm)
                                sl_, sx_ = sub(sb, ly.LAM + ci, qm), sub(sb, ly.X + ci, qm)
                                up, dn = nbr_rows(h, H)
                                h = s0_[:, :, e] * up + s2_[:, :, e] * dn + sl_[:, :, e] * sx_[:, :, e] + s1_[:, :, e] * h
                        hs[ci] = h
                    it += 1
                # ---------------- pass 2
                carry = [np.zeros((32, P)) for _ in range(NC)]
                pend = None
                for blk in range(nblk - 1, -1, -1):
                    stg = it % NS
                    s0 = fill(stg, vert, rev, q, blk, True)
                    sb = stg * ly.stage_bytes
                    zero_taps(sb)
                    nr = min(S, Ls - blk * S)
                    hb = np.zeros((NC, S + 1, 32, P)); hls = np.zeros((NC, S, 32)); hrs = np.zeros((NC, S, 32))
                    for ci in range(NC):
                        ckb = ci * nblk * ly.Lpad + blk * ly.Lpad
                        for k in range(P):
                            hb[ci, 0, :, k] = ckpt[ckb + P * lanes + k] if vert else ckpt[ckb + 32 * k + lanes]
                        for r in range(nr):
                            if vert:
                                rs = S - 1 - r if rev else r
                                w0, w1, w2 = vld(sb, 0, rs), vld(sb, 1, rs), vld(sb, 2, rs)
                                la, xx = vld(sb, ly.LAM + ci, rs), vld(sb, ly.X + ci, rs)
                                hl, hr = shfl_up(hb[ci, r, :, P - 1]), shfl_dn(hb[ci, r, :, 0])
                                hl[first_lane] = 0.0; hr[last_lane] = 0.0
                                hls[ci, r], hrs[ci, r] = hl, hr
                                for k in range(P):
                                    l = hl if k == 0 else hb[ci, r, :, k - 1]
                                    rr = hr if k == P - 1 else hb[ci, r, :, k + 1]
                                    hb[ci, r + 1, :, k] = w0[:, k] * l + w2[:, k] * rr + la[:, k] * xx[:, k] + w1[:, k] * hb[ci, r, :, k]
                            else:
                                qq, tt = divmod(r, 4)
                                qm = 1 - qq if rev else qq
                                e = 3 - tt if rev else tt
                                s0_, s1_, s2_ = sub(sb, 0, qm), sub(sb, 1, qm), sub(sb, 2, qm)
                                sl_, sx_ = sub(sb, ly.LAM + ci, qm), sub(sb, ly.X + ci, qm)
                                up, dn = nbr_rows(hb[ci, r], H)
                                hb[ci, r + 1] = s0_[:, :, e] * up + s2_[:, :, e] * dn + sl_[:, :, e] * sx_[:, :, e] + s1_[:, :, e] * hb[ci, r]
                    buf = ob & 1
                    obb = buf * ly.out_bytes
                    outs.a[outs.ix(obb):outs.ix(obb + ly.out_bytes)] = np.nan
                    first_bar = True
                    for gq in (1, 0):
                        if 4 * gq >= nr:
                            continue
                        qm = 1 - gq if rev else gq
                        for ci in range(NC):
                            tm = tms[ci]
                            pbuf = ((grp & 1) * NC + ci) * ly.part_stride
                            if vert:
                                for t in (3, 2, 1, 0):
                                    r = 4 * gq + t
                                    if r >= nr:
                                        continue
                                    rs = S - 1 - r if rev else r
                                    i = H - 1 - (blk * S + r) if rev else blk * S + r
                                    w0, w1, w2 = vld(sb, 0, rs), vld(sb, 1, rs), vld(sb, 2, rs)
                                    lf, xf = vld(sb, ly.LAM + ci, rs), vld(sb, ly.X + ci, rs)
                                    uu, dyf = vld(sb, ly.U + ci, rs), vld(sb, ly.DY + ci, rs)
                                    gh = dyf * uu + carry[ci]
                                    du_, dl_ = dyf * hb[ci, r + 1], xf * gh
                                    pv = [np.empty((32, P)) for _ in range(3)]
                                    for k in range(P):
                                        pv[0][:, k] = gh[:, k] * (hls[ci, r] if k == 0 else hb[ci, r, :, k - 1])
                                        pv[1][:, k] = gh[:, k] * hb[ci, r, :, k]
                                        pv[2][:, k] = gh[:, k] * (hrs[ci, r] if k == P - 1 else hb[ci, r, :, k + 1])
                                    t0, t1, t2 = w0 * gh, w1 * gh, w2 * gh
                                    tl, tr = shfl_up(t2[:, P - 1]), shfl_dn(t0[:, 0])
                                    tl[first_lane] = 0.0; tr[last_lane] = 0.0
                                    nc = np.empty((32, P))
                                    for k in range(P):
                                        nc[:, k] = (tl if k == 0 else t2[:, k - 1]) + t1[:, k] + (tr if k == P - 1 else t0[:, k + 1])
                                    carry[ci] = nc
                                    col = slice(i * P, i * P + P)
                                    tm.m[:, col] = (tm.m[:, col] if acc else 0.0) + lf * gh
                                    for tap in range(3):
                                        for k in range(P):
                                            part[pbuf + (t * 3 + tap) * ly.Lpad + P * lanes + k] = pv[tap][:, k]
                                    for ln in range(WP):
                                        for k in range(P):
                                            outs.a[outs.ix(obb + (ly.ODLAM + ci) * pb) + rs * W + P * ln + k] = dl_[ln, k]
                                            outs.a[outs.ix(obb + (ly.ODU + ci) * pb) + rs * W + P * ln + k] = du_[ln, k]
                            else:
                                sv = {n: sub(sb, sl, qm) for n, sl in (("0", 0), ("1", 1), ("2", 2), ("l", ly.LAM + ci), ("x", ly.X + ci),
                                                                      ("u", ly.U + ci), ("y", ly.DY + ci))}
                                j0 = s0 + 4 * qm
                                dxv = np.zeros((32, P, 4)); dlv = np.zeros((32, P, 4)); duv = np.zeros((32, P, 4))
                                if acc:
                                    for k in range(P):
                                        if 32 * k < H:
                                            dxv[:, k] = tm.m[:, k * 32 * P + j0:k * 32 * P + j0 + 4]
                                for t in (3, 2, 1, 0):
                                    r = 4 * gq + t
                                    e = 3 - t if rev else t
                                    if r >= nr:
                                        continue
                                    hu, hd = nbr_rows(hb[ci, r], H)
                                    dyf = sv["y"][:, :, e]
                                    gh = dyf * sv["u"][:, :, e] + carry[ci]
                                    duv[:, :, e] = dyf * hb[ci, r + 1]
                                    dlv[:, :, e] = sv["x"][:, :, e] * gh
                                    lg = sv["l"][:, :, e] * gh
                                    dxv[:, :, e] = dxv[:, :, e] + lg if acc else lg
                                    for k in range(P):
                                        part[pbuf + (t * 3 + 0) * ly.Lpad + 32 * k + lanes] = (gh * hu)[:, k]
                                        part[pbuf + (t * 3 + 1) * ly.Lpad + 32 * k + lanes] = (gh * hb[ci, r])[:, k]
                                        part[pbuf + (t * 3 + 2) * ly.Lpad + 32 * k + lanes] = (gh * hd)[:, k]
                                    t0, t1, t2 = sv["0"][:, :, e] * gh, sv["1"][:, :, e] * gh, sv["2"][:, :, e] * gh
                                    a2, _ = nbr_rows(t2, H)
                                    _, a0 = nbr_rows(t0, H)
                                    carry[ci] = a2 + t1 + a0
                                for k in range(P):
                                    if 32 * k < H:
                                        tm.m[:, k * 32 * P + j0:k * 32 * P + j0 + 4] = dxv[:, k]
                                    for ln in range(32):
                                        if ln + 32 * k < H:
                                            row = ln + 32 * k
                                            off = (row * 16 + qm * 8) if ES == 2 else ((qm * H + row) * 16)
                                            i0 = outs.ix(obb + (ly.ODLAM + ci) * pb + off); outs.a[i0:i0 + 4] = dlv[ln, k]
                                            i0 = outs.ix(obb + (ly.ODU + ci) * pb + off); outs.a[i0:i0 + 4] = duv[ln, k]
                        # ---- barrier; warp 0 issues the pending store at the first barrier of a block
                        if first_bar and pend is not None:
                            issue_store(*pend)
                            pend = None
                        first_bar = False
                        pp = (grp & 1) * NC * ly.part_stride
                        if vert:
                            for cw in range(NC):
                                for t in range(cw, 4, NC):
                                    r = 4 * gq + t
                                    if r >= nr:
                                        continue
                                    rs = S - 1 - r if rev else r
                                    for tap in range(3):
                                        for ln in range(WP):
                                            for k in range(P):
                                                a = part[pp + (t * 3 + tap) * ly.Lpad + P * ln + k]
                                                for cc in range(1, NC):
                                                    a = a + part[pp + cc * ly.part_stride + (t * 3 + tap) * ly.Lpad + P * ln + k]
                                                outs.a[outs.ix(obb + (ly.ODW + tap) * pb) + rs * W + P * ln + k] = a
                        else:
                            for cw in range(NC):
                                for k in range(cw, P, NC):
                                    for ln in range(32):
                                        row = ln + 32 * k
                                        if row >= H:
                                            continue
                                        off = (row * 16 + qm * 8) if ES == 2 else ((qm * H + row) * 16)
                                        for tap in range(3):
                                            sm4 = np.zeros(4)
                                            for t in range(4):
                                                e = 3 - t if rev else t
                                                a = 0.0
                                                if 4 * gq + t < nr:
                                                    a = part[pp + (t * 3 + tap) * ly.Lpad + 32 * k + ln]
                                                    for cc in range(1, NC):
                                                        a = a + part[pp + cc * ly.part_stride + (t * 3 + tap) * ly.Lpad + 32 * k + ln]
                                                sm4[e] = a
                                            i0 = outs.ix(obb + (ly.ODW + tap) * pb + off); outs.a[i0:i0 + 4] = sm4
                        grp += 1
                    pend = (buf, s0, vert, q)
                    ob += 1
                    it += 1
                if pend is not None:
                    issue_store(*pend)
                for ci in range(NC):
                    for k in range(P):
                        for ln in range(32):
                            if vert and ln < WP:
                                out["dh0"][q, b, c0 + ci, P * ln + k] = carry[ci][ln, k]
                            if not vert and ln + 32 * k < H:
                                out["dh0"][q, b, c0 + ci, ln + 32 * k] = carry[ci][ln, k]
                acc = True
            for ci in range(NC):
                tm = tms[ci]
                if any_h:
                    for k in range(P):
                        if 32 * k >= H:
                            continue
                        for ln in range(32):
                            if ln + 32 * k < H:
                                out["dx"][b, c0 + ci, ln + 32 * k] = tm.m[ln, k * 32 * P:k * 32 * P + W]
                else:
                    for i in range(H):
                        for a in range(W // P):
                            out["dx"][b, c0 + ci, i, P * a:P * a + P] = tm.m[a, i * P:i * P + P]
    return out


# shapes the kernel accepts: rows of a multiple of 16 bytes in the storage width under test
CASES = [  # (B, C, H, W, G, mask, ES)
    (1, 2, 8, 8, 1, 15, 2), (1, 2, 8, 8, 1, 15, 4), (1, 4, 16, 16, 1, 15, 2), (1, 2, 12, 16, 2, 15, 2), (1, 2, 40, 48, 1, 15, 2),
    (1, 2, 20, 12, 1, 15, 4), (1, 2, 36, 40, 2, 15, 4), (1, 1, 66, 72, 1, 15, 2), (1, 2, 8, 24, 1, 12, 2), (1, 2, 24, 8, 2, 3, 2),
    (1, 2, 9, 8, 1, 9, 2), (1, 2, 8, 8, 1, 6, 4), (2, 2, 8, 8, 2, 5, 2), (1, 8, 8, 8, 1, 15, 2),
]


@pytest.mark.parametrize("case", CASES, ids=["x".join(map(str, c)) for c in CASES])
def test_backward_addressing_matches_the_oracle(case):
    B, C, H, W, G, mask, ES = case
    assert (W * ES) % 16 == 0
    rng = np.random.default_rng(300 + H * W + mask + ES)
    x, w3, lam, u = rand_problem(rng, B, C, H, W, G, mask)
    dy = rng.standard_normal(x.shape)
    D = bin(mask).count("1")
    h0 = rng.standard_normal((D, B, C, max(H, W)))
    got = model(x, w3, lam, u, dy, G, mask, h0, ES)
    ref = orc.bwd(x, w3, lam, u, dy, G, mask, h0=h0)
    for k in ("dx", "dlambda", "du", "dw3"):
        np.testing.assert_allclose(got[k], ref[k], rtol=1e-10, atol=1e-10, err_msg=k)
    qi = 0
    for d in range(4):
        if mask >> d & 1:
            n = W if d < 2 else H
            np.testing.assert_allclose(got["dh0"][qi, ..., :n], ref["dh0"][qi, ..., :n], rtol=1e-10, atol=1e-10, err_msg="dh0")
            qi += 1
