// gspn_chain_bwd.cu -- fused backward scan of libgspn, "chain" design:
// ONE launch, one CTA per (b, group) unit, the serial recurrences on dedicated WARPS (one per channel
// and role), every pointwise output on separate output warps.
//
// The adjoint recurrence (include/gspn.h "Backward scan"; derived from Eq. 1-2,
// the paper reports backward timings only).  Per direction, over
// blocks of kBlk = 4 scan steps:
//   pass 1 (scan order)    ROLE_A warp of channel c: h[s] = w[s] h[s-1] + lambda[s]*x[s], h in
//                          registers, the state entering each block kept as an fp32 checkpoint on chip;
//   pass 2 (reverse order) ROLE_F warp of channel c: h of the block's steps recomputed from its
//                          checkpoint;  ROLE_A warp: gh[s] = dy[s]*u[s] + carry, carry = w[s]^T gh
//                          (neighbours by warp shuffle, no block barrier);  both hand their 4 lines to
//                          the output warps through a double-buffered fp32 block buffer (mbarriers);
//                          output warp j: step j of the block for ALL channels of the group:
//                          du = dy*h[s], dlambda = x*gh, dx += lambda*gh, dw3[k] = sum_c gh_c*h_c[s-1,p+k-1].
// dx of the group's channels is accumulated over the directions in an fp32 plane per channel on chip
// (directions run one after another and a step owns one image line, so every element has a single
// writer) and rounded once at the end.  dw3 (Eq. 5: taps shared by the channels of a group,
// PAPER.md:131-134) is summed over the channels in registers, in ascending channel order
// (deterministic, no atomics, no exchange between warps).  Vertical outputs are stored straight from
// registers (lanes own consecutive columns); horizontal outputs go through 8-column tiles so that every
// store instruction writes 16-byte row pieces (the transposed tile on the way out).
//
// Operands: gspn_chain.cuh.  kChNPW producer warps stream, for the current direction and pass, a ring
// of stages: for T->B / B->T a block of 4 image rows of every operand plane (one 1-D bulk copy per plane
// over its 16-byte-aligned superset), for L->R / R->L one chunk column (4 columns of every row of
// every plane, cp.async of the aligned chunk; a row keeps NSH+1 chunk slots contiguous, slot NSH
// mirrors slot 0, so the two chunks a block of 4 columns touches are always contiguous).
#include "gspn_chain.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

constexpr int kChMaxNS = 4;                       // channels per group the kernel takes
constexpr int kChNO = kBlk;                       // output warps: one per step of a block
constexpr int kChBars = 2 * kChSlots + 4;         // full[8] empty[8] ready[2] free[2]
constexpr int kChNPW = 4;                         // producer warps
constexpr int kChMaxPlanes = 3 + 4 * kChMaxNS;    // w0 w1 w2, lambda[c], x[c], u[c], dy[c]
constexpr int kTilePitch = 10;                    // elements per row of an 8-column output tile (odd word pitch)

struct ChainBwdParams {
    Shape sh;
    const void *x, *w3, *lam, *u, *h0, *dy;
    void *dx, *dlam, *du, *dw3, *dh0;
    int NS;                         // chain warps = channels per group
    int NSV, NSH, NQ;               // ring slots (row blocks / chunk columns); chunk columns per row
    int Wp;                         // row pitch of the dx planes in floats
    uint32_t vslot, vstage, hrow, hplane;
    uint32_t off_tab, off_dx, off_ring, off_ckpt, off_hb, off_gb, off_tile, total;
    uint32_t ckpt_warp;             // checkpoint bytes per channel
    int q[4];                       // slab index of each direction, -1 = not in dir_mask
    unsigned long long bytes_x, bytes_c, bytes_w;
};

enum { KW0 = 0, KW1, KW2, KLAM, KX, KU, KDY, KNUM };

// hand-over of one block's h / gh lines from the chain warps to the output warps (double buffered)
struct BlockSync {
    uint64_t *ready, *freeb;      // [2] each
    uint32_t n;                   // blocks handed over so far (all directions)
    __device__ __forceinline__ int buf() const { return n & 1u; }
    __device__ __forceinline__ void producer_wait() { mbar_wait(&freeb[n & 1u], ((n >> 1) & 1u) ^ 1u); }
    __device__ __forceinline__ void producer_done(int lane) { __syncwarp(); if (lane == 0) mbar_arrive(&ready[n & 1u]); ++n; }
    __device__ __forceinline__ void consumer_wait() { mbar_wait(&ready[n & 1u], (n >> 1) & 1u); }
    __device__ __forceinline__ void consumer_done(int lane) { __syncwarp(); if (lane == 0) mbar_arrive(&freeb[n & 1u]); ++n; }
};

// ---------------------------------------------------------------------------------------------------
// Chain warps of channel c, one direction.  VH = false: T->B / B->T (lanes own columns), true:
// L->R / R->L (lanes own rows); REV = the direction walks the image lines downwards.
//   ROLE_A  pass 1: h[s] = w[s] h[s-1] + lambda[s]*x[s] in scan order, the state entering every block
//                   stored as a checkpoint; pass 2: the adjoint chain gh[s] = dy[s]*u[s] + w[s+1]^T gh[s+1]
//                   in reverse order, gh of every step handed to the output warps; dh0 at the end.
//   ROLE_F  pass 2: h of the block's steps recomputed from its checkpoint, handed to the output warps.
// Lane-dependent conditions (position inside the line, first / last position) are 32-bit AND masks in
// ordinary registers: values of positions past the line are forced to +0 exactly.
enum { ROLE_A = 0, ROLE_F = 1 };

template <typename ST, int P, bool VH, bool REV, int ROLE>
__device__ __forceinline__ void chain_bwd_dir(const ChainBwdParams& p, uint8_t* smem, const int d, const int b,
                                              const int g, const int c, const int lane, uint32_t& pf,
                                              BlockSync& bs) {
    using E = Elem<ST>;
    using raw_t = typename E::raw_t;
    constexpr int ES = sizeof(ST);
    constexpr int CB = kBlk * ES;
    constexpr unsigned FULLM = 0xffffffffu;
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, NS = p.NS;
    const int Ls = VH ? W : H, Lp = VH ? H : W, Lmax = sh.Lmax();
    const int NB = (Ls + kBlk - 1) / kBlk;
    const uint32_t rowB = (uint32_t)W * ES;
    const int qd = p.q[d];
    const ChPlane* tb = reinterpret_cast<const ChPlane*>(smem + p.off_tab) + d * kChMaxPlanes;
    const uint32_t ring = smem_u32(smem + p.off_ring);
    const int sidx[KNUM] = {0, 1, 2, 3 + c, 3 + NS + c, 3 + 2 * NS + c, 3 + 3 * NS + c};
    RingSync<VH> rs{reinterpret_cast<uint64_t*>(smem), reinterpret_cast<uint64_t*>(smem) + kChSlots,
                    p.NSV, p.NSH, p.NQ, lane, 0, pf};

    bool ok[P];
    uint32_t okm[P], m_w2[P];
    const int last_lane = (Lp - 1) / P, last_e = (Lp - 1) % P;
#pragma unroll
    for (int e = 0; e < P; ++e) {
        ok[e] = P * lane + e < Lp;
        okm[e] = ok[e] ? 0xffffffffu : 0u;
        m_w2[e] = (lane == last_lane && e == last_e) ? 0u : 0xffffffffu;      // out-of-grid taps are never used
    }
    const uint32_t m_first = lane == 0 ? 0u : 0xffffffffu;
    const uint32_t m_31 = lane == 31 ? 0u : 0xffffffffu;

    const size_t pc = ((size_t)qd * sh.B + b) * sh.C + (size_t)g * NS + c;    // plane in [D,B,C]
    const uint32_t cks = smem_u32(smem + p.off_ckpt) + c * p.ckpt_warp + lane * 4;             // [NB][P][32]
    const uint32_t hbuf = smem_u32(smem + p.off_hb) + (uint32_t)c * 2 * (kBlk + 1) * P * 128 + lane * 4;  // [2][kBlk+1][P][32]
    const uint32_t gbuf = smem_u32(smem + p.off_gb) + (uint32_t)c * 2 * kBlk * P * 128 + lane * 4;        // [2][kBlk][P][32]

    // operand addresses inside the ring
    uint32_t phs[KNUM];          // vertical: byte phase (mod 16) of each plane
    uint32_t vb[KNUM];           // vertical: per block, address of (local line 0, this lane's first column)
    uint32_t hb[KNUM][P];        // horizontal: address of (this lane's row e, chunk slot 0) + the row's byte phase
    if constexpr (!VH) {
#pragma unroll
        for (int k = 0; k < KNUM; ++k) { phs[k] = (uint32_t)(tb[sidx[k]].b0 & 15ull); vb[k] = 0; }
    } else {
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const int row = min(P * lane + e, H - 1);          // rows past the plane re-read the last row
#pragma unroll
            for (int k = 0; k < KNUM; ++k)
                hb[k][e] = ring + sidx[k] * p.hplane + row * p.hrow +
                           (uint32_t)((tb[sidx[k]].b0 + (unsigned long long)row * rowB) % CB);
        }
    }
    // element e of operand k on image-local line tl of the current block (plain loads: the mbarrier
    // waits / arrives carry memory clobbers and keep them inside the stage's lifetime)
    const uint8_t* const sbase = smem - smem_u32(smem);           // generic address of shared offset 0
    auto ldr = [&](int k, int tl, uint32_t so, int e) -> raw_t {
        if constexpr (!VH) return *reinterpret_cast<const raw_t*>(sbase + (vb[k] + tl * rowB + e * ES));
        else return *reinterpret_cast<const raw_t*>(sbase + (hb[k][e] + so + tl * ES));
    };
    uint32_t hso = 0;
    auto block_setup = [&](int bi) -> uint32_t {
        if constexpr (!VH) {
            const uint32_t stage = ring + (bi % p.NSV) * p.vstage;
            const uint32_t rb = ((uint32_t)(kBlk * bi) * rowB) & 15u;
#pragma unroll
            for (int k = 0; k < KNUM; ++k)
                vb[k] = stage + sidx[k] * p.vslot + ((phs[k] + rb) & 15u) + lane * (P * ES);
            return 0u;
        } else {
            // fold the block's chunk-slot offset into the row addresses once per block
            const uint32_t nso = (uint32_t)(bi % p.NSH) * CB;
#pragma unroll
            for (int e = 0; e < P; ++e)
#pragma unroll
                for (int k = 0; k < KNUM; ++k) hb[k][e] += nso - hso;
            hso = nso;
            return 0u;
        }
    };

    // one forward step on image-local line tl: hout = w[s] hin + lambda[s]*x[s]
    auto fwd_step = [&](const float (&hin)[P], int tl, uint32_t so, float (&hout)[P]) {
        raw_t w0r[P], w1r[P], w2r[P], lr[P], xr[P];
#pragma unroll
        for (int e = 0; e < P; ++e) {
            w0r[e] = ldr(KW0, tl, so, e); w1r[e] = ldr(KW1, tl, so, e); w2r[e] = ldr(KW2, tl, so, e);
            lr[e] = ldr(KLAM, tl, so, e); xr[e] = ldr(KX, tl, so, e);
        }
        const float hl = maskf(__shfl_up_sync(FULLM, hin[P - 1], 1), m_first);
        const float hr = __shfl_down_sync(FULLM, hin[0], 1);     // lane 31: masked through m_w2 / okm
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const float w0f = e == 0 ? maskf(E::f(w0r[e]), m_first) : E::f(w0r[e]);
            const float w2f = maskf(E::f(w2r[e]), m_w2[e]);
            const float left = e ? hin[e - 1] : hl;
            const float right = e < P - 1 ? hin[e + 1] : hr;
            float acc = E::f(w1r[e]) * hin[e];
            acc = fmaf(w0f, left, acc);
            acc = fmaf(w2f, right, acc);
            acc = E::fma2(lr[e], xr[e], acc);
            hout[e] = maskf(acc, okm[e]);                               // positions past the line stay +0
        }
    };

    // ================= pass 1: scan order, checkpoints (ROLE_A; ROLE_F only follows the ring) ===========
    rs.begin_pass(REV);
    {
        float h[P];
#pragma unroll
        for (int e = 0; e < P; ++e) {
            h[e] = 0.f;
            if (ROLE == ROLE_A && p.h0 && ok[e]) h[e] = ld_f(reinterpret_cast<const ST*>(p.h0) + pc * Lmax + P * lane + e);
        }
        for (int n = 0; n < NB; ++n) {
            const int bi = REV ? NB - 1 - n : n;
            const int nb = min(kBlk, Ls - kBlk * bi);
            rs.acquire(bi, REV);
            if constexpr (ROLE == ROLE_A) {
#pragma unroll
                for (int e = 0; e < P; ++e) sts32(cks + (bi * P + e) * 128, h[e]);
                const uint32_t so = block_setup(bi);
#pragma unroll
                for (int t = 0; t < kBlk; ++t) {
                    const int tl = REV ? kBlk - 1 - t : t;
                    if (tl < nb) {
                        float hn[P];
                        fwd_step(h, tl, so, hn);
#pragma unroll
                        for (int e = 0; e < P; ++e) h[e] = hn[e];
                    }
                }
            }
            rs.release(bi, REV, n == NB - 1);
        }
    }
    // the checkpoints written by ROLE_A are read by ROLE_F of the same channel
    named_bar_sync(2 + c, 64);

    // ================= pass 2: reverse order ===========================================================
    constexpr bool desc2 = !REV;
    float carry[P];
#pragma unroll
    for (int e = 0; e < P; ++e) carry[e] = 0.f;
    rs.begin_pass(desc2);
    for (int n = 0; n < NB; ++n) {
        const int bi = desc2 ? NB - 1 - n : n;
        const int nb = min(kBlk, Ls - kBlk * bi);
        rs.acquire(bi, desc2);
        const uint32_t so = block_setup(bi);
        bs.producer_wait();
        if constexpr (ROLE == ROLE_F) {
            // hs[t] = state entering the t-th step (scan order) of the block
            const uint32_t hw = hbuf + bs.buf() * ((kBlk + 1) * P * 128);
            float hs[kBlk + 1][P];
#pragma unroll
            for (int e = 0; e < P; ++e) { hs[0][e] = lds32(cks + (bi * P + e) * 128); sts32(hw + e * 128, hs[0][e]); }
#pragma unroll
            for (int t = 0; t < kBlk; ++t) {
                const int tl = REV ? kBlk - 1 - t : t;
                if (tl < nb) {
                    fwd_step(hs[t], tl, so, hs[t + 1]);
                } else {
#pragma unroll
                    for (int e = 0; e < P; ++e) hs[t + 1][e] = hs[t][e];
                }
#pragma unroll
                for (int e = 0; e < P; ++e) sts32(hw + ((t + 1) * P + e) * 128, hs[t + 1][e]);
            }
        } else {
            const uint32_t gw = gbuf + bs.buf() * (kBlk * P * 128);
#pragma unroll
            for (int tt = 0; tt < kBlk; ++tt) {
                const int t = kBlk - 1 - tt;
                const int tl = REV ? kBlk - 1 - t : t;
                if (tl < nb) {
                    raw_t w0r[P], w1r[P], w2r[P], ur[P], dyr[P];
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        ur[e] = ldr(KU, tl, so, e); dyr[e] = ldr(KDY, tl, so, e);
                        w0r[e] = ldr(KW0, tl, so, e); w1r[e] = ldr(KW1, tl, so, e); w2r[e] = ldr(KW2, tl, so, e);
                    }
                    float gh[P];
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        gh[e] = maskf(E::fma2(dyr[e], ur[e], carry[e]), okm[e]);
                        sts32(gw + (t * P + e) * 128, gh[e]);
                    }
                    // carry = w[s]^T gh: position p receives from p-1 (its tap k=2), p (k=1), p+1 (k=0)
                    float a2[P], c0[P];
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        const float w0f = e == 0 ? maskf(E::f(w0r[e]), m_first) : E::f(w0r[e]);
                        a2[e] = maskf(E::f(w2r[e]), m_w2[e]) * gh[e];
                        c0[e] = w0f * gh[e];
                    }
                    const float al = maskf(__shfl_up_sync(FULLM, a2[P - 1], 1), m_first);
                    const float cr = maskf(__shfl_down_sync(FULLM, c0[0], 1), m_31);
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        float acc = fmaf(E::f(w1r[e]), gh[e], e ? a2[e - 1] : al);
                        acc += e < P - 1 ? c0[e + 1] : cr;
                        carry[e] = acc;
                    }
                }
            }
        }
        bs.producer_done(lane);
        rs.release(bi, desc2, n == NB - 1);
    }
    if (ROLE == ROLE_A && p.dh0) {
        ST* d0 = reinterpret_cast<ST*>(p.dh0) + pc * Lmax;
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const int pos = P * lane + e;
            if (pos < Lmax) E::stg(d0 + pos, E::pack(ok[e] ? carry[e] : 0.f));
        }
    }
    // ROLE_A must not overwrite the checkpoints (next direction) while ROLE_F still reads them
    named_bar_sync(2 + c, 64);
    pf = rs.pf;
}

// ---------------------------------------------------------------------------------------------------
// Output warp j of one direction: every block, scan-order step j of ALL channels of the group.  Given
// h[s], h[s-1] (from the ROLE_F warps) and gh[s] (from the ROLE_A warps) every output is pointwise:
//     du = dy*h[s]   dlambda = x*gh   dx += lambda*gh   dw3[k] = sum_c gh_c * h_c[s-1, p+k-1]
// so the sum over the group's channels (Eq. 5: shared taps) is a register
// accumulation in ascending channel order -- no exchange between warps, no atomics.  A step owns one
// image line (row or column), so the fp32 dx planes have a single writer per element.
template <typename ST, int P, bool VH>
__device__ __forceinline__ void chain_bwd_out(const ChainBwdParams& p, uint8_t* smem, const int d, const int b,
                                              const int g, const int j, const int lane, uint32_t& pf,
                                              BlockSync& bs) {
    using E = Elem<ST>;
    using raw_t = typename E::raw_t;
    constexpr int ES = sizeof(ST);
    constexpr int CB = kBlk * ES;
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, NS = p.NS;
    const bool rev = d & 1;
    const int Ls = VH ? W : H, Lp = VH ? H : W;
    const int NB = (Ls + kBlk - 1) / kBlk;
    const uint32_t rowB = (uint32_t)W * ES;
    const int qd = p.q[d];
    const size_t HW = (size_t)H * W;
    const ChPlane* tb = reinterpret_cast<const ChPlane*>(smem + p.off_tab) + d * kChMaxPlanes;
    const uint32_t ring = smem_u32(smem + p.off_ring);
    const uint8_t* const sbase = smem - smem_u32(smem);
    RingSync<VH> rs{reinterpret_cast<uint64_t*>(smem), reinterpret_cast<uint64_t*>(smem) + kChSlots,
                    p.NSV, p.NSH, p.NQ, lane, 0, pf};

    bool ok[P];
#pragma unroll
    for (int e = 0; e < P; ++e) ok[e] = P * lane + e < Lp;
    const uint32_t m_first = lane == 0 ? 0u : 0xffffffffu;
    const uint32_t m_31 = lane == 31 ? 0u : 0xffffffffu;

    const size_t pc0 = ((size_t)qd * sh.B + b) * sh.C + (size_t)g * NS;       // plane of channel 0 in [D,B,C]
    const size_t pw = (((size_t)qd * sh.B + b) * sh.G + g) * 3;                // first tap plane in [D,B,G,3]
    const bool w_du = p.du != nullptr, w_dl = p.dlam != nullptr, w_dw = p.dw3 != nullptr, w_dx = p.dx != nullptr;
    ST* du0 = reinterpret_cast<ST*>(p.du) + pc0 * HW;
    ST* dl0 = reinterpret_cast<ST*>(p.dlam) + pc0 * HW;
    ST* dw0 = reinterpret_cast<ST*>(p.dw3) + pw * HW;
    const uint32_t dxs = smem_u32(smem + p.off_dx);                            // [NS][H][Wp] fp32
    const uint32_t hb0 = smem_u32(smem + p.off_hb) + lane * 4;                 // [NS][2][kBlk+1][P][32]
    const uint32_t gb0 = smem_u32(smem + p.off_gb) + lane * 4;                 // [NS][2][kBlk][P][32]
    const uint32_t tile = smem_u32(smem + p.off_tile);                         // [2NS+3][Lp][kTilePitch]
    const uint32_t tplane = (uint32_t)Lp * kTilePitch * ES;

    uint32_t rowadr[P], rowph[P], rowdx[P], rowtl[P];      // horizontal: per row of this lane
    if constexpr (VH) {
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const int row = min(P * lane + e, H - 1);
            rowadr[e] = ring + row * p.hrow;
            rowph[e] = (uint32_t)(((unsigned long long)row * rowB) % CB);
            rowdx[e] = (uint32_t)row * p.Wp * 4;
            rowtl[e] = (uint32_t)row * kTilePitch * ES;
        }
    }

    // pass 1: nothing to do, follow the ring
    rs.begin_pass(rev);
    for (int n = 0; n < NB; ++n) {
        const int bi = rev ? NB - 1 - n : n;
        rs.acquire(bi, rev);
        rs.release(bi, rev, n == NB - 1);
    }
    const bool desc2 = !rev;
    rs.begin_pass(desc2);
    const int t = j;                                     // scan-order step of every block this warp owns
    const int tl = rev ? kBlk - 1 - t : t;               // its image-local line
    for (int n = 0; n < NB; ++n) {
        const int bi = desc2 ? NB - 1 - n : n;
        const int nb = min(kBlk, Ls - kBlk * bi);
        rs.acquire(bi, desc2);
        bs.consumer_wait();
        if (tl < nb) {
            const int li = kBlk * bi + tl;                                       // image line (row / column)
            const uint32_t hoff = bs.buf() * ((kBlk + 1) * P * 128) + t * P * 128;
            const uint32_t goff = bs.buf() * (kBlk * P * 128) + t * P * 128;
            const uint32_t so = VH ? (uint32_t)(bi % p.NSH) * CB + tl * ES : 0u;
            const uint32_t vst = VH ? 0u : ring + (bi % p.NSV) * p.vstage + lane * (P * ES) + tl * rowB;
            const uint32_t rb = ((uint32_t)(kBlk * bi) * rowB) & 15u;
            const uint32_t cs = (uint32_t)((bi & 1) * kBlk + tl) * ES;
            float dw[3][P];
#pragma unroll
            for (int e = 0; e < P; ++e) { dw[0][e] = 0.f; dw[1][e] = 0.f; dw[2][e] = 0.f; }
#pragma unroll 1
            for (int c = 0; c < NS; ++c) {
                const uint32_t hc = hb0 + (uint32_t)c * 2 * (kBlk + 1) * P * 128 + hoff;
                const uint32_t gc = gb0 + (uint32_t)c * 2 * kBlk * P * 128 + goff;
                float hn[P], hp[P], gh[P], dxo[P];
                uint32_t dxa[P];
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    hp[e] = lds32(hc + e * 128);
                    hn[e] = lds32(hc + (P + e) * 128);
                    gh[e] = lds32(gc + e * 128);
                    // the dx accumulators of this step are read together with the block buffers: one shared-memory
                    // round trip per channel instead of a read -> write -> read chain per position
                    if constexpr (!VH) dxa[e] = dxs + (((uint32_t)c * H + li) * p.Wp + P * lane + e) * 4;
                    else dxa[e] = dxs + (uint32_t)c * H * p.Wp * 4 + rowdx[e] + li * 4;
                    dxo[e] = 0.f;
                    if (w_dx && ok[e]) dxo[e] = lds32(dxa[e]);
                }
                const float hpl = maskf(lds32(hc + (P - 1) * 128 - 4), m_first);     // h[s-1] of position p-1 (lane-1)
                const float hpr = maskf(lds32(hc + 4), m_31);                        // h[s-1] of position p+1 (lane+1)
                // operand addresses: lambda, x, dy planes of channel c
                raw_t lr[P], xr[P], dyr[P];
                {
                    const int sl = 3 + c, sx = 3 + NS + c, sy = 3 + 3 * NS + c;
                    const uint32_t bl = (uint32_t)tb[sl].b0, bx = (uint32_t)tb[sx].b0, by = (uint32_t)tb[sy].b0;
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        uint32_t al, ax, ay;
                        if constexpr (!VH) {
                            al = vst + sl * p.vslot + ((bl + rb) & 15u) + e * ES;
                            ax = vst + sx * p.vslot + ((bx + rb) & 15u) + e * ES;
                            ay = vst + sy * p.vslot + ((by + rb) & 15u) + e * ES;
                        } else {
                            al = rowadr[e] + sl * p.hplane + ((bl + rowph[e]) & (CB - 1)) + so;
                            ax = rowadr[e] + sx * p.hplane + ((bx + rowph[e]) & (CB - 1)) + so;
                            ay = rowadr[e] + sy * p.hplane + ((by + rowph[e]) & (CB - 1)) + so;
                        }
                        lr[e] = *reinterpret_cast<const raw_t*>(sbase + al);
                        xr[e] = *reinterpret_cast<const raw_t*>(sbase + ax);
                        dyr[e] = *reinterpret_cast<const raw_t*>(sbase + ay);
                    }
                }
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    const float left = e ? hp[e - 1] : hpl;
                    const float right = e < P - 1 ? hp[e + 1] : hpr;
                    dw[0][e] = fmaf(gh[e], left, dw[0][e]);
                    dw[1][e] = fmaf(gh[e], hp[e], dw[1][e]);
                    dw[2][e] = fmaf(gh[e], right, dw[2][e]);
                    const raw_t duv = E::pack(E::f(dyr[e]) * hn[e]);
                    const raw_t dlv = E::pack(E::f(xr[e]) * gh[e]);
                    if constexpr (!VH) {
                        const size_t o = (size_t)c * HW + (size_t)li * W + P * lane + e;
                        if (w_du && ok[e]) E::stg(du0 + o, duv);
                        if (w_dl && ok[e]) E::stg(dl0 + o, dlv);
                        if (w_dx && ok[e]) sts32(dxa[e], fmaf(E::f(lr[e]), gh[e], dxo[e]));
                    } else {
                        if (w_du && ok[e]) E::sts(tile + c * tplane + rowtl[e] + cs, duv);
                        if (w_dl && ok[e]) E::sts(tile + (NS + c) * tplane + rowtl[e] + cs, dlv);
                        if (w_dx && ok[e]) sts32(dxa[e], fmaf(E::f(lr[e]), gh[e], dxo[e]));
                    }
                }
            }
            if (w_dw) {
#pragma unroll
                for (int k = 0; k < 3; ++k)
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        if constexpr (!VH) {
                            if (ok[e]) E::stg(dw0 + (size_t)k * HW + (size_t)li * W + P * lane + e, E::pack(dw[k][e]));
                        } else {
                            if (ok[e]) E::sts(tile + (2 * NS + k) * tplane + rowtl[e] + cs, E::pack(dw[k][e]));
                        }
                    }
            }
        }
        bs.consumer_done(lane);
        // horizontal outputs: a pair of blocks = 8 columns is complete -> 16-byte row pieces to global
        if constexpr (VH) {
            const bool pair_done = desc2 ? ((bi & 1) == 0) : ((bi & 1) == 1 || bi == NB - 1);
            if (pair_done) {
                named_bar_sync(10, 128);
                const int col0 = 2 * kBlk * (bi >> 1);
                const int ncols = min(2 * kBlk, W - col0);
                const int col = lane & 7, rsub = lane >> 3;
                if (col < ncols) {
                    for (int pl = j; pl < 2 * NS + 3; pl += kBlk) {
                        ST* gp;
                        if (pl < NS) gp = w_du ? du0 + (size_t)pl * HW : nullptr;
                        else if (pl < 2 * NS) gp = w_dl ? dl0 + (size_t)(pl - NS) * HW : nullptr;
                        else gp = w_dw ? dw0 + (size_t)(pl - 2 * NS) * HW : nullptr;
                        if (gp) {
                            gp += (size_t)rsub * W + col0 + col;
                            uint32_t ta = tile + pl * tplane + (rsub * kTilePitch + col) * ES;
                            for (int r = rsub; r < Lp; r += 4) {
                                E::stg(gp, E::lds(ta));
                                ta += 4 * kTilePitch * ES; gp += 4 * W;
                            }
                        }
                    }
                }
                named_bar_sync(10, 128);
            }
        }
        rs.release(bi, desc2, n == NB - 1);
    }
    pf = rs.pf;
}

// ---------------------------------------------------------------------------------------------------
template <typename ST, int P>
__global__ void __launch_bounds__(32 * (kChNPW + 2 * kChMaxNS + kChNO), P == 1 ? 2 : 1)
chain_bwd_kernel(const ChainBwdParams p) {
    constexpr int ES = sizeof(ST);
    constexpr int CB = kBlk * ES;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    uint64_t* empty = full + kChSlots;
    ChPlane* tab = reinterpret_cast<ChPlane*>(smem + p.off_tab);       // [4][kChMaxPlanes]
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, NS = p.NS;
    const int np = 3 + 4 * NS;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int b = blockIdx.x / sh.G, g = blockIdx.x % sh.G;
    const int c0 = g * NS;
    const unsigned long long HW = (unsigned long long)H * W;
    const uint32_t rowB = (uint32_t)W * ES;

    // shared memory starts as zeros: lanes past a line's end read (and discard) finite values
    for (uint32_t o = threadIdx.x * 16; o < p.total; o += blockDim.x * 16)
        *reinterpret_cast<uint4*>(smem + o) = make_uint4(0, 0, 0, 0);
    __syncthreads();
    for (int idx = threadIdx.x; idx < 4 * kChMaxPlanes; idx += blockDim.x) {
        const int d = idx / kChMaxPlanes, s = idx % kChMaxPlanes;
        if (p.q[d] >= 0 && s < np) {
            const unsigned long long q = p.q[d];
            ChPlane e;
            if (s < 3) {
                e.base = (const uint8_t*)p.w3; e.tbytes = p.bytes_w;
                e.b0 = ((((q * sh.B + b) * sh.G + g) * 3 + s) * HW) * ES;
            } else {
                const int t = (s - 3) / NS, c = (s - 3) % NS;          // 0 lambda, 1 x, 2 u, 3 dy
                const unsigned long long slab = (((q * sh.B + b) * sh.C + c0 + c) * HW) * ES;
                const unsigned long long img = (((unsigned long long)b * sh.C + c0 + c) * HW) * ES;
                if (t == 0)      { e.base = (const uint8_t*)p.lam; e.tbytes = p.bytes_c; e.b0 = slab; }
                else if (t == 1) { e.base = (const uint8_t*)p.x;   e.tbytes = p.bytes_x; e.b0 = img; }
                else if (t == 2) { e.base = (const uint8_t*)p.u;   e.tbytes = p.bytes_c; e.b0 = slab; }
                else             { e.base = (const uint8_t*)p.dy;  e.tbytes = p.bytes_x; e.b0 = img; }
            }
            tab[idx] = e;
        }
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < kChSlots; ++s) { mbar_init(&full[s], kChNPW * 33); mbar_init(&empty[s], 2 * NS + kChNO); }
        for (int s = 0; s < 2; ++s) { mbar_init(&empty[kChSlots + s], 2 * NS); mbar_init(&empty[kChSlots + 2 + s], kChNO); }
        mbar_init_fence();
    }
    fence_proxy_async();      // zeros (generic proxy) before bulk copies
    __syncthreads();

    if (warp < kChNPW) {
        // ---------------- producer warp pw: planes pw, pw + NPW, ... of every stage ----------------------
        const int pw = warp;
        const uint32_t ring = smem_u32(smem + p.off_ring);
        uint8_t* ringp = smem + p.off_ring;
        uint32_t pe = 0;
        bool drained = false;
        // horizontal: this lane copies rows lane, lane+32, ... of each of its planes
        uint32_t rowoff[4], rowdst[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) { rowoff[r] = (uint32_t)(lane + 32 * r) * rowB; rowdst[r] = (uint32_t)(lane + 32 * r) * p.hrow; }
        for (int d = 0; d < 4; ++d) {
            if (p.q[d] < 0) continue;
            const bool vh = d >> 1, rev = d & 1;
            const ChPlane* tb = tab + d * kChMaxPlanes;
            {   // announce every operand plane of this direction to L2
                const int s = lane * kChNPW + pw;
                if (s < np) l2_prefetch_plane(tb[s].base, tb[s].b0, tb[s].tbytes, HW * ES);
            }
            if (vh && !drained) {
                // row-block stages and chunk columns lay the ring out differently: every slot must be
                // released before the first chunk column is written
                for (int s = 0; s < kChSlots; ++s) mbar_wait(&empty[s], ((pe >> s) & 1u) ^ 1u);
                drained = true;
            }
            for (int pass = 0; pass < 2; ++pass) {
                const int npp = pass == 0 ? 3 + 2 * NS : np;
                const bool desc = rev != (pass == 1);
                if (!vh) {
                    const int NB = (H + kBlk - 1) / kBlk;
                    const int s = lane * kChNPW + pw;                 // this lane's plane
                    ChPlane e{nullptr, 0, 0};
                    if (s < npp) e = tb[s];
                    for (int n = 0; n < NB; ++n) {
                        const int bi = desc ? NB - 1 - n : n;
                        const int slot = bi % p.NSV;
                        const int r0 = kBlk * bi, r1 = min(H, r0 + kBlk);
                        mbar_wait(&empty[slot], ((pe >> slot) & 1u) ^ 1u);
                        pe ^= 1u << slot;
                        uint64_t* fb = &full[slot];
                        int nbytes = 0;
                        unsigned long long a0 = 0;
                        uint8_t* dst = ringp + (size_t)slot * p.vstage + (size_t)s * p.vslot;
                        if (s < npp) {
                            const unsigned long long byte0 = e.b0 + (unsigned long long)r0 * rowB;
                            const unsigned long long byte1 = e.b0 + (unsigned long long)r1 * rowB;
                            a0 = byte0 & ~15ull;
                            const unsigned long long lim = e.tbytes & ~15ull;
                            unsigned long long a1 = (byte1 + 15) & ~15ull;
                            if (a1 > lim) a1 = lim;
                            nbytes = a1 > a0 ? (int)(a1 - a0) : 0;
                            if (byte1 > a1)      // bytes past the tensor's last whole 16-byte chunk: ordinary loads
                                for (unsigned long long o = (a1 > byte0 ? a1 : byte0); o < byte1; o += ES)
                                    *reinterpret_cast<ST*>(dst + (o - a0)) = *reinterpret_cast<const ST*>(e.base + o);
                        }
                        const int total = warp_sum(nbytes);
                        __syncwarp();
                        if (lane == 0) mbar_arrive_expect_tx(fb, (uint32_t)total);
                        __syncwarp();
                        if (nbytes > 0) bulk_load_1d(dst, e.base + a0, (uint32_t)nbytes, fb);
                        mbar_arrive(fb);
                    }
                } else {
                    for (int n = 0; n < p.NQ; ++n) {
                        const int qn = desc ? p.NQ - 1 - n : n;
                        const int slot = qn % p.NSH;
                        mbar_wait(&empty[slot], ((pe >> slot) & 1u) ^ 1u);
                        pe ^= 1u << slot;
                        uint64_t* fb = &full[slot];
                        const unsigned long long qoff = (unsigned long long)qn * CB;
                        for (int s = pw; s < npp; s += kChNPW) {
                            const ChPlane e = tb[s];
                            const uint32_t dpl = ring + s * p.hplane + slot * CB;
                            // every chunk this plane can ask for lies inside the tensor: no per-chunk bound checks
                            const bool safe = e.b0 + HW * ES + (unsigned long long)(p.NQ + 1) * CB <= e.tbytes;
#pragma unroll
                            for (int r = 0; r < 4; ++r) {
                                if (lane + 32 * r < H) {
                                    const unsigned long long cb = ((e.b0 + rowoff[r]) & ~(unsigned long long)(CB - 1)) + qoff;
                                    const uint32_t dst = dpl + rowdst[r];
                                    if (safe || cb + CB <= e.tbytes) {
                                        cp_async_cb<CB>(dst, e.base + cb);
                                        if (slot == 0) cp_async_cb<CB>(dst + p.NSH * CB, e.base + cb);
                                    } else if (cb < e.tbytes) {
                                        uint8_t* dp = ringp + (dst - ring);
                                        for (unsigned long long o = cb; o < e.tbytes; o += ES) {
                                            const ST v = *reinterpret_cast<const ST*>(e.base + o);
                                            *reinterpret_cast<ST*>(dp + (o - cb)) = v;
                                            if (slot == 0) *reinterpret_cast<ST*>(dp + p.NSH * CB + (o - cb)) = v;
                                        }
                                    }
                                }
                            }
                        }
                        cp_async_arrive_noinc(fb);
                        __syncwarp();
                        if (lane == 0) mbar_arrive(fb);
                    }
                }
            }
        }
    } else if (warp < kChNPW + 2 * NS) {
        // ---------------- chain warps: ROLE_A (pass 1 + adjoint chain) and ROLE_F (recompute) of channel c --
        const bool roleF = warp >= kChNPW + NS;
        const int c = warp - kChNPW - (roleF ? NS : 0);
        uint32_t pf = 0;
        BlockSync bs{empty + kChSlots, empty + kChSlots + 2, 0u};
        if (!roleF) {
            if (p.q[0] >= 0) chain_bwd_dir<ST, P, false, false, ROLE_A>(p, smem, 0, b, g, c, lane, pf, bs);
            if (p.q[1] >= 0) chain_bwd_dir<ST, P, false, true, ROLE_A>(p, smem, 1, b, g, c, lane, pf, bs);
            if (p.q[2] >= 0) chain_bwd_dir<ST, P, true, false, ROLE_A>(p, smem, 2, b, g, c, lane, pf, bs);
            if (p.q[3] >= 0) chain_bwd_dir<ST, P, true, true, ROLE_A>(p, smem, 3, b, g, c, lane, pf, bs);
        } else {
            if (p.q[0] >= 0) chain_bwd_dir<ST, P, false, false, ROLE_F>(p, smem, 0, b, g, c, lane, pf, bs);
            if (p.q[1] >= 0) chain_bwd_dir<ST, P, false, true, ROLE_F>(p, smem, 1, b, g, c, lane, pf, bs);
            if (p.q[2] >= 0) chain_bwd_dir<ST, P, true, false, ROLE_F>(p, smem, 2, b, g, c, lane, pf, bs);
            if (p.q[3] >= 0) chain_bwd_dir<ST, P, true, true, ROLE_F>(p, smem, 3, b, g, c, lane, pf, bs);
        }
    } else if (warp < kChNPW + 2 * NS + kChNO) {
        // ---------------- output warp j: step j of every block, all channels -----------------------------
        const int j = warp - kChNPW - 2 * NS;
        uint32_t pf = 0;
        BlockSync bs{empty + kChSlots, empty + kChSlots + 2, 0u};
        for (int d = 0; d < 4; ++d) {
            if (p.q[d] < 0) continue;
            if (d < 2) chain_bwd_out<ST, P, false>(p, smem, d, b, g, j, lane, pf, bs);
            else       chain_bwd_out<ST, P, true>(p, smem, d, b, g, j, lane, pf, bs);
        }
    }
    __syncthreads();

    // ---------------- dx = sum over directions, one RNE, coalesced rows --------------------------------
    if (p.dx) {
        const float* DX = reinterpret_cast<const float*>(smem + p.off_dx);
        ST* dxg = reinterpret_cast<ST*>(p.dx) + ((size_t)b * sh.C + c0) * HW;
        const int nw = blockDim.x >> 5;
        for (int ci = warp; ci < NS * H; ci += nw)
            for (int j = lane; j < W; j += 32) st_f(dxg + (size_t)ci * W + j, DX[(size_t)ci * p.Wp + j]);
    }
}

// ---- host side -----------------------------------------------------------------------------------
static size_t chain_bwd_layout(const Shape& sh, int es, int P, int NSV, int NSH, ChainBwdParams* prm) {
    const int NS = sh.cg(), np = 3 + 4 * NS;
    const bool vact = sh.mask & 3u, hact = sh.mask & 12u;
    const int CB = kBlk * es;
    const int Lmax = sh.Lmax();
    size_t off = kChBars * sizeof(uint64_t);
    prm->off_tab = (uint32_t)off;
    off += (size_t)4 * kChMaxPlanes * sizeof(ChPlane);
    off = (off + 127) / 128 * 128;
    prm->Wp = sh.W | 1;
    prm->off_dx = (uint32_t)off;
    off += (size_t)NS * sh.H * prm->Wp * 4;
    off = (off + 127) / 128 * 128;
    const int over = 32 * P > sh.W ? 32 * P - sh.W : 0;        // lanes past the row end read (and discard) this much
    prm->vslot = (uint32_t)(((size_t)kBlk * sh.W * es + 32 + (size_t)over * es + 15) / 16 * 16);
    prm->vstage = (uint32_t)(np * prm->vslot);
    prm->hrow = (uint32_t)((NSH + 1) * CB);
    prm->hplane = (uint32_t)(sh.H * prm->hrow);
    prm->off_ring = (uint32_t)off;
    size_t ringb = 0;
    if (vact) ringb = (size_t)NSV * prm->vstage;
    if (hact && (size_t)np * prm->hplane + 64 > ringb) ringb = (size_t)np * prm->hplane + 64;
    // the vertical directions use the whole ring region: as many row-block stages as fit (deeper prefetch)
    prm->NSV = NSV;
    if (vact && ringb / prm->vstage > (size_t)NSV) prm->NSV = (int)(ringb / prm->vstage < (size_t)kChSlots ? ringb / prm->vstage : kChSlots);
    off += ringb;
    off = (off + 127) / 128 * 128;
    const int NBmax = (Lmax + kBlk - 1) / kBlk;
    prm->ckpt_warp = (uint32_t)((size_t)NBmax * P * 32 * 4);
    prm->off_ckpt = (uint32_t)off;
    off += (size_t)NS * prm->ckpt_warp;
    off += 128;                                                  // the output warps read one float before / after a line
    prm->off_hb = (uint32_t)off;
    off += (size_t)NS * 2 * (kBlk + 1) * P * 32 * 4;
    prm->off_gb = (uint32_t)off;
    off += (size_t)NS * 2 * kBlk * P * 32 * 4 + 128;
    prm->off_tile = (uint32_t)off;
    if (hact) off += ((size_t)(2 * NS + 3) * sh.H * kTilePitch * es + 15) / 16 * 16;
    off = (off + 15) / 16 * 16;
    prm->total = (uint32_t)off;
    return off;
}

template <typename ST, int P>
static int launch_chain_bwd(const ChainBwdParams& prm, int items, int threads, cudaStream_t st) {
    auto kern = chain_bwd_kernel<ST, P>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("chain bwd: cudaFuncSetAttribute(%u B): %s", prm.total, cudaGetErrorString(e)); return GSPN_ECUDA; }
    GSPN_LAUNCH(kern, items, threads, prm.total, st, prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("chain bwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int chain_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    const Shape& sh = a.sh;
    const int L = sh.Lmax(), NS = sh.cg();
    if (NS > kChMaxNS) { set_error("chain bwd: C/G = %d channels per group (max %d)", NS, kChMaxNS); return GSPN_EUNSUPPORTED; }
    const int P = (L + 31) / 32;
    if (P > 4) { set_error("chain bwd: max(H,W) = %d > 128", L); return GSPN_EUNSUPPORTED; }
    ChainBwdParams prm{};
    bool fit = false;
    for (int NSH = 6; NSH >= 3 && !fit; --NSH)
        for (int NSV = 4; NSV >= 2 && !fit; --NSV)
            if (NSH <= kChSlots && chain_bwd_layout(sh, ES, P, NSV, NSH, &prm) <= (size_t)kMaxSmemOptin) {
                prm.NSH = NSH;        // prm.NSV was set by the layout
                fit = true;
            }
    if (!fit) {
        set_error("chain bwd: %d channels of a %dx%d plane do not fit in shared memory", NS, sh.H, sh.W);
        return GSPN_EUNSUPPORTED;
    }
    prm.sh = sh;
    prm.x = a.x; prm.w3 = a.w3; prm.lam = a.lam; prm.u = a.u; prm.h0 = a.h0; prm.dy = a.dy;
    prm.dx = a.dx; prm.dlam = a.dlam; prm.du = a.du; prm.dw3 = a.dw3; prm.dh0 = a.dh0;
    prm.NS = NS;
    prm.NQ = (kBlk * ES - ES + sh.W * ES + kBlk * ES - 1) / (kBlk * ES);
    const unsigned long long n = (unsigned long long)sh.B * sh.C * sh.H * sh.W;
    prm.bytes_x = n * ES;
    prm.bytes_c = (unsigned long long)sh.D() * n * ES;
    prm.bytes_w = (unsigned long long)sh.D() * sh.B * sh.G * 3 * sh.H * sh.W * ES;
    int q = 0;
    for (int d = 0; d < 4; ++d) prm.q[d] = (sh.mask >> d & 1u) ? q++ : -1;
    const int threads = 32 * (kChNPW + 2 * NS + kChNO), items = sh.B * sh.G;
    int rc = GSPN_EUNSUPPORTED;
    switch (P) {
    case 1: rc = launch_chain_bwd<ST, 1>(prm, items, threads, st); break;
    case 2: rc = launch_chain_bwd<ST, 2>(prm, items, threads, st); break;
    case 3: rc = launch_chain_bwd<ST, 3>(prm, items, threads, st); break;
    case 4: rc = launch_chain_bwd<ST, 4>(prm, items, threads, st); break;
    }
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "chain_bwd"; }
    return rc;
}

template int chain_bwd_launch<float>(const BwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int chain_bwd_launch<__nv_bfloat16>(const BwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
