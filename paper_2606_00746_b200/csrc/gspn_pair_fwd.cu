// gspn_pair_fwd.cu -- whole-plane forward scan of libgspn, "plane_fwd": ONE launch,
// every direction of dir_mask and the merge over directions (Eq. 9), for small planes whose
// operands fit on chip whole (rows and planes need not be 16-byte aligned).
//
//   * a CTA owns NC channels of one (b, group) unit; every operand plane of all four directions arrives by one 1-D
//     bulk copy (16-byte-aligned superset at its byte phase, one mbarrier per direction: no rings, no gathers);
//   * ONE warp carries a channel set of its direction: P consecutive cross positions per lane and channel, the taps
//     of the group (Eq. 5) are read and widened once per line for the set, neighbours come by two
//     shuffles per line and channel;
//   * the two opposite directions of an axis add u*h (Eq. 2) into the same fp32 plane set: they never
//     touch a line at the same time (each first takes its half of the blocks, they meet once at a named barrier and
//     swap halves); one RNE at the very end.
// (Round 1 also kept a ring-staged A/B variant of this design in this file, `pair_fwd`; nothing selected it -- 0.74 ms
// against 0.59 ms for chain_fwd at the 1K config -- and it was removed in round 2.  The file keeps its name.)
#include "gspn_chain.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

constexpr int kPfR = 4;                           // image rows per vertical stage
constexpr int kPfSlots = 8;                       // mbarrier pairs per ring
constexpr int kPfNSH = 4;                         // chunk slots per row of the horizontal ring
constexpr int kPfMaxNC = 2;
constexpr int kPfBars = 4 * kPfSlots + 1;         // full[2][S], empty[2][S], x

struct PairFwdParams {
    Shape sh;
    const void *x, *w3, *lam, *u, *h0;
    void* y;
    int Wp, NSV, NQ;
    uint32_t vslot, vstage, hrow, hplane, xslot;
    uint32_t off_y, off_x, off_ring, ringb, total;
    uint32_t off_y2, off_pl, plslot;      // whole-plane kernel: second Y plane set (horizontal axis), operand planes [4][NP] of plslot bytes
    int q[4];
    unsigned long long bytes_x, bytes_c, bytes_w;
};

struct PfPlane { const uint8_t* base; unsigned long long b0, tbytes; };

// operand plane k of direction slab qd: 0..2 taps, 3+c lambda, 3+NC+c u (c = channel inside the CTA)
template <int NC, int ES>
__device__ __forceinline__ PfPlane pf_plane(const PairFwdParams& p, int qd, int b, int g, int c0, int k) {
    const Shape& sh = p.sh;
    const unsigned long long HW = (unsigned long long)sh.H * sh.W, q = (unsigned long long)qd;
    PfPlane e;
    if (k < 3) {
        e.base = (const uint8_t*)p.w3; e.tbytes = p.bytes_w;
        e.b0 = ((((q * sh.B + b) * sh.G + g) * 3 + k) * HW) * ES;
    } else {
        const int t = (k - 3) / NC, c = (k - 3) % NC;
        e.base = (const uint8_t*)(t == 0 ? p.lam : p.u); e.tbytes = p.bytes_c;
        e.b0 = (((q * sh.B + b) * sh.C + c0 + c) * HW) * ES;
    }
    return e;
}

template <typename ST> struct PfTap;
template <> struct PfTap<__nv_bfloat16> {           // widen and mask a tap in one PRMT
    static __device__ __forceinline__ uint32_t sel(bool keep) { return keep ? 0x1044u : 0x4444u; }
    static __device__ __forceinline__ float wm(unsigned short r, uint32_t s) {
        return __uint_as_float(__byte_perm((uint32_t)r, 0u, s));
    }
};
template <> struct PfTap<float> {
    static __device__ __forceinline__ uint32_t sel(bool keep) { return keep ? 0xffffffffu : 0u; }
    static __device__ __forceinline__ float wm(float r, uint32_t s) { return __uint_as_float(__float_as_uint(r) & s); }
};

// named barrier of the two warps of an axis and channel set (ids 1.. vertical, 8.. horizontal: the axes of the
// whole-plane kernel run at the same time)
template <bool SECOND = false> __device__ __forceinline__ void pf_pair_bar(int set = 0) {
    if constexpr (SECOND) named_bar_sync(8 + set, 64);
    else named_bar_sync(1 + set, 64);
}

// One direction, all NC channels of the CTA, on one warp.  VH = false: T->B / B->T (lanes own columns), true:
// L->R / R->L (lanes own rows); REV = the direction walks the image lines downwards.
// WHOLE = false: operands come through the rings of this file's producer warps; true (plane_fwd_kernel): every
// operand plane of the direction already lies in shared memory as a whole (16-byte-aligned superset at its byte
// phase), the two axes run at the same time on two Y plane sets and meet at their own named barriers.
// NCC = channels of the CTA (layout of the operand planes), NC = channels of this warp, the CTA's channels
// [cw, cw + NC): the whole-plane kernel splits a direction's channels over NCC / NC warps.
template <typename ST, int P, int NC, bool VH, bool REV, bool WHOLE = false, int NCC = NC>
__device__ __forceinline__ void pair_fwd_dir(const PairFwdParams& p, uint8_t* smem, const int qd, const int b,
                                             const int g, const int c0, const int lane, uint32_t& pf,
                                             const bool pair_sync, const int d = 0, const int cw = 0) {
    using E = Elem<ST>;
    using T = PfTap<ST>;
    using raw_t = typename E::raw_t;
    constexpr int ES = sizeof(ST), NP = 3 + 2 * NC;
    constexpr int CB = ES == 2 ? 8 : 16;
    constexpr int BLK = (VH && !WHOLE) ? CB / ES : kPfR;   // scan steps per block (= ring stage)
    constexpr unsigned FULLM = 0xffffffffu;
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W;
    const int Ls = VH ? W : H, Lp = VH ? H : W, Lmax = sh.Lmax();
    const int NB = (Ls + BLK - 1) / BLK, mb = NB / 2;
    const uint32_t rowB = (uint32_t)W * ES;
    const int pr = REV ? 1 : 0;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    const uint32_t ring = smem_u32(smem + p.off_ring) + pr * p.ringb;
    RingSync<VH> rs{bars + pr * kPfSlots, bars + (2 + pr) * kPfSlots, p.NSV, kPfNSH, p.NQ, lane, 0, pf};

    bool ok[P];
    uint32_t okm[P], s_w0, s_w2[P];
#pragma unroll
    for (int e = 0; e < P; ++e) {
        ok[e] = P * lane + e < Lp;
        okm[e] = ok[e] ? 0xffffffffu : 0u;
        s_w2[e] = T::sel(P * lane + e != Lp - 1);                  // out-of-grid taps are never used
    }
    s_w0 = T::sel(lane != 0);

    // operand addresses: vertical = byte phase of every plane (the block offset is added per stage);
    // horizontal = ring row of every (plane, own row) plus that row's byte phase inside its first chunk
    uint32_t ph[NP], vb[NP], hb[NP][P], xb[NC][P], yb[NC][P];
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        // plane index inside the CTA's set: taps, lambda of channel cw + c, u of channel cw + c
        const int kc = k < 3 ? k : (k < 3 + NC ? k + cw : k - NC + NCC + cw);
        const unsigned long long b0 = pf_plane<NCC, ES>(p, qd, b, g, c0, kc).b0;
        ph[k] = (uint32_t)(b0 & 15ull); vb[k] = 0;
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const int row = min(P * lane + e, H - 1);             // rows past the plane re-read the last row
            hb[k][e] = ring + k * p.hplane + row * p.hrow + (uint32_t)((b0 + (unsigned long long)row * rowB) % CB);
            if constexpr (WHOLE) {      // plane k of direction d, element (own cross position, scan step 0)
                const int pos = min(P * lane + e, Lp - 1);
                hb[k][e] = smem_u32(smem + p.off_pl) + (uint32_t)(d * (3 + 2 * NCC) + kc) * p.plslot + ph[k] +
                           (VH ? (uint32_t)pos * rowB : (uint32_t)(P * lane + e) * ES);
            }
        }
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const unsigned long long xb0 = (((unsigned long long)b * sh.C + c0 + cw + c) * H * W) * ES;
        const uint32_t xs = smem_u32(smem + p.off_x) + (cw + c) * p.xslot + (uint32_t)(xb0 & 15ull);
        const uint32_t ys = smem_u32(smem + ((WHOLE && VH) ? p.off_y2 : p.off_y)) + (uint32_t)(cw + c) * H * p.Wp * 4;
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const int pos = min(P * lane + e, Lp - 1);
            xb[c][e] = VH ? xs + pos * rowB : xs + (P * lane + e) * ES;
            yb[c][e] = VH ? ys + (uint32_t)pos * p.Wp * 4 : ys + (P * lane + e) * 4;
        }
    }

    float h[NC][P];
#pragma unroll
    for (int c = 0; c < NC; ++c)
#pragma unroll
        for (int e = 0; e < P; ++e) {
            h[c][e] = 0.f;
            if (p.h0 && ok[e])
                h[c][e] = ld_f(reinterpret_cast<const ST*>(p.h0) +
                               (((size_t)qd * sh.B + b) * sh.C + c0 + cw + c) * Lmax + P * lane + e);
        }

    if constexpr (WHOLE) mbar_wait(bars + d, 0);                    // this direction's planes have landed
    else rs.begin_pass(REV);
    for (int n = 0; n < NB; ++n) {
        const int bi = REV ? NB - 1 - n : n;
        if (REV && pair_sync && bi == mb) pf_pair_bar<WHOLE && VH>(cw / NC);   // the upward warp is done with blocks <= mb
        const int s0 = BLK * bi, nb = min(BLK, Ls - s0);
        if constexpr (!WHOLE) rs.acquire(bi, REV);
        uint32_t ao[NP][P], ax[NC][P];                              // this block's operand addresses (step 0)
        if constexpr (WHOLE) {
            const uint32_t so = (uint32_t)s0 * (VH ? (uint32_t)ES : rowB);
#pragma unroll
            for (int k = 0; k < NP; ++k)
#pragma unroll
                for (int e = 0; e < P; ++e) ao[k][e] = hb[k][e] + so;
#pragma unroll
            for (int c = 0; c < NC; ++c)
#pragma unroll
                for (int e = 0; e < P; ++e) ax[c][e] = xb[c][e] + so;
        } else if constexpr (!VH) {
            const uint32_t stage = ring + (bi % p.NSV) * p.vstage;
            const uint32_t rb = ((uint32_t)s0 * rowB) & 15u;
#pragma unroll
            for (int k = 0; k < NP; ++k) {
                vb[k] = stage + k * p.vslot + ((ph[k] + rb) & 15u) + lane * (P * ES);
#pragma unroll
                for (int e = 0; e < P; ++e) ao[k][e] = vb[k] + e * ES;
            }
#pragma unroll
            for (int c = 0; c < NC; ++c)
#pragma unroll
                for (int e = 0; e < P; ++e) ax[c][e] = xb[c][e] + (uint32_t)s0 * rowB;
        } else {
            const uint32_t so = ((uint32_t)bi * CB) & (kPfNSH * CB - 1);
#pragma unroll
            for (int k = 0; k < NP; ++k)
#pragma unroll
                for (int e = 0; e < P; ++e) ao[k][e] = hb[k][e] + so;
#pragma unroll
            for (int c = 0; c < NC; ++c)
#pragma unroll
                for (int e = 0; e < P; ++e) ax[c][e] = xb[c][e] + (uint32_t)s0 * ES;
        }
        const uint32_t step = VH ? (uint32_t)ES : rowB;             // bytes from one scan step to the next

        raw_t wr[2][3][P], lr[2][NC][P], xr[2][NC][P], ur[BLK][NC][P];
        float hs[BLK][NC][P];
        auto load = [&](int buf, int tl) {
            const uint32_t o = tl * step;
#pragma unroll
            for (int e = 0; e < P; ++e) {
#pragma unroll
                for (int k = 0; k < 3; ++k) wr[buf][k][e] = E::lds(ao[k][e] + o);
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    lr[buf][c][e] = E::lds(ao[3 + c][e] + o);
                    xr[buf][c][e] = E::lds(ax[c][e] + o);
                    ur[tl][c][e] = E::lds(ao[3 + NC + c][e] + o);
                }
            }
        };
        load(0, REV ? BLK - 1 : 0);
#pragma unroll
        for (int t = 0; t < BLK; ++t) {
            const int tl = REV ? BLK - 1 - t : t;
            const int buf = t & 1;
            if (t + 1 < BLK) load(buf ^ 1, REV ? tl - 1 : tl + 1);
            if (tl < nb) {
                float w0f[P], w1f[P], w2f[P];
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    w0f[e] = e == 0 ? T::wm(wr[buf][0][e], s_w0) : E::f(wr[buf][0][e]);
                    w1f[e] = E::f(wr[buf][1][e]);
                    w2f[e] = T::wm(wr[buf][2][e], s_w2[e]);
                }
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const float hl = __shfl_up_sync(FULLM, h[c][P - 1], 1);      // lane 0: w0f[0] is masked
                    const float hr = __shfl_down_sync(FULLM, h[c][0], 1);        // lane 31: masked by s_w2 / okm
                    float hn[P];
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        const float left = e ? h[c][e - 1] : hl;
                        const float right = e < P - 1 ? h[c][e + 1] : hr;
                        float acc = w1f[e] * h[c][e];
                        acc = fmaf(w0f[e], left, acc);
                        acc = fmaf(w2f[e], right, acc);
                        acc = E::fma2(lr[buf][c][e], xr[buf][c][e], acc);
                        hn[e] = maskf(acc, okm[e]);                              // positions past the line stay +0
                    }
#pragma unroll
                    for (int e = 0; e < P; ++e) { h[c][e] = hn[e]; hs[tl][c][e] = hn[e]; }
                }
            }
        }
        // Y += u*h for the whole block (single writer: see the header): all reads first, then all writes, so the
        // shared-memory round trips overlap instead of serialising read -> write -> read
        float yo[BLK][NC][P];
#pragma unroll
        for (int tl = 0; tl < BLK; ++tl)
#pragma unroll
            for (int c = 0; c < NC; ++c)
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    const uint32_t a = yb[c][e] + (VH ? (uint32_t)(s0 + tl) * 4 : (uint32_t)(s0 + tl) * p.Wp * 4);
                    if (tl < nb && ok[e]) yo[tl][c][e] = lds32(a);
                }
#pragma unroll
        for (int tl = 0; tl < BLK; ++tl)
#pragma unroll
            for (int c = 0; c < NC; ++c)
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    const uint32_t a = yb[c][e] + (VH ? (uint32_t)(s0 + tl) * 4 : (uint32_t)(s0 + tl) * p.Wp * 4);
                    if (tl < nb && ok[e]) sts32(a, fmaf(E::f(ur[tl][c][e]), hs[tl][c][e], yo[tl][c][e]));
                }
        if constexpr (!WHOLE) rs.release(bi, REV, n == NB - 1);
        if (!REV && pair_sync && bi == mb) pf_pair_bar<WHOLE && VH>(cw / NC);   // blocks <= mb are finished: swap halves
    }
    pf = rs.pf;
}

// ---------------------------------------------------------------------------------------------------
// Whole-plane variant for small planes (the 378-px config's 27x27 and the like): every operand plane of the CTA's
// NC channels and of all four directions is brought in by ONE bulk copy each (no rings, no gathers, no hand-shakes
// beyond one mbarrier per direction), the four directions run at the same time on four warps: T->B / B->T share
// the Y plane set of the vertical axis, L->R / R->L the one of the horizontal axis (half-swap as above), and
// y = Yv + Yh is rounded once at the end.
__device__ __forceinline__ int pf_bulk_window(uint8_t* dst, const uint8_t* base, unsigned long long byte0,
                                              unsigned long long nbytes_plane, unsigned long long tbytes, int es,
                                              unsigned long long* a0_out) {
    const unsigned long long byte1 = byte0 + nbytes_plane;
    const unsigned long long a0 = byte0 & ~15ull, lim = tbytes & ~15ull;
    unsigned long long a1 = (byte1 + 15) & ~15ull;
    if (a1 > lim) a1 = lim;
    if (byte1 > a1)          // bytes past the tensor's last whole 16-byte chunk: ordinary loads
        for (unsigned long long o = (a1 > byte0 ? a1 : byte0); o < byte1; o += es) {
            if (es == 2) *reinterpret_cast<unsigned short*>(dst + (o - a0)) = *reinterpret_cast<const unsigned short*>(base + o);
            else *reinterpret_cast<float*>(dst + (o - a0)) = *reinterpret_cast<const float*>(base + o);
        }
    *a0_out = a0;
    return a1 > a0 ? (int)(a1 - a0) : 0;
}

template <typename ST, int P, int NC, int NCW>
__global__ void __launch_bounds__(32 * (4 * (NC / NCW) + 1))
plane_fwd_kernel(const PairFwdParams p) {
    constexpr int ES = sizeof(ST), NP = 3 + 2 * NC;
    constexpr int NCMP = 4 * (NC / NCW);                          // compute warps: (direction, channel set)
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);           // [0..3] direction planes, [4] x
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int slices = sh.cg() / NC;
    const int b = blockIdx.x / (sh.G * slices);
    const int g = (blockIdx.x / slices) % sh.G;
    const int c0 = g * sh.cg() + (blockIdx.x % slices) * NC;
    const unsigned long long HW = (unsigned long long)H * W;

    {   // both Y plane sets accumulate from zero
        uint8_t* yz = smem + p.off_y;
        const uint32_t ybytes = p.off_x - p.off_y;
        for (uint32_t o = threadIdx.x * 16; o < ybytes; o += blockDim.x * 16)
            *reinterpret_cast<uint4*>(yz + o) = make_uint4(0, 0, 0, 0);
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < 4; ++s) mbar_init(&bars[s], NP);           // one arrival per operand plane
        mbar_init(&bars[4], NC);
        mbar_init_fence();
    }
    __syncthreads();

    const bool act[4] = {p.q[0] >= 0, p.q[1] >= 0, p.q[2] >= 0, p.q[3] >= 0};
    if (warp == NCMP) {
        // every plane has its own lane (x first: every direction needs it, then the directions in the order the
        // warps consume them); a lane announces its bytes on the plane's barrier and issues the copy at once, so
        // all copies of the CTA are in flight after two rounds
        for (int i = lane; i < NC + 4 * NP; i += 32) {
            const int t = i < NC ? -1 : (i - NC) / NP, k = i < NC ? i : (i - NC) % NP;
            if (t >= 0 && !act[t]) continue;
            unsigned long long a0 = 0;
            const uint8_t* base;
            uint8_t* dst;
            int nbytes;
            if (t < 0) {
                base = (const uint8_t*)p.x;
                dst = smem + p.off_x + (size_t)k * p.xslot;
                nbytes = pf_bulk_window(dst, base, (((unsigned long long)b * sh.C + c0 + k) * HW) * ES, HW * ES,
                                        p.bytes_x, ES, &a0);
            } else {
                const PfPlane e = pf_plane<NC, ES>(p, p.q[t], b, g, c0, k);
                base = e.base;
                dst = smem + p.off_pl + (size_t)(t * NP + k) * p.plslot;
                nbytes = pf_bulk_window(dst, base, e.b0, HW * ES, e.tbytes, ES, &a0);
            }
            uint64_t* fb = &bars[t < 0 ? 4 : t];
            mbar_arrive_expect_tx(fb, (uint32_t)nbytes);             // also publishes the tail bytes written above
            if (nbytes > 0) bulk_load_1d(dst, base + a0, (uint32_t)nbytes, fb);
        }
    } else {
        uint32_t pf = 0;
        mbar_wait(&bars[4], 0);
        const int d = warp & 3, cw = (warp >> 2) * NCW;            // one direction per scheduler
        if (d == 0 && act[0]) pair_fwd_dir<ST, P, NCW, false, false, true, NC>(p, smem, p.q[0], b, g, c0, lane, pf, act[1], 0, cw);
        if (d == 1 && act[1]) pair_fwd_dir<ST, P, NCW, false, true, true, NC>(p, smem, p.q[1], b, g, c0, lane, pf, act[0], 1, cw);
        if (d == 2 && act[2]) pair_fwd_dir<ST, P, NCW, true, false, true, NC>(p, smem, p.q[2], b, g, c0, lane, pf, act[3], 2, cw);
        if (d == 3 && act[3]) pair_fwd_dir<ST, P, NCW, true, true, true, NC>(p, smem, p.q[3], b, g, c0, lane, pf, act[2], 3, cw);
    }
    __syncthreads();

    // ---------------- y = Yv + Yh, one RNE, coalesced rows ------------------------------------------------
    {
        const float* Yv = reinterpret_cast<const float*>(smem + p.off_y);
        const float* Yh = reinterpret_cast<const float*>(smem + p.off_y2);
        ST* yg = reinterpret_cast<ST*>(p.y) + ((size_t)b * sh.C + c0) * HW;
        if (p.Wp == W) {
            // odd W: the Y planes have the pitch of the image rows, so the CTA's NC output planes are one
            // contiguous run both on chip and in HBM
            const int total = NC * H * W;
            for (int idx = threadIdx.x; idx < total; idx += 32 * (NCMP + 1)) st_f(yg + idx, Yv[idx] + Yh[idx]);
        } else {
            for (int ci = warp; ci < NC * H; ci += NCMP + 1)
                for (int j = lane; j < W; j += 32)
                    st_f(yg + (size_t)ci * W + j, Yv[(size_t)ci * p.Wp + j] + Yh[(size_t)ci * p.Wp + j]);
        }
    }
}

static size_t plane_fwd_layout(const Shape& sh, int es, int P, int NC, PairFwdParams* prm) {
    const int np = 3 + 2 * NC;
    size_t off = 128;                                           // 5 mbarriers
    prm->Wp = sh.W | 1;
    const size_t yset = ((size_t)NC * sh.H * prm->Wp * 4 + 127) / 128 * 128;
    prm->off_y = (uint32_t)off;
    prm->off_y2 = (uint32_t)(off + yset);
    off += 2 * yset;
    prm->off_x = (uint32_t)off;
    prm->xslot = (uint32_t)(((size_t)sh.H * sh.W * es + 32 + 15) / 16 * 16);
    off += (size_t)NC * prm->xslot;
    prm->off_pl = (uint32_t)off;
    prm->plslot = prm->xslot;
    off += (size_t)4 * np * prm->plslot;
    // discarded reads past the last plane: lanes past a row's end, lines past the last block
    off += (size_t)32 * P * es + (size_t)kPfR * sh.Lmax() * es + 64;
    off = (off + 15) / 16 * 16;
    prm->total = (uint32_t)off;
    return off;
}

template <typename ST, int P, int NC, int NCW>
static int launch_plane_fwd(const PairFwdParams& prm, int items, cudaStream_t st) {
    auto kern = plane_fwd_kernel<ST, P, NC, NCW>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("plane fwd: cudaFuncSetAttribute(%u B): %s", prm.total, cudaGetErrorString(e)); return GSPN_ECUDA; }
    GSPN_LAUNCH(kern, items, 32 * (4 * (NC / NCW) + 1), prm.total, st, prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("plane fwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int plane_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    const Shape& sh = a.sh;
    const int L = sh.Lmax(), cg = sh.cg();
    const int P = (L + 31) / 32;
    if (P > 2) { set_error("plane fwd: max(H,W) = %d > 64", L); return GSPN_EUNSUPPORTED; }
    // channels per warp: as many as share the taps (4, 2, 1) while at least two CTAs fit an SM
    PairFwdParams prm{};
    int NC = 0;
    for (int nc = 4; nc >= 1; nc /= 2) {
        if (cg % nc) continue;
        if (P * nc > 4) continue;                              // at most 4 recurrences per lane (registers)
        if (2 * (plane_fwd_layout(sh, ES, P, nc, &prm) + 1024) <= (size_t)228 * 1024) { NC = nc; break; }
    }
    if (!NC) {
        set_error("plane fwd: the planes of a %dx%d unit do not fit in shared memory twice per SM", sh.H, sh.W);
        return GSPN_EUNSUPPORTED;
    }
    prm.sh = sh;
    prm.x = a.x; prm.w3 = a.w3; prm.lam = a.lam; prm.u = a.u; prm.h0 = a.h0; prm.y = a.y;
    const unsigned long long n = (unsigned long long)sh.B * sh.C * sh.H * sh.W;
    prm.bytes_x = n * ES;
    prm.bytes_c = (unsigned long long)sh.D() * n * ES;
    prm.bytes_w = (unsigned long long)sh.D() * sh.B * sh.G * 3 * sh.H * sh.W * ES;
    int q = 0;
    for (int d = 0; d < 4; ++d) prm.q[d] = (sh.mask >> d & 1u) ? q++ : -1;
    const int items = sh.B * sh.G * (cg / NC);
    int rc = GSPN_EUNSUPPORTED;
    // channels per warp: 2 share the taps; a CTA's other channels go to more warps (measured on the 378-px
    // config, B200: 4 channels per warp 0.369 ms, 2 per warp 0.327 ms, 1 per warp 0.348 ms)
    const int ncw = NC < 2 ? NC : 2;
#define GSPN_PL(PP, NCC, NW) launch_plane_fwd<ST, PP, NCC, NW>(prm, items, st)
    if (P == 1) {
        if (NC == 4) rc = ncw == 4 ? GSPN_PL(1, 4, 4) : ncw == 2 ? GSPN_PL(1, 4, 2) : GSPN_PL(1, 4, 1);
        else if (NC == 2) rc = ncw == 2 ? GSPN_PL(1, 2, 2) : GSPN_PL(1, 2, 1);
        else rc = GSPN_PL(1, 1, 1);
    } else {
        if (NC == 2) rc = ncw == 2 ? GSPN_PL(2, 2, 2) : GSPN_PL(2, 2, 1);
        else rc = GSPN_PL(2, 1, 1);
    }
#undef GSPN_PL
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "plane_fwd"; }
    return rc;
}

template int plane_fwd_launch<float>(const FwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int plane_fwd_launch<__nv_bfloat16>(const FwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
