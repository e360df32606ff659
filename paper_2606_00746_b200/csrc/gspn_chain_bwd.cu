// gspn_chain_bwd.cu -- fused backward scan of libgspn, "chain" design:
// ONE launch, one CTA per (b, group) unit, one WARP per channel of the group.
//
// The adjoint recurrence (include/gspn.h "Backward scan"; derived from Eq. 1-2,
// the paper reports backward timings only).  Per direction the
// warp of channel c makes two passes over the scan line blocks of kBlk = 4 steps:
//   pass 1 (scan order)    h[s] = w[s] h[s-1] + lambda[s]*x[s], h in registers, the state entering
//                          each block kept as a checkpoint in shared memory (fp32);
//   pass 2 (reverse order) per block: h of the block's steps recomputed from its checkpoint into
//                          registers, then gh[s] = dy[s]*u[s] + carry; du = dy*h[s];
//                          dlambda = x*gh; dx += lambda*gh; dw3[k] partial = gh * h[s-1, p+k-1];
//                          carry = w[s]^T gh  (neighbours by warp shuffle, no block barrier).
// dx of the group's channels is accumulated over the directions in an fp32 plane per channel on chip
// (the directions run one after another, so the plane has a single writer) and rounded once at the
// end.  dw3 (Eq. 5: taps shared by the channels of a group) is reduced over the
// channels through a small exchange buffer once per block, in ascending channel order (deterministic,
// no atomics).  Vertical outputs are stored straight from registers (lanes own consecutive columns);
// horizontal outputs go through 8-column tiles so that every store instruction writes 16-byte row
// pieces (the transposed tile on the way out).
//
// Operands: gspn_chain.cuh.  One producer warp streams, for the current direction and pass, a ring of
// stages: for T->B / B->T a block of 4 image rows of every operand plane (one 1-D bulk copy per plane
// over its 16-byte-aligned superset), for L->R / R->L one chunk column (4 columns of every row of
// every plane, cp.async of the aligned chunk; a row keeps NSH+1 chunk slots contiguous, slot NSH
// mirrors slot 0, so the two chunks a block of 4 columns touches are always contiguous).
#include "gspn_chain.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

constexpr int kChMaxNS = 8;                       // channels per group the kernel takes
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
    uint32_t off_tab, off_dx, off_ring, off_ckpt, off_exch, off_tile, off_dwtile, total;
    uint32_t ckpt_warp, tile_warp;  // bytes per chain warp
    int q[4];                       // slab index of each direction, -1 = not in dir_mask
    unsigned long long bytes_x, bytes_c, bytes_w;
};

enum { KW0 = 0, KW1, KW2, KLAM, KX, KU, KDY, KNUM };

__device__ __forceinline__ float maskf(float v, uint32_t m) { return __uint_as_float(__float_as_uint(v) & m); }
__device__ __forceinline__ float lds32(uint32_t a) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v)); }

// ---------------------------------------------------------------------------------------------------
// One direction of one channel: the warp-level adjoint scan.  VH = false: T->B / B->T (lanes own
// columns), true: L->R / R->L (lanes own rows); REV = the direction walks the image lines downwards.
// Lane-dependent conditions (position inside the line, first / last position) are 32-bit AND masks in
// ordinary registers, not predicates: values of positions past the line are forced to +0 exactly.
template <typename ST, int P, bool VH, bool REV>
__device__ __forceinline__ void chain_bwd_dir(const ChainBwdParams& p, uint8_t* smem, const int d, const int b,
                                              const int g, const int c, const int lane, uint32_t& pf) {
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
    const size_t HW = (size_t)H * W;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    uint64_t* empty = full + kChSlots;
    const ChPlane* tb = reinterpret_cast<const ChPlane*>(smem + p.off_tab) + d * kChMaxPlanes;
    const uint32_t ring = smem_u32(smem + p.off_ring);
    const int sidx[KNUM] = {0, 1, 2, 3 + c, 3 + NS + c, 3 + 2 * NS + c, 3 + 3 * NS + c};

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
    const size_t pw = (((size_t)qd * sh.B + b) * sh.G + g) * 3;                // first tap plane in [D,B,G,3]
    const bool w_du = p.du != nullptr, w_dl = p.dlam != nullptr, w_dw = p.dw3 != nullptr, w_dx = p.dx != nullptr;
    // this lane's first element of each output plane (vertical: column P*lane, horizontal: see the tile write-out)
    ST* du_l = reinterpret_cast<ST*>(p.du) + pc * HW + (VH ? 0 : P * lane);
    ST* dl_l = reinterpret_cast<ST*>(p.dlam) + pc * HW + (VH ? 0 : P * lane);
    ST* dw_l = reinterpret_cast<ST*>(p.dw3) + pw * HW + (VH ? 0 : P * lane);
    const uint32_t dxs = smem_u32(smem + p.off_dx) + (uint32_t)c * H * p.Wp * 4;               // this channel's fp32 dx plane
    const uint32_t cks = smem_u32(smem + p.off_ckpt) + c * p.ckpt_warp + lane * 4;             // [NB][P][32]
    const uint32_t exs = smem_u32(smem + p.off_exch) + lane * 4;                               // [NS][3][kBlk][P][32]
    const uint32_t exw = exs + (uint32_t)c * 3 * kBlk * P * 128;
    const uint32_t tile = smem_u32(smem + p.off_tile) + c * p.tile_warp;                       // [2][Lp][kTilePitch]
    const uint32_t dwtile = smem_u32(smem + p.off_dwtile);                                     // [3][Lp][kTilePitch]
    const uint32_t tplane = (uint32_t)Lp * kTilePitch * ES;

    // operand addresses inside the ring
    uint32_t phs[KNUM];          // vertical: byte phase (mod 16) of each plane
    uint32_t vb[KNUM];           // vertical: per block, address of (local line 0, this lane's first column)
    uint32_t hb[KNUM][P];        // horizontal: address of (this lane's row e, chunk slot 0) + the row's byte phase
    uint32_t dxh[P], tlh[P];     // horizontal: dx / tile row addresses of this lane's rows
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
            dxh[e] = dxs + (uint32_t)row * p.Wp * 4;
            tlh[e] = tile + (uint32_t)row * kTilePitch * ES;
        }
    }
    // address of element e of operand k on image-local line tl of the current block
    // (plain loads: the scheduler may hoist them over the asm stores of the previous step; the mbarrier
    //  waits / arrives carry memory clobbers and keep them inside the stage's lifetime)
    const uint8_t* const sbase = smem - smem_u32(smem);           // generic address of shared offset 0
    auto ldr = [&](int k, int tl, uint32_t so, int e) -> raw_t {
        if constexpr (!VH) return *reinterpret_cast<const raw_t*>(sbase + (vb[k] + tl * rowB + e * ES));
        else return *reinterpret_cast<const raw_t*>(sbase + (hb[k][e] + so + tl * ES));
    };

    // ring hand-shake: block bi needs row block bi (vertical) / chunk columns bi and bi+1 (horizontal)
    int hq = 0;
    auto wait_full = [&](int slot) {
        mbar_wait(&full[slot], (pf >> slot) & 1u);
        pf ^= 1u << slot;
    };
    auto begin_pass = [&](bool desc) { hq = desc ? p.NQ - 1 : 0; };
    auto acquire = [&](int bi, bool desc) {
        if constexpr (!VH) {
            wait_full(bi % p.NSV);
        } else if (!desc) {
            const int need = min(bi + 1, p.NQ - 1);
            for (; hq <= need; ++hq) wait_full(hq % p.NSH);
        } else {
            for (; hq >= bi; --hq) wait_full(hq % p.NSH);
        }
    };
    auto release = [&](int bi, bool desc, bool last) {
        __syncwarp();
        if (lane == 0) {
            if constexpr (!VH) {
                mbar_arrive(&empty[bi % p.NSV]);
            } else if (!desc) {
                mbar_arrive(&empty[bi % p.NSH]);
                if (last) for (int qq = bi + 1; qq < p.NQ; ++qq) mbar_arrive(&empty[qq % p.NSH]);
            } else {
                if (bi + 1 < p.NQ) mbar_arrive(&empty[(bi + 1) % p.NSH]);
                if (last) mbar_arrive(&empty[bi % p.NSH]);
            }
        }
    };
    auto block_setup = [&](int bi) -> uint32_t {        // returns the block's chunk-slot offset (horizontal)
        if constexpr (!VH) {
            const uint32_t stage = ring + (bi % p.NSV) * p.vstage;
            const uint32_t rb = ((uint32_t)(kBlk * bi) * rowB) & 15u;
#pragma unroll
            for (int k = 0; k < KNUM; ++k)
                vb[k] = stage + sidx[k] * p.vslot + ((phs[k] + rb) & 15u) + lane * (P * ES);
            return 0u;
        } else {
            return (uint32_t)(bi % p.NSH) * CB;
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

    // ================= pass 1: scan order, checkpoints =================================================
    float h[P];
#pragma unroll
    for (int e = 0; e < P; ++e) {
        h[e] = 0.f;
        if (p.h0 && ok[e]) h[e] = ld_f(reinterpret_cast<const ST*>(p.h0) + pc * Lmax + P * lane + e);
    }
    begin_pass(REV);
    for (int n = 0; n < NB; ++n) {
        const int bi = REV ? NB - 1 - n : n;
        const int nb = min(kBlk, Ls - kBlk * bi);
        acquire(bi, REV);
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
        release(bi, REV, n == NB - 1);
    }

    // ================= pass 2: reverse order ===========================================================
    constexpr bool desc2 = !REV;
    float carry[P];
#pragma unroll
    for (int e = 0; e < P; ++e) carry[e] = 0.f;
    begin_pass(desc2);
    for (int n = 0; n < NB; ++n) {
        const int bi = desc2 ? NB - 1 - n : n;
        const int nb = min(kBlk, Ls - kBlk * bi);
        acquire(bi, desc2);
        const uint32_t so = block_setup(bi);
        float hs[kBlk + 1][P];                  // hs[t] = state entering the t-th step (scan order) of the block
#pragma unroll
        for (int e = 0; e < P; ++e) hs[0][e] = lds32(cks + (bi * P + e) * 128);
#pragma unroll
        for (int t = 0; t < kBlk; ++t) {
            const int tl = REV ? kBlk - 1 - t : t;
            if (tl < nb) {
                fwd_step(hs[t], tl, so, hs[t + 1]);
            } else {
#pragma unroll
                for (int e = 0; e < P; ++e) hs[t + 1][e] = hs[t][e];
            }
        }
        // per-block output / accumulator addresses
        const int l0 = kBlk * bi;                                   // first image line of the block
        uint32_t dxv = 0, thb = 0;
        ST *du_b = nullptr, *dl_b = nullptr;
        if constexpr (!VH) {
            dxv = dxs + ((uint32_t)l0 * p.Wp + P * lane) * 4;
            du_b = du_l + (size_t)l0 * W;
            dl_b = dl_l + (size_t)l0 * W;
        } else {
            thb = (uint32_t)((bi & 1) * kBlk) * ES;
        }
#pragma unroll
        for (int tt = 0; tt < kBlk; ++tt) {
            const int t = kBlk - 1 - tt;
            const int tl = REV ? kBlk - 1 - t : t;
            if (tl < nb) {
                raw_t w0r[P], w1r[P], w2r[P], lr[P], xr[P], ur[P], dyr[P];
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    ur[e] = ldr(KU, tl, so, e); dyr[e] = ldr(KDY, tl, so, e);
                    lr[e] = ldr(KLAM, tl, so, e); xr[e] = ldr(KX, tl, so, e);
                    w0r[e] = ldr(KW0, tl, so, e); w1r[e] = ldr(KW1, tl, so, e); w2r[e] = ldr(KW2, tl, so, e);
                }
                float gh[P];
#pragma unroll
                for (int e = 0; e < P; ++e) gh[e] = maskf(E::fma2(dyr[e], ur[e], carry[e]), okm[e]);
                // du, dlambda
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    const raw_t duv = E::pack(E::f(dyr[e]) * hs[t + 1][e]);
                    const raw_t dlv = E::pack(E::f(xr[e]) * gh[e]);
                    if constexpr (!VH) {
                        if (w_du && ok[e]) E::stg(du_b + tl * W + e, duv);
                        if (w_dl && ok[e]) E::stg(dl_b + tl * W + e, dlv);
                    } else {
                        if (w_du && ok[e]) E::sts(tlh[e] + thb + tl * ES, duv);
                        if (w_dl && ok[e]) E::sts(tlh[e] + tplane + thb + tl * ES, dlv);
                    }
                }
                // dx += lambda * gh
                if (w_dx) {
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        const uint32_t a = VH ? dxh[e] + (l0 + tl) * 4 : dxv + (tl * p.Wp + e) * 4;
                        if (ok[e]) sts32(a, fmaf(E::f(lr[e]), gh[e], lds32(a)));
                    }
                }
                // dw3 partials of this channel: gh * h[s-1, p+k-1]
                if (w_dw) {
                    const float hpl = maskf(__shfl_up_sync(FULLM, hs[t][P - 1], 1), m_first);
                    const float hpr = maskf(__shfl_down_sync(FULLM, hs[t][0], 1), m_31);
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        const float left = e ? hs[t][e - 1] : hpl;
                        const float right = e < P - 1 ? hs[t][e + 1] : hpr;
                        const uint32_t a = exw + (tl * P + e) * 128;
                        sts32(a, gh[e] * left);
                        sts32(a + kBlk * P * 128, gh[e] * hs[t][e]);
                        sts32(a + 2 * kBlk * P * 128, gh[e] * right);
                    }
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
        // dw3 of the block: sum over the group's channels in ascending order, one RNE
        if (w_dw) {
            if (NS > 1) chain_bar(NS * 32); else __syncwarp();
            for (int kt = c; kt < 3 * kBlk; kt += NS) {
                const int k = kt / kBlk, tl = kt % kBlk;
                if (tl < nb) {
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        const uint32_t a = exs + ((k * kBlk + tl) * P + e) * 128;
                        float sum = lds32(a);
                        for (int s = 1; s < NS; ++s) sum += lds32(a + s * (3 * kBlk * P * 128));
                        if constexpr (!VH) {
                            if (ok[e]) E::stg(dw_l + (size_t)k * HW + (size_t)(l0 + tl) * W + e, E::pack(sum));
                        } else {
                            const int row = P * lane + e;
                            if (ok[e]) E::sts(dwtile + ((k * Lp + row) * kTilePitch) * ES + thb + tl * ES, E::pack(sum));
                        }
                    }
                }
            }
            if (NS > 1) chain_bar(NS * 32); else __syncwarp();
        }
        // horizontal outputs: a pair of blocks = 8 columns is complete -> 16-byte row pieces to global
        if constexpr (VH) {
            const bool pair_done = desc2 ? ((bi & 1) == 0) : ((bi & 1) == 1 || bi == NB - 1);
            if (pair_done) {
                const int col0 = 2 * kBlk * (bi >> 1);
                const int ncols = min(2 * kBlk, W - col0);
                const int col = lane & 7, rsub = lane >> 3;
                __syncwarp();
                if (col < ncols) {
                    uint32_t ta = tile + (rsub * kTilePitch + col) * ES;
                    const size_t o = (size_t)rsub * W + col0 + col;
                    ST* g0 = du_l + o;
                    ST* g1 = dl_l + o;
                    for (int r = rsub; r < Lp; r += 4) {
                        if (w_du) E::stg(g0, E::lds(ta));
                        if (w_dl) E::stg(g1, E::lds(ta + tplane));
                        ta += 4 * kTilePitch * ES; g0 += 4 * W; g1 += 4 * W;
                    }
                    if (w_dw)
                        for (int k = c; k < 3; k += NS) {
                            uint32_t tw = dwtile + ((k * Lp + rsub) * kTilePitch + col) * ES;
                            ST* g2 = dw_l + (size_t)k * HW + o;
                            for (int r = rsub; r < Lp; r += 4) {
                                E::stg(g2, E::lds(tw));
                                tw += 4 * kTilePitch * ES; g2 += 4 * W;
                            }
                        }
                }
                __syncwarp();
            }
        }
        release(bi, desc2, n == NB - 1);
    }
    if (p.dh0) {
        ST* d0 = reinterpret_cast<ST*>(p.dh0) + pc * Lmax;
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const int pos = P * lane + e;
            if (pos < Lmax) E::stg(d0 + pos, E::pack(ok[e] ? carry[e] : 0.f));
        }
    }
}

// ---------------------------------------------------------------------------------------------------
template <typename ST, int P>
__global__ void __launch_bounds__(32 * (kChNPW + kChMaxNS), 1)
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
        for (int s = 0; s < kChSlots; ++s) { mbar_init(&full[s], kChNPW * 33); mbar_init(&empty[s], NS); }
        mbar_init_fence();
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // zeros (generic proxy) before bulk copies
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
    } else if (warp < kChNPW + NS) {
        // ---------------- chain warp of channel c ------------------------------------------------------
        const int c = warp - kChNPW;
        uint32_t pf = 0;
        if (p.q[0] >= 0) chain_bwd_dir<ST, P, false, false>(p, smem, 0, b, g, c, lane, pf);
        if (p.q[1] >= 0) chain_bwd_dir<ST, P, false, true>(p, smem, 1, b, g, c, lane, pf);
        if (p.q[2] >= 0) chain_bwd_dir<ST, P, true, false>(p, smem, 2, b, g, c, lane, pf);
        if (p.q[3] >= 0) chain_bwd_dir<ST, P, true, true>(p, smem, 3, b, g, c, lane, pf);
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
static size_t chain_bwd_layout(const Shape& sh, int es, int P, int NSV, int NSH, bool want_dw, ChainBwdParams* prm) {
    const int NS = sh.cg(), np = 3 + 4 * NS;
    const bool vact = sh.mask & 3u, hact = sh.mask & 12u;
    const int CB = kBlk * es;
    const int Lmax = sh.Lmax();
    size_t off = 2 * kChSlots * sizeof(uint64_t);
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
    off += ringb;
    off = (off + 127) / 128 * 128;
    const int NBmax = (Lmax + kBlk - 1) / kBlk;
    prm->ckpt_warp = (uint32_t)((size_t)NBmax * P * 32 * 4);
    prm->off_ckpt = (uint32_t)off;
    off += (size_t)NS * prm->ckpt_warp;
    prm->off_exch = (uint32_t)off;
    if (want_dw) off += (size_t)NS * 3 * kBlk * P * 32 * 4;
    off = (off + 127) / 128 * 128;
    prm->tile_warp = (uint32_t)(((size_t)2 * sh.H * kTilePitch * es + 15) / 16 * 16);
    prm->off_tile = (uint32_t)off;
    if (hact) off += (size_t)NS * prm->tile_warp;
    prm->off_dwtile = (uint32_t)off;
    if (hact && want_dw) off += ((size_t)3 * sh.H * kTilePitch * es + 15) / 16 * 16;
    off = (off + 15) / 16 * 16;
    prm->total = (uint32_t)off;
    return off;
}

template <typename ST, int P>
static int launch_chain_bwd(const ChainBwdParams& prm, int items, int threads, cudaStream_t st) {
    auto kern = chain_bwd_kernel<ST, P>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prm.total);
    if (e != cudaSuccess) { set_error("chain bwd: cudaFuncSetAttribute(%u B): %s", prm.total, cudaGetErrorString(e)); return GSPN_ECUDA; }
    kern<<<items, threads, prm.total, st>>>(prm);
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
            if (NSH <= kChSlots && chain_bwd_layout(sh, ES, P, NSV, NSH, a.dw3 != nullptr, &prm) <= (size_t)kMaxSmemOptin) {
                prm.NSV = NSV; prm.NSH = NSH;
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
    const int threads = 32 * (kChNPW + NS), items = sh.B * sh.G;
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
