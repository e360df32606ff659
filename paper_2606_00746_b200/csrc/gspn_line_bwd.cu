// gspn_line_bwd.cu -- backward scan for 16-byte-aligned rows: ONE launch, all four
// directions, every gradient written once.  Derived from Eq. 1-2 (the paper gives timings only);
// the recurrences are DESIGN.md section 4.
//
// CTA = the NC = C/G channels of one (b, group) unit (the whole group, so that dw3 is summed inside the CTA).
// Warp c < NC: channel c; warp NC: the TMA producer and the issuer of the output stores.  The directions run one
// after another.  Per direction every channel warp makes two passes over its line:
//   pass 1  the forward recurrence (taps, lambda, x), leaving h at the start of every stage of kLineSteps steps
//           in shared memory (fp32 checkpoints);
//   pass 2  stage by stage in reverse order: h of the stage recomputed from its checkpoint into registers, then the
//           adjoint steps in reverse: gh = dy u + carry, du = dy h, dlambda = x gh, dx += lambda gh,
//           dw3 partial = gh h[s-1, p+k-1], carry = sum_k w_k gh (shifted), dh0 = the carry left after step 0.
// dx is summed over the directions in TENSOR MEMORY (fp32, one lane quarter per channel, the layouts of
// gspn_line_fwd.cu: column owners for T->B / B->T, row owners for L->R / R->L, turned in place in between).
// dw3 is summed over the group's channels in a fixed order without atomics: every warp leaves its fp32 partials of
// four steps in shared memory, the warps meet at a named barrier, and each then reduces a quarter of them.
// dlambda, du and dw3 leave through shared-memory stages and TMA stores (one RNE per element).
#include "gspn_line.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {
namespace {

constexpr int kBwdStages = 2;          // ring stages (operands) and output stages

struct LineBwdParams {
    int B, C, H, W, G;
    unsigned mask;
    int slab[4];          // slab index of each direction inside w3 / lambda / u and the per-direction outputs
    int pitch;            // floats per row of the transposition tile
    int multi;            // 1: one TMA box per operand / output (all its planes), else one per plane
    uint32_t pb;          // bytes between planes inside an operand or output stage
    uint32_t tm_cols;     // tensor-memory columns of the CTA
    uint32_t plane_cols;  // tensor-memory columns of one channel plane (channels c and c + 4 share a lane quarter)
    uint32_t ring_off, out_off, part_off, ckpt_off, bar_off;     // shared-memory layout (bytes)
    uint32_t part_stride; // floats per (channel) partial block: 4 steps x 3 taps x Lpad
    int Lpad;             // positions per line rounded up to 32 * P
    int nblk_max;
    const void* h0;
    void *dx, *dh0;
    int want_dlam, want_du, want_dw3;
};

// what a channel warp knows
struct BwdCtx {
    int H, W, lane, c, NCrt;
    unsigned char *ring, *out;
    float *part, *ckpt;
    uint64_t *full, *empty;
    uint32_t pb, stage_bytes, out_bytes;
    uint32_t tb;                  // tensor-memory address of this channel's plane, column 0
    int it;                       // operand stages consumed so far (all directions, both passes)
    int ob;                       // output stages written so far
    int grp;                      // four-step groups finished so far (parity of the partial buffer)
    int Lpad;
    uint32_t part_stride;
};

// stage planes: [taps 3][lambda NC][x NC][u NC][dy NC]; output planes: [dlambda NC][du NC][dw3 3]
template <int NC> struct BwdPlanes {
    static constexpr int LAM = 3, X = 3 + NC, U = 3 + 2 * NC, DY = 3 + 3 * NC, N1 = 3 + 2 * NC, N2 = 3 + 4 * NC;
    static constexpr int ODLAM = 0, ODU = NC, ODW = 2 * NC, NOUT = 2 * NC + 3;
};

// P storage elements -> packed words (one RNE per element) and a P*ES-byte store
template <typename ST, int P> __device__ __forceinline__ void bwd_store(ST* p, const float (&f)[P]) {
    if constexpr (sizeof(ST) == 4) {
        stf<P>(reinterpret_cast<float*>(p), f);
    } else if constexpr (P == 1) {
        *p = __float2bfloat16_rn(f[0]);
    } else {
        uint32_t r[P / 2];
        Store<__nv_bfloat16>::template pack<2 * P>(f, r);
        st_vec<2 * P>(p, r);
    }
}

// every warp zeroes the taps that leave the grid in the stage it is about to read (see gspn_line_fwd.cu)
template <typename ST>
__device__ __forceinline__ void bwd_zero_edge_taps_v(unsigned char* sb, uint32_t pb, int W, int lane) {
    if (lane < kLineSteps) {
        *(reinterpret_cast<ST*>(sb) + lane * W) = ST(0.f);
        *(reinterpret_cast<ST*>(sb + 2 * pb) + lane * W + W - 1) = ST(0.f);
    }
    __syncwarp();
}

// where the outputs of the current direction go
struct BwdOut {
    const CUtensorMap *mdlam, *mdu, *mdw;      // store maps of the current axis
    int pc, pw;                                // first plane of this CTA inside dlambda / du, inside dw3
    int want_dlam, want_du, want_dw3;
};

// warp 0, lane 0: the output stage `buf` (rows / columns from s0 on) leaves; vertical: 3-D maps, coordinate 1 = row
template <int NC, bool VERT>
__device__ __forceinline__ void bwd_issue_store(const BwdCtx& cx, const BwdOut& oo, int buf, int s0, int multi, int K) {
    using PL = BwdPlanes<NC>;
    const unsigned char* ob = cx.out + (size_t)buf * cx.out_bytes;
    const int nlam = multi ? 1 : NC, nw = multi ? 1 : 3;
    for (int i = 0; i < nlam; ++i) {
        if (oo.want_dlam) {
            if (VERT) tma_store_3d(oo.mdlam, ob + (size_t)(PL::ODLAM + i) * cx.pb, 0, s0, oo.pc + i);
            else tma_store_4d(oo.mdlam, ob + (size_t)(PL::ODLAM + i) * cx.pb, 0, 0, s0 / K, oo.pc + i);
        }
        if (oo.want_du) {
            if (VERT) tma_store_3d(oo.mdu, ob + (size_t)(PL::ODU + i) * cx.pb, 0, s0, oo.pc + i);
            else tma_store_4d(oo.mdu, ob + (size_t)(PL::ODU + i) * cx.pb, 0, 0, s0 / K, oo.pc + i);
        }
    }
    if (oo.want_dw3)
        for (int i = 0; i < nw; ++i) {
            if (VERT) tma_store_3d(oo.mdw, ob + (size_t)(PL::ODW + i) * cx.pb, 0, s0, oo.pw + i);
            else tma_store_4d(oo.mdw, ob + (size_t)(PL::ODW + i) * cx.pb, 0, 0, s0 / K, oo.pw + i);
        }
    bulk_commit();
}

__device__ __forceinline__ void bwd_release_stage(uint64_t* empty_bar, int lane) {
    fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(empty_bar);
}

// ---- T->B (rev = false) / B->T (rev = true): lane a owns the P adjacent columns P*a + k -----------------------------
template <typename ST, int NC, int P>
__device__ __forceinline__ void bwd_dir_v(BwdCtx& cx, const bool rev, const bool acc, const ST* h0p, ST* dh0p,
                                          const BwdOut& oo, int multi) {
    using PL = BwdPlanes<NC>;
    constexpr int S = kLineSteps, NS = kBwdStages, ES = sizeof(ST);
    const int H = cx.H, W = cx.W, lane = cx.lane, c = cx.c;
    const int WP = W / P;
    const bool active = lane < WP, first_lane = lane == 0, last_lane = lane == WP - 1;
    const int lp = active ? lane : 0;
    const uint32_t pbe = cx.pb / ES;
    const int nblk = (H + S - 1) / S;
    float* const ck = cx.ckpt + (size_t)c * ((H + S - 1) / S) * cx.Lpad + P * lane;

    float h[P];
#pragma unroll
    for (int k = 0; k < P; ++k) h[k] = (h0p && active) ? ld_f(h0p + P * lane + k) : 0.f;

    // ---- pass 1: the forward recurrence, h at the start of every stage kept
    for (int blk = 0; blk < nblk; ++blk, ++cx.it) {
        const int stg = cx.it % NS;
        mbar_wait(&cx.full[stg], (cx.it / NS) & 1);
        unsigned char* sb = cx.ring + (size_t)stg * cx.stage_bytes;
        bwd_zero_edge_taps_v<ST>(sb, cx.pb, W, lane);
        stf<P>(ck + (size_t)blk * cx.Lpad, h);
        const int nr = min(S, H - blk * S);
        const ST* base = reinterpret_cast<const ST*>(sb) + P * lp;
        for (int r = 0; r < nr; ++r) {
            const ST* row = base + (rev ? S - 1 - r : r) * W;
            float w0[P], w1[P], w2[P];
            LineRaw<ST, P> la, xx;
            line_ld<ST, P>(row, w0);
            line_ld<ST, P>(row + pbe, w1);
            line_ld<ST, P>(row + 2 * pbe, w2);
            line_ld_raw<ST, P>(row + (PL::LAM + c) * pbe, la);
            line_ld_raw<ST, P>(row + (PL::X + c) * pbe, xx);
            const float hl = __shfl_up_sync(0xffffffffu, h[P - 1], 1);
            const float hr = __shfl_down_sync(0xffffffffu, h[0], 1);
            float hn[P];
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const float l = k == 0 ? hl : h[k - 1];
                const float rr = k == P - 1 ? hr : h[k + 1];
                hn[k] = fmaf(w0[k], l, fmaf(w2[k], rr, line_fma_raw<ST>(la.w, xx.w, k, w1[k] * h[k])));
            }
#pragma unroll
            for (int k = 0; k < P; ++k) h[k] = hn[k];
        }
        bwd_release_stage(&cx.empty[stg], lane);
    }

    // ---- pass 2: stages in reverse order
    float carry[P];
#pragma unroll
    for (int k = 0; k < P; ++k) carry[k] = 0.f;
    int pend_buf = -1, pend_s0 = 0;                     // the output stage whose stores wait for its last reduction
    for (int blk = nblk - 1; blk >= 0; --blk, ++cx.it) {
        const int stg = cx.it % NS;
        mbar_wait(&cx.full[stg], (cx.it / NS) & 1);
        unsigned char* sb = cx.ring + (size_t)stg * cx.stage_bytes;
        bwd_zero_edge_taps_v<ST>(sb, cx.pb, W, lane);
        const int nr = min(S, H - blk * S);
        const ST* base = reinterpret_cast<const ST*>(sb) + P * lp;
        // h of the stage, recomputed from its checkpoint: hb[r] = h before step r, hb[r + 1] = h after it
        float hb[S + 1][P], hl[S], hr[S];
        ldf<P>(ck + (size_t)blk * cx.Lpad, hb[0]);
#pragma unroll
        for (int r = 0; r < S; ++r) {
            if (r < nr) {
                const ST* row = base + (rev ? S - 1 - r : r) * W;
                float w0[P], w1[P], w2[P];
                LineRaw<ST, P> la, xx;
                line_ld<ST, P>(row, w0);
                line_ld<ST, P>(row + pbe, w1);
                line_ld<ST, P>(row + 2 * pbe, w2);
                line_ld_raw<ST, P>(row + (PL::LAM + c) * pbe, la);
                line_ld_raw<ST, P>(row + (PL::X + c) * pbe, xx);
                hl[r] = __shfl_up_sync(0xffffffffu, hb[r][P - 1], 1);
                hr[r] = __shfl_down_sync(0xffffffffu, hb[r][0], 1);
                if (first_lane) hl[r] = 0.f;                      // outside the grid: h = 0 (dw3 reads these)
                if (last_lane) hr[r] = 0.f;
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const float l = k == 0 ? hl[r] : hb[r][k - 1];
                    const float rr = k == P - 1 ? hr[r] : hb[r][k + 1];
                    hb[r + 1][k] = fmaf(w0[k], l, fmaf(w2[k], rr, line_fma_raw<ST>(la.w, xx.w, k, w1[k] * hb[r][k])));
                }
            }
        }
        const int buf = cx.ob & 1;
        unsigned char* ob = cx.out + (size_t)buf * cx.out_bytes;
        const int s0 = rev ? H - (blk + 1) * S : blk * S;      // first image row of the stage
        bool first_bar = true;
#pragma unroll
        for (int g = S / 4 - 1; g >= 0; --g) {
            if (4 * g < nr) {
                float* pbuf = cx.part + ((size_t)(cx.grp & 1) * NC + c) * cx.part_stride + P * lane;
#pragma unroll
                for (int t = 3; t >= 0; --t) {
                    const int r = 4 * g + t;
                    if (r < nr) {
                        const int rs = rev ? S - 1 - r : r;                  // row inside the stage
                        const int i = rev ? H - 1 - (blk * S + r) : blk * S + r;
                        const ST* row = base + rs * W;
                        float w0[P], w1[P], w2[P], lf[P], xf[P], dyf[P];
                        LineRaw<ST, P> uu, dy;
                        line_ld<ST, P>(row, w0);
                        line_ld<ST, P>(row + pbe, w1);
                        line_ld<ST, P>(row + 2 * pbe, w2);
                        line_ld<ST, P>(row + (PL::LAM + c) * pbe, lf);
                        line_ld<ST, P>(row + (PL::X + c) * pbe, xf);
                        line_ld_raw<ST, P>(row + (PL::U + c) * pbe, uu);
                        line_ld_raw<ST, P>(row + (PL::DY + c) * pbe, dy);
                        line_ld<ST, P>(row + (PL::DY + c) * pbe, dyf);
                        float dxv[P];
                        if (acc) tm_ld<P>(cx.tb + i * P, dxv);
                        float gh[P], dl[P], du[P], p0[P], p1[P], p2[P], t0[P], t1[P], t2[P];
#pragma unroll
                        for (int k = 0; k < P; ++k) {
                            gh[k] = line_fma_raw<ST>(dy.w, uu.w, k, carry[k]);
                            du[k] = dyf[k] * hb[r + 1][k];
                            dl[k] = xf[k] * gh[k];
                            p0[k] = gh[k] * (k == 0 ? hl[r] : hb[r][k - 1]);
                            p1[k] = gh[k] * hb[r][k];
                            p2[k] = gh[k] * (k == P - 1 ? hr[r] : hb[r][k + 1]);
                            t0[k] = w0[k] * gh[k];
                            t1[k] = w1[k] * gh[k];
                            t2[k] = w2[k] * gh[k];
                        }
                        float tl = __shfl_up_sync(0xffffffffu, t2[P - 1], 1);
                        float tr = __shfl_down_sync(0xffffffffu, t0[0], 1);
                        if (first_lane) tl = 0.f;
                        if (last_lane) tr = 0.f;
#pragma unroll
                        for (int k = 0; k < P; ++k)
                            carry[k] = (k == 0 ? tl : t2[k - 1]) + t1[k] + (k == P - 1 ? tr : t0[k + 1]);
                        if (acc) {
                            tm_wait_ld<P>(dxv);
#pragma unroll
                            for (int k = 0; k < P; ++k) dxv[k] = fmaf(lf[k], gh[k], dxv[k]);
                        } else {
#pragma unroll
                            for (int k = 0; k < P; ++k) dxv[k] = lf[k] * gh[k];
                        }
                        tm_st<P>(cx.tb + i * P, dxv);
                        stf<P>(pbuf + (size_t)(t * 3 + 0) * cx.Lpad, p0);
                        stf<P>(pbuf + (size_t)(t * 3 + 1) * cx.Lpad, p1);
                        stf<P>(pbuf + (size_t)(t * 3 + 2) * cx.Lpad, p2);
                        if (active) {
                            bwd_store<ST, P>(reinterpret_cast<ST*>(ob + (size_t)(PL::ODLAM + c) * cx.pb) + rs * W + P * lane, dl);
                            bwd_store<ST, P>(reinterpret_cast<ST*>(ob + (size_t)(PL::ODU + c) * cx.pb) + rs * W + P * lane, du);
                        }
                    }
                }
                // the warps of the unit meet: the partials of these four steps are complete
                if (c == 0 && lane == 0 && g == 0) bulk_wait_read<0>();      // the stage before last has left
                fence_proxy_async();
                named_bar_sync(1, NC * 32);
                if (first_bar && c == 0 && lane == 0 && pend_buf >= 0) bwd_issue_store<NC, true>(cx, oo, pend_buf, pend_s0, multi, 1);
                first_bar = false;
                // dw3 of these steps: fixed channel order, no atomics; warp w takes step 4g + w (+ NC, ...)
                for (int t = c; t < 4; t += NC) {
                    const int r = 4 * g + t;
                    if (r < nr && active) {
                        const int rs = rev ? S - 1 - r : r;
                        const float* pp = cx.part + (size_t)(cx.grp & 1) * NC * cx.part_stride + P * lane;
#pragma unroll
                        for (int tap = 0; tap < 3; ++tap) {
                            float sum[P];
                            ldf<P>(pp + (size_t)(t * 3 + tap) * cx.Lpad, sum);
                            for (int cc = 1; cc < NC; ++cc) {
                                float v[P];
                                ldf<P>(pp + (size_t)cc * cx.part_stride + (size_t)(t * 3 + tap) * cx.Lpad, v);
#pragma unroll
                                for (int k = 0; k < P; ++k) sum[k] += v[k];
                            }
                            bwd_store<ST, P>(reinterpret_cast<ST*>(ob + (size_t)(PL::ODW + tap) * cx.pb) + rs * W + P * lane, sum);
                        }
                    }
                }
                ++cx.grp;
            }
        }
        pend_buf = buf; pend_s0 = s0;
        ++cx.ob;
        bwd_release_stage(&cx.empty[stg], lane);
    }
    // the last stage of this direction leaves
    if (c == 0 && lane == 0) bulk_wait_read<0>();
    fence_proxy_async();
    named_bar_sync(1, NC * 32);
    if (c == 0 && lane == 0 && pend_buf >= 0) bwd_issue_store<NC, true>(cx, oo, pend_buf, pend_s0, multi, 1);
    if (dh0p) {
        if (active) {
#pragma unroll
            for (int k = 0; k < P; ++k) st_f(dh0p + P * lane + k, carry[k]);
        }
        for (int p = W + lane; p < (H > W ? H : W); p += 32) st_f(dh0p + p, 0.f);     // entries past the line are zeros
    }
}

// ---- L->R (rev = false) / R->L (rev = true): lane b owns the rows b + 32k; a stage is kLineSteps columns held as
// 16-byte column pieces [chunk][row][16 B]; operands are read four steps (one sub-piece) at a time ---------------------
template <typename ST> struct Sub {                     // four consecutive columns of one row: ES raw words
    static constexpr int NW = sizeof(ST);
    uint32_t w[NW];
};
template <typename ST> __device__ __forceinline__ void sub_ld(const unsigned char* p, Sub<ST>& s) { lds_vec<4 * sizeof(ST)>(p, s.w); }
template <typename ST> __device__ __forceinline__ float sub_elem(const Sub<ST>& s, int t) {
    if constexpr (sizeof(ST) == 4) return __uint_as_float(s.w[t]);
    else return (t & 1) ? __uint_as_float(s.w[t >> 1] & 0xffff0000u) : __uint_as_float(s.w[t >> 1] << 16);
}
// byte offset of the four-column sub-piece `q` (0, 1: columns 0-3, 4-7 of the stage) of row `row` inside a stage plane
template <typename ST> __device__ __forceinline__ uint32_t sub_off(int row, int q, int H) {
    if constexpr (sizeof(ST) == 4) return (uint32_t)((q * H + row) * 16);      // fp32: a piece is four columns
    else return (uint32_t)(row * 16 + q * 8);                                    // bf16: a piece is eight columns
}

// neighbours of every slot in the row-owner layout: up[k] = v at row - 1, dn[k] = v at row + 1, 0 outside the grid
template <int P>
__device__ __forceinline__ void nbr_rows(const float (&v)[P], float (&up)[P], float (&dn)[P], int lane, int H) {
    const int src_up = (lane + 31) & 31, src_dn = (lane + 1) & 31;
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const float su = (k > 0 && lane == 31) ? v[k > 0 ? k - 1 : 0] : v[k];         // lane 31 only serves lane 0
        const float sd = (k < P - 1 && lane == 0) ? v[k < P - 1 ? k + 1 : k] : v[k];  // lane 0 only serves lane 31
        up[k] = __shfl_sync(0xffffffffu, su, src_up);
        dn[k] = __shfl_sync(0xffffffffu, sd, src_dn);
        if (k == 0 && lane == 0) up[k] = 0.f;
        if (lane + 32 * k >= H - 1) dn[k] = 0.f;
    }
}

template <int P> __device__ __forceinline__ void nbr_up(const float (&v)[P], float (&up)[P], int lane) {
    const int src_up = (lane + 31) & 31;
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const float su = (k > 0 && lane == 31) ? v[k > 0 ? k - 1 : 0] : v[k];
        up[k] = __shfl_sync(0xffffffffu, su, src_up);
        if (k == 0 && lane == 0) up[k] = 0.f;
    }
}
template <int P> __device__ __forceinline__ void nbr_dn(const float (&v)[P], float (&dn)[P], int lane, int H) {
    const int src_dn = (lane + 1) & 31;
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const float sd = (k < P - 1 && lane == 0) ? v[k < P - 1 ? k + 1 : k] : v[k];
        dn[k] = __shfl_sync(0xffffffffu, sd, src_dn);
        if (lane + 32 * k >= H - 1) dn[k] = 0.f;
    }
}

template <typename ST>
__device__ __forceinline__ void bwd_zero_edge_taps_h(unsigned char* sb, uint32_t pb, int H, int lane) {
    constexpr int NCH = kLineSteps * sizeof(ST) / 16;
    if (lane < NCH) {
        *reinterpret_cast<uint4*>(sb + ((size_t)lane * H) * 16) = make_uint4(0, 0, 0, 0);                   // tap 0, row 0
        *reinterpret_cast<uint4*>(sb + 2 * pb + ((size_t)lane * H + H - 1) * 16) = make_uint4(0, 0, 0, 0);  // tap 2, row H-1
    }
    __syncwarp();
}

template <typename ST, int NC, int P, bool REV>
__device__ __forceinline__ void bwd_dir_h(BwdCtx& cx, const bool acc, const ST* h0p, ST* dh0p,
                                          const BwdOut& oo, int multi) {
    constexpr bool rev = REV;          // compile-time: the element order inside a sub-piece indexes registers
    using PL = BwdPlanes<NC>;
    constexpr int S = kLineSteps, NS = kBwdStages, ES = sizeof(ST), K = 16 / ES;
    const int H = cx.H, W = cx.W, lane = cx.lane, c = cx.c;
    const uint32_t pb = cx.pb;
    const int nblk = (W + S - 1) / S;
    float* const ck = cx.ckpt + (size_t)c * nblk * cx.Lpad + lane;          // [blk][k * 32 + lane]
    int rowc[P];                                                             // this lane's rows, clamped for addressing
#pragma unroll
    for (int k = 0; k < P; ++k) rowc[k] = lane + 32 * k < H ? lane + 32 * k : 0;

    float h[P];
#pragma unroll
    for (int k = 0; k < P; ++k) h[k] = (h0p && lane + 32 * k < H) ? ld_f(h0p + lane + 32 * k) : 0.f;

    // ---- pass 1
    for (int blk = 0; blk < nblk; ++blk, ++cx.it) {
        const int stg = cx.it % NS;
        mbar_wait(&cx.full[stg], (cx.it / NS) & 1);
        unsigned char* sb = cx.ring + (size_t)stg * cx.stage_bytes;
        bwd_zero_edge_taps_h<ST>(sb, pb, H, lane);
#pragma unroll
        for (int k = 0; k < P; ++k) ck[(size_t)blk * cx.Lpad + 32 * k] = h[k];
        const int nr = min(S, W - blk * S);
#pragma unroll
        for (int qq = 0; qq < 2; ++qq) {
            if (4 * qq < nr) {
                const int q = rev ? 1 - qq : qq;                    // sub-piece in memory order
                Sub<ST> s0[P], s1[P], s2[P], sl[P], sx[P];
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const unsigned char* p = sb + sub_off<ST>(rowc[k], q, H);
                    sub_ld<ST>(p, s0[k]);
                    sub_ld<ST>(p + pb, s1[k]);
                    sub_ld<ST>(p + 2 * pb, s2[k]);
                    sub_ld<ST>(p + (size_t)(PL::LAM + c) * pb, sl[k]);
                    sub_ld<ST>(p + (size_t)(PL::X + c) * pb, sx[k]);
                }
#pragma unroll
                for (int tt = 0; tt < 4; ++tt) {
                    if (4 * qq + tt < nr) {
                        const int e = rev ? 3 - tt : tt;
                        float up[P], dn[P];
                        nbr_rows<P>(h, up, dn, lane, H);
#pragma unroll
                        for (int k = 0; k < P; ++k)
                            h[k] = fmaf(sub_elem<ST>(s0[k], e), up[k],
                                        fmaf(sub_elem<ST>(s2[k], e), dn[k],
                                             fmaf(sub_elem<ST>(sl[k], e), sub_elem<ST>(sx[k], e), sub_elem<ST>(s1[k], e) * h[k])));
                    }
                }
            }
        }
        bwd_release_stage(&cx.empty[stg], lane);
    }

    // ---- pass 2
    float carry[P];
#pragma unroll
    for (int k = 0; k < P; ++k) carry[k] = 0.f;
    int pend_buf = -1, pend_s0 = 0;
    for (int blk = nblk - 1; blk >= 0; --blk, ++cx.it) {
        const int stg = cx.it % NS;
        mbar_wait(&cx.full[stg], (cx.it / NS) & 1);
        unsigned char* sb = cx.ring + (size_t)stg * cx.stage_bytes;
        bwd_zero_edge_taps_h<ST>(sb, pb, H, lane);
        const int nr = min(S, W - blk * S);
        float hb[S + 1][P];
#pragma unroll
        for (int k = 0; k < P; ++k) hb[0][k] = ck[(size_t)blk * cx.Lpad + 32 * k];
#pragma unroll
        for (int qq = 0; qq < 2; ++qq) {
            if (4 * qq < nr) {
                const int q = rev ? 1 - qq : qq;
                Sub<ST> s0[P], s1[P], s2[P], sl[P], sx[P];
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const unsigned char* p = sb + sub_off<ST>(rowc[k], q, H);
                    sub_ld<ST>(p, s0[k]);
                    sub_ld<ST>(p + pb, s1[k]);
                    sub_ld<ST>(p + 2 * pb, s2[k]);
                    sub_ld<ST>(p + (size_t)(PL::LAM + c) * pb, sl[k]);
                    sub_ld<ST>(p + (size_t)(PL::X + c) * pb, sx[k]);
                }
#pragma unroll
                for (int tt = 0; tt < 4; ++tt) {
                    const int r = 4 * qq + tt;
                    if (r < nr) {
                        const int e = rev ? 3 - tt : tt;
                        float up[P], dn[P];
                        nbr_rows<P>(hb[r], up, dn, lane, H);
#pragma unroll
                        for (int k = 0; k < P; ++k)
                            hb[r + 1][k] = fmaf(sub_elem<ST>(s0[k], e), up[k],
                                                fmaf(sub_elem<ST>(s2[k], e), dn[k],
                                                     fmaf(sub_elem<ST>(sl[k], e), sub_elem<ST>(sx[k], e),
                                                          sub_elem<ST>(s1[k], e) * hb[r][k])));
                    }
                }
            }
        }
        const int buf = cx.ob & 1;
        unsigned char* ob = cx.out + (size_t)buf * cx.out_bytes;
        const int s0c = rev ? W - (blk + 1) * S : blk * S;       // first image column of the stage
        bool first_bar = true;
#pragma unroll
        for (int g = 1; g >= 0; --g) {
            if (4 * g < nr) {
                const int q = rev ? 1 - g : g;
                float* pbuf = cx.part + ((size_t)(cx.grp & 1) * NC + c) * cx.part_stride + lane;
                Sub<ST> s0[P], s1[P], s2[P], sl[P], sx[P], su[P], sy[P];
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const unsigned char* p = sb + sub_off<ST>(rowc[k], q, H);
                    sub_ld<ST>(p, s0[k]);
                    sub_ld<ST>(p + pb, s1[k]);
                    sub_ld<ST>(p + 2 * pb, s2[k]);
                    sub_ld<ST>(p + (size_t)(PL::LAM + c) * pb, sl[k]);
                    sub_ld<ST>(p + (size_t)(PL::X + c) * pb, sx[k]);
                    sub_ld<ST>(p + (size_t)(PL::U + c) * pb, su[k]);
                    sub_ld<ST>(p + (size_t)(PL::DY + c) * pb, sy[k]);
                }
                const int j0 = s0c + 4 * q;                        // lowest image column of this group
                float dxv[P][4], dlv[P][4], duv[P][4];
                if (acc) {
#pragma unroll
                    for (int k = 0; k < P; ++k) {
                        if (32 * k < H) tm_ld<4>(cx.tb + k * 32 * P + j0, dxv[k]);  // slots past the plane own no columns
                        else dxv[k][0] = dxv[k][1] = dxv[k][2] = dxv[k][3] = 0.f;
                    }
#pragma unroll
                    for (int k = 0; k < P; ++k) if (32 * k < H) tm_wait_ld<4>(dxv[k]);
                }
#pragma unroll
                for (int t = 3; t >= 0; --t) {
                    const int r = 4 * g + t;
                    if (r < nr) {
                        const int e = rev ? 3 - t : t;              // column inside the group (memory order)
                        float gh[P], t0[P], t1[P], t2[P], hu[P], hd[P];
                        nbr_rows<P>(hb[r], hu, hd, lane, H);
#pragma unroll
                        for (int k = 0; k < P; ++k) {
                            const float dyf = sub_elem<ST>(sy[k], e);
                            gh[k] = fmaf(dyf, sub_elem<ST>(su[k], e), carry[k]);
                            duv[k][e] = dyf * hb[r + 1][k];
                            dlv[k][e] = sub_elem<ST>(sx[k], e) * gh[k];
                            const float lg = sub_elem<ST>(sl[k], e) * gh[k];
                            dxv[k][e] = acc ? dxv[k][e] + lg : lg;
                            pbuf[(size_t)(t * 3 + 0) * cx.Lpad + 32 * k] = gh[k] * hu[k];
                            pbuf[(size_t)(t * 3 + 1) * cx.Lpad + 32 * k] = gh[k] * hb[r][k];
                            pbuf[(size_t)(t * 3 + 2) * cx.Lpad + 32 * k] = gh[k] * hd[k];
                            t0[k] = sub_elem<ST>(s0[k], e) * gh[k];
                            t1[k] = sub_elem<ST>(s1[k], e) * gh[k];
                            t2[k] = sub_elem<ST>(s2[k], e) * gh[k];
                        }
                        float a2[P], a0[P];
                        nbr_up<P>(t2, a2, lane);                      // t2 at row - 1
                        nbr_dn<P>(t0, a0, lane, H);                   // t0 at row + 1
#pragma unroll
                        for (int k = 0; k < P; ++k) carry[k] = a2[k] + t1[k] + a0[k];
                    } else {
                        const int e = rev ? 3 - t : t;
#pragma unroll
                        for (int k = 0; k < P; ++k) { duv[k][e] = 0.f; dlv[k][e] = 0.f; if (!acc) dxv[k][e] = 0.f; }
                    }
                }
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    if (32 * k < H) tm_st<4>(cx.tb + k * 32 * P + j0, dxv[k]);
                    if (lane + 32 * k < H) {
                        const uint32_t off = sub_off<ST>(lane + 32 * k, q, H);
                        bwd_store<ST, 4>(reinterpret_cast<ST*>(ob + (size_t)(PL::ODLAM + c) * pb + off), dlv[k]);
                        bwd_store<ST, 4>(reinterpret_cast<ST*>(ob + (size_t)(PL::ODU + c) * pb + off), duv[k]);
                    }
                }
                if (c == 0 && lane == 0 && g == 0) bulk_wait_read<0>();
                fence_proxy_async();
                named_bar_sync(1, NC * 32);
                if (first_bar && c == 0 && lane == 0 && pend_buf >= 0) bwd_issue_store<NC, false>(cx, oo, pend_buf, pend_s0, multi, K);
                first_bar = false;
                // dw3 of this group: warp w takes the row slots w, w + NC, ...; four steps = four adjacent columns
                for (int k = c; k < P; k += NC) {
                    if (lane + 32 * k < H) {
                        const float* pp = cx.part + (size_t)(cx.grp & 1) * NC * cx.part_stride + 32 * k + lane;
                        const uint32_t off = sub_off<ST>(lane + 32 * k, q, H);
#pragma unroll
                        for (int tap = 0; tap < 3; ++tap) {
                            float sum[4];
#pragma unroll
                            for (int t = 0; t < 4; ++t) {
                                const int e = rev ? 3 - t : t;
                                float a = 0.f;
                                if (4 * g + t < nr) {
                                    a = pp[(size_t)(t * 3 + tap) * cx.Lpad];
                                    for (int cc = 1; cc < NC; ++cc) a += pp[(size_t)cc * cx.part_stride + (size_t)(t * 3 + tap) * cx.Lpad];
                                }
                                sum[e] = a;
                            }
                            bwd_store<ST, 4>(reinterpret_cast<ST*>(ob + (size_t)(PL::ODW + tap) * pb + off), sum);
                        }
                    }
                }
                ++cx.grp;
            }
        }
        pend_buf = buf; pend_s0 = s0c;
        ++cx.ob;
        bwd_release_stage(&cx.empty[stg], lane);
    }
    if (c == 0 && lane == 0) bulk_wait_read<0>();
    fence_proxy_async();
    named_bar_sync(1, NC * 32);
    if (c == 0 && lane == 0 && pend_buf >= 0) bwd_issue_store<NC, false>(cx, oo, pend_buf, pend_s0, multi, K);
    if (dh0p) {
#pragma unroll
        for (int k = 0; k < P; ++k) if (lane + 32 * k < H) st_f(dh0p + lane + 32 * k, carry[k]);
        for (int p = H + lane; p < (H > W ? H : W); p += 32) st_f(dh0p + p, 0.f);     // entries past the line are zeros
    }
}

struct BwdMaps {
    CUtensorMap lx, lw, ll, lu, ldy;       // loads: x, w3, lambda, u, dy
    CUtensorMap sl, su, sw;                // stores: dlambda, du, dw3
};

template <typename ST, int NC, int P>
__global__ void __launch_bounds__((NC + 1) * 32, 1)
line_bwd_kernel(const __grid_constant__ BwdMaps mv, const __grid_constant__ BwdMaps mh, const LineBwdParams prm) {
    using PL = BwdPlanes<NC>;
    constexpr int ES = sizeof(ST), K = 16 / ES, S = kLineSteps, NS = kBwdStages;

    extern __shared__ __align__(128) unsigned char smem[];
    const int H = prm.H, W = prm.W;
    const uint32_t stage_bytes = PL::N2 * prm.pb, out_bytes = PL::NOUT * prm.pb;
    unsigned char* const ring = smem + prm.ring_off;
    uint64_t* const bars = reinterpret_cast<uint64_t*>(smem + prm.bar_off);
    uint64_t* const full = bars;               // [NS]
    uint64_t* const empty = bars + NS;         // [NS]
    uint32_t* const tm_slot = reinterpret_cast<uint32_t*>(bars + 2 * NS);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = blockIdx.x % prm.G, b = blockIdx.x / prm.G;
    const int c0 = g * NC;
    const unsigned mask = prm.mask;
    const int Lmax = H > W ? H : W;

    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NC); }
        mbar_init_fence();
    }
    if (warp == NC) tm_alloc(tm_slot, prm.tm_cols);
    tm_fence_before();
    __syncthreads();
    tm_fence_after();
    const uint32_t tm_base = *tm_slot;

    if (warp == NC) {
        // ------------------------------------------------------------------ producer: the stages in consumption order
        int it = 0;
        for (int dir = 0; dir < 4; ++dir) {
            if (!(mask >> dir & 1u)) continue;
            const bool vert = dir < 2, rev = dir & 1;
            const int q = prm.slab[dir];
            const BwdMaps& mm = vert ? mv : mh;
            const int pw = ((q * prm.B + b) * prm.G + g) * 3, pc = (q * prm.B + b) * prm.C + c0, px = b * prm.C + c0;
            // box number n of a stage: operand map, first plane in its tensor, plane slot in the stage, pass-1 member?
            // (multi: 5 boxes, one per operand; else one per plane: up to 3 + 4 NC = 35, more than a warp has lanes)
            const int nbox = prm.multi ? 5 : PL::N2;
            auto box = [&](int n, const CUtensorMap*& map, int& plane, int& slot, bool& in1) {
                if (prm.multi) {
                    if (n == 0) { map = &mm.lw; plane = pw; slot = 0; in1 = true; }
                    else if (n == 1) { map = &mm.ll; plane = pc; slot = PL::LAM; in1 = true; }
                    else if (n == 2) { map = &mm.lx; plane = px; slot = PL::X; in1 = true; }
                    else if (n == 3) { map = &mm.lu; plane = pc; slot = PL::U; in1 = false; }
                    else { map = &mm.ldy; plane = px; slot = PL::DY; in1 = false; }
                } else {
                    slot = n;
                    in1 = n < PL::N1;
                    if (n < 3) { map = &mm.lw; plane = pw + n; }
                    else if (n < PL::X) { map = &mm.ll; plane = pc + n - PL::LAM; }
                    else if (n < PL::U) { map = &mm.lx; plane = px + n - PL::X; }
                    else if (n < PL::DY) { map = &mm.lu; plane = pc + n - PL::U; }
                    else { map = &mm.ldy; plane = px + n - PL::DY; }
                }
            };
            const int Ls = vert ? H : W, Lc = vert ? W : H;
            const int nblk = (Ls + S - 1) / S;
            const uint32_t plane_tx = (uint32_t)(S * ES) * (uint32_t)Lc;       // bytes one plane brings per stage
            for (int pass = 0; pass < 2; ++pass)
                for (int n = 0; n < nblk; ++n, ++it) {
                    const int blk = pass ? nblk - 1 - n : n;
                    const int stg = it % NS;
                    if (it >= NS) mbar_wait(&empty[stg], ((it / NS) - 1) & 1);
                    if (lane == 0) mbar_arrive_expect_tx(&full[stg], plane_tx * (pass ? PL::N2 : PL::N1));
                    __syncwarp();
                    const int s0 = rev ? Ls - (blk + 1) * S : blk * S;
                    for (int bx = lane; bx < nbox; bx += 32) {
                        const CUtensorMap* map = nullptr;
                        int plane = 0, slot = 0;
                        bool in1 = false;
                        box(bx, map, plane, slot, in1);
                        if (pass || in1) {
                            unsigned char* dst = ring + (size_t)stg * stage_bytes + (size_t)slot * prm.pb;
                            if (vert) tma_load_3d(dst, map, 0, s0, plane, &full[stg]);
                            else tma_load_4d(dst, map, 0, 0, s0 / K, plane, &full[stg]);
                        }
                    }
                }
        }
    } else {
        // ------------------------------------------------------------------ channel c
        BwdCtx cx;
        cx.H = H; cx.W = W; cx.lane = lane; cx.c = warp; cx.NCrt = NC;
        cx.ring = ring; cx.out = smem + prm.out_off;
        cx.part = reinterpret_cast<float*>(smem + prm.part_off);
        cx.ckpt = reinterpret_cast<float*>(smem + prm.ckpt_off);
        cx.full = full; cx.empty = empty;
        cx.pb = prm.pb; cx.stage_bytes = stage_bytes; cx.out_bytes = out_bytes;
        cx.tb = tm_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(warp >> 2) * prm.plane_cols;
        cx.it = 0; cx.ob = 0; cx.grp = 0; cx.Lpad = prm.Lpad; cx.part_stride = prm.part_stride;
        const int c = warp, ch = c0 + c;
        const bool any_v = (mask & 3u) != 0, any_h = (mask & 12u) != 0;
        bool acc = false;
        for (int dir = 0; dir < 4; ++dir) {
            if (dir == 2 && any_v && any_h) {
                // the dx plane turns into the row-owner layout: the tiles alias the partial buffers, a few warps at a time
                const int tile_floats = 32 * prm.pitch;
                const int ntile = max(1, (int)((2u * NC * prm.part_stride) / (uint32_t)tile_floats));
                tm_wait_st();
                for (int rnd = 0; rnd * ntile < NC; ++rnd) {
                    if (c / ntile == rnd) line_transpose<P>(cx.tb, cx.part + (size_t)(c % ntile) * tile_floats, prm.pitch, H, W, lane);
                    named_bar_sync(1, NC * 32);
                }
            }
            if (dir == 2 && !any_v) acc = false;
            if (!(mask >> dir & 1u)) continue;
            const int q = prm.slab[dir];
            const size_t line = ((size_t)(q * prm.B + b) * prm.C + ch) * Lmax;
            const ST* h0p = prm.h0 ? reinterpret_cast<const ST*>(prm.h0) + line : nullptr;
            ST* dh0p = prm.dh0 ? reinterpret_cast<ST*>(prm.dh0) + line : nullptr;
            BwdOut oo;
            const BwdMaps& mm = dir < 2 ? mv : mh;
            oo.mdlam = &mm.sl; oo.mdu = &mm.su; oo.mdw = &mm.sw;
            oo.pc = (q * prm.B + b) * prm.C + c0; oo.pw = ((q * prm.B + b) * prm.G + g) * 3;
            oo.want_dlam = prm.want_dlam; oo.want_du = prm.want_du; oo.want_dw3 = prm.want_dw3;
            if (dir < 2) bwd_dir_v<ST, NC, P>(cx, dir & 1, acc, h0p, dh0p, oo, prm.multi);
            else if (dir & 1) bwd_dir_h<ST, NC, P, true>(cx, acc, h0p, dh0p, oo, prm.multi);
            else bwd_dir_h<ST, NC, P, false>(cx, acc, h0p, dh0p, oo, prm.multi);
            acc = true;
        }
        // ---- dx leaves: one RNE per element
        tm_wait_st();
        if (prm.dx) {
            ST* xg = reinterpret_cast<ST*>(prm.dx) + ((size_t)b * prm.C + ch) * H * W;
            if (any_h) {
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const int i = lane + 32 * k;
                    if (32 * k >= H) continue;
                    for (int jc = 0; jc * K < W; ++jc) {
                        float f[K];
                        tm_ld<K>(cx.tb + k * 32 * P + jc * K, f);
                        tm_wait_ld<K>(f);
                        uint32_t r[4];
                        Store<ST>::template pack<16>(f, r);
                        if (i < H) *reinterpret_cast<uint4*>(xg + (size_t)i * W + jc * K) = make_uint4(r[0], r[1], r[2], r[3]);
                    }
                }
            } else {
                for (int i = 0; i < H; ++i) {
                    float f[P];
                    tm_ld<P>(cx.tb + i * P, f);
                    tm_wait_ld<P>(f);
                    if (lane < W / P) bwd_store<ST, P>(xg + (size_t)i * W + P * lane, f);
                }
            }
        }
        if (c == 0 && lane == 0) bulk_wait_all<0>();       // the output stages are read before shared memory goes away
    }
    tm_fence_before();
    __syncthreads();
    if (warp == NC) tm_dealloc(tm_base, prm.tm_cols);
}

}  // namespace

// ---- host side ---------------------------------------------------------------------------------------------------
template <typename ST, int NC, int P>
static int line_bwd_run(const BwdArgs<ST>& a, cudaStream_t st) {
    using PL = BwdPlanes<NC>;
    constexpr int ES = sizeof(ST), K = 16 / ES, S = kLineSteps, NS = kBwdStages;
    const Shape& sh = a.sh;
    const int H = sh.H, W = sh.W, L = sh.Lmax();
    LineBwdParams prm{};
    prm.B = sh.B; prm.C = sh.C; prm.H = H; prm.W = W; prm.G = sh.G;
    prm.mask = sh.mask;
    int q = 0;
    for (int d = 0; d < 4; ++d) prm.slab[d] = (sh.mask >> d & 1u) ? q++ : -1;
    prm.pitch = line_pitch(W);
    prm.pb = (uint32_t)((S * L * ES + 127) / 128 * 128);
    prm.multi = (H == W && (uint32_t)(S * L * ES) == prm.pb) ? 1 : 0;
    uint32_t cols = 32;
    while (cols < (uint32_t)((H + 31) / 32 * 32 * P)) cols *= 2;
    prm.plane_cols = cols;
    prm.tm_cols = NC > 4 ? 2 * cols : cols;
    if (prm.tm_cols > 512) return GSPN_EUNSUPPORTED;
    prm.Lpad = 32 * P;
    prm.nblk_max = (L + S - 1) / S;
    prm.part_stride = (uint32_t)(4 * 3 * prm.Lpad);
    size_t off = 0;
    prm.ring_off = 0; off += (size_t)NS * PL::N2 * prm.pb;
    prm.out_off = (uint32_t)off; off += (size_t)2 * PL::NOUT * prm.pb;
    prm.part_off = (uint32_t)off; off += (size_t)2 * NC * prm.part_stride * 4;
    prm.ckpt_off = (uint32_t)off; off += (size_t)NC * prm.nblk_max * prm.Lpad * 4;
    prm.bar_off = (uint32_t)((off + 15) / 16 * 16); off = prm.bar_off + (2 * NS) * 8 + 16;
    if (off > (size_t)kMaxSmemOptin) return GSPN_EUNSUPPORTED;
    if ((size_t)2 * NC * prm.part_stride * 4 < (size_t)32 * prm.pitch * 4) return GSPN_EUNSUPPORTED;   // transposition tile
    prm.h0 = a.h0; prm.dx = a.dx; prm.dh0 = a.dh0;
    prm.want_dlam = a.dlam != nullptr; prm.want_du = a.du != nullptr; prm.want_dw3 = a.dw3 != nullptr;

    const int D = sh.D();
    const uint64_t nC = (uint64_t)D * sh.B * sh.C, nX = (uint64_t)sh.B * sh.C, nW = (uint64_t)D * sh.B * sh.G * 3;
    const uint64_t row_b = (uint64_t)W * ES, plane_b = (uint64_t)H * W * ES;
    BwdMaps mv, mh;
    struct T { CUtensorMap *v, *h; const void* p; uint64_t planes; uint32_t np; };
    const T ts[8] = {
        {&mv.lx, &mh.lx, a.x, nX, (uint32_t)NC}, {&mv.lw, &mh.lw, a.w3, nW, 3u}, {&mv.ll, &mh.ll, a.lam, nC, (uint32_t)NC},
        {&mv.lu, &mh.lu, a.u, nC, (uint32_t)NC}, {&mv.ldy, &mh.ldy, a.dy, nX, (uint32_t)NC},
        {&mv.sl, &mh.sl, a.dlam ? (const void*)a.dlam : a.lam, nC, (uint32_t)NC},
        {&mv.su, &mh.su, a.du ? (const void*)a.du : a.u, nC, (uint32_t)NC},
        {&mv.sw, &mh.sw, a.dw3 ? (const void*)a.dw3 : a.w3, nW, 3u}};
    for (const T& t : ts) {
        const uint32_t np = prm.multi ? t.np : 1u;
        const uint64_t dv[3] = {(uint64_t)W, (uint64_t)H, t.planes};
        const uint64_t sv[2] = {row_b, plane_b};
        const uint32_t bv[3] = {(uint32_t)W, (uint32_t)S, np};
        if (!encode_tensor_map(t.v, ES, const_cast<void*>(t.p), 3, dv, sv, bv)) return GSPN_ECUDA;
        const uint64_t dh[4] = {(uint64_t)K, (uint64_t)H, (uint64_t)(W / K), t.planes};
        const uint64_t shh[3] = {row_b, 16u, plane_b};
        const uint32_t bh[4] = {(uint32_t)K, (uint32_t)H, (uint32_t)(S / K), np};
        if (!encode_tensor_map(t.h, ES, const_cast<void*>(t.p), 4, dh, shh, bh)) return GSPN_ECUDA;
    }
    auto kern = line_bwd_kernel<ST, NC, P>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("line bwd: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    GSPN_LAUNCH(kern, sh.B * sh.G, (NC + 1) * 32, off, st, mv, mh, prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("line bwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST, int P>
static int line_bwd_nc(const BwdArgs<ST>& a, cudaStream_t st) {
    switch (a.sh.cg()) {
    case 1: return line_bwd_run<ST, 1, P>(a, st);
    case 2: return line_bwd_run<ST, 2, P>(a, st);
    case 4: return line_bwd_run<ST, 4, P>(a, st);
    case 8: if constexpr (P <= 2) return line_bwd_run<ST, 8, P>(a, st); else return GSPN_EUNSUPPORTED;
    default: return GSPN_EUNSUPPORTED;
    }
}

template <typename ST>
int line_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    const Shape& sh = a.sh;
    if ((sh.W * ES) % 16 != 0) { set_error("line bwd: rows of %d B are not 16-byte aligned", sh.W * ES); return GSPN_EUNSUPPORTED; }
    if (sh.Lmax() > 128) { set_error("line bwd: lines of %d positions exceed 4 per lane", sh.Lmax()); return GSPN_EUNSUPPORTED; }
    const int P = sh.Lmax() <= 32 ? 1 : sh.Lmax() <= 64 ? 2 : 4;
    int rc = P == 1 ? line_bwd_nc<ST, 1>(a, st) : P == 2 ? line_bwd_nc<ST, 2>(a, st) : line_bwd_nc<ST, 4>(a, st);
    if (rc == GSPN_EUNSUPPORTED)
        set_error("line bwd: C/G = %d channels of %dx%d do not fit one CTA (shared or tensor memory)", sh.cg(), sh.H, sh.W);
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "line_bwd"; }
    return rc;
}

template int line_bwd_launch<float>(const BwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int line_bwd_launch<__nv_bfloat16>(const BwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
