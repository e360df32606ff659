// gspn_line_fwd.cu -- forward scan for 16-byte-aligned rows (the 2K config 128x128, the classification stage 56x56,
// the tiny config): ONE launch, all four directions, y written once.
//
// CTA = NC <= 4 channels of one (b, group) unit.  Warp w < 8: the scan line of channel c = w % 4 in direction
// d = w / 4 of the current axis pair (T->B / B->T first, then L->R / R->L); warps 8, 9: one TMA producer per
// direction of the pair.  The taps of a stage are shared by the NC channel warps (Eq. 5).
//
// The fp32 sum y = sum_d u_d h_d lives in TENSOR MEMORY, not in shared memory: channel c owns lane quarter c (the
// quarter warps c and c + 4 can reach), one lane per thread, so shared memory is left to the operand ring -- what
// bounds this kernel is the bytes in flight per SM (measured: about 1.9 us per stage fetch under load).
//   T->B / B->T: lane a owns the P adjacent columns P*a + k; pixel (i, P*a + k) is column i*P + k of lane a.
//   L->R / R->L: lane b owns the rows b + 32*k;              pixel (b + 32*k, j) is column k*32*P + j of lane b.
// Between the two axes warp c turns its plane from the first layout into the second, 32 image rows at a time and in
// place (rows 32*t .. 32*t+31 occupy columns [32*P*t, 32*P*(t+1)) in both layouts), through a shared-memory tile.
// The two directions of an axis start at opposite ends; each owns its half of the plane until they meet at a named
// barrier and swap halves, so every element has one writer at a time; the half a direction touches first on an
// untouched plane is stored, not read.  One RNE per output element when the finished plane leaves (Eq. 2, 9).
#include "gspn_line.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {
namespace {
#ifndef LINE_EXP
#define LINE_EXP 0
#endif
#ifdef LINE_SPIN
#define mbar_wait mbar_wait_spin
#endif

#ifndef GSPN_EMU
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#else
inline unsigned long long gtime() { return 0; }
#endif
struct LineFwdParams {
    int B, C, H, W, G, cg;
    unsigned mask;
    int slab[4];          // slab index of each direction inside w3 / lambda / u (ascending bit order)
    int pitch;            // floats per row of the transposition tile
    uint32_t pb_bytes;    // bytes between operand planes inside a row stage (T->B / B->T)
    uint32_t pbh_bytes;   // bytes between operand planes inside a column stage (L->R / R->L): H rows of 32 bytes
    uint32_t ring_bytes;  // max(2 * kLineStages row stages, 3 column stages)
    int multi;            // 1: one TMA box brings all planes of an operand (taps x3, lambda / u / x x NC)
    uint32_t tm_cols;     // tensor-memory columns of the CTA (power of two >= 32)
    const void* h0;
    const void *x, *w3, *lam, *u;   // the same tensors as the maps, for 1-D bulk copies of whole rows
    void* y;
};

// what a scan-line warp knows about its place in the CTA
struct LineCtx {
    int H, W, lane, c, d;
    unsigned char* ring;          // the ring of this warp's direction slot d: kLineStages stages
    uint64_t *full, *empty;       // [kLineStages] barriers of direction slot d
    uint32_t pb, stage_bytes, pbh;
    uint32_t tb;                  // tensor-memory address of this channel's lane quarter, column 0
    int it;                       // stages this direction slot has consumed so far
    void* dbg;
};

// The taps that leave the grid are never used (reading 3): every warp zeroes them in the stage it is about
// to read -- all warps of a direction write the same zeros, each before its own reads -- so that the scan steps need
// no boundary selects and a NaN stored there cannot reach h through 0 * NaN.
template <typename ST>
__device__ __forceinline__ void line_zero_edge_taps_v(unsigned char* sb, uint32_t pb, int W, int lane) {
    if (lane < kLineSteps) {
        ST* t0 = reinterpret_cast<ST*>(sb) + lane * W;                   // tap 0 of column 0
        ST* t2 = reinterpret_cast<ST*>(sb + 2 * pb) + lane * W + W - 1;  // tap 2 of column W-1
        *t0 = ST(0.f);
        *t2 = ST(0.f);
    }
    __syncwarp();
}
// offset of 16-byte piece hh of row r inside a column-stage plane (32-byte rows, TMA SWIZZLE_32B: address bit 4 ^= bit 7)
__device__ __forceinline__ uint32_t line_hoff(int r, int hh) { return (uint32_t)(r * 32 + ((hh ^ ((r >> 2) & 1)) << 4)); }
__device__ __forceinline__ void line_zero_edge_taps_h(unsigned char* sb, uint32_t pbh, int H, int lane) {
    if (lane < 2) {
        *reinterpret_cast<uint4*>(sb + line_hoff(0, lane)) = make_uint4(0, 0, 0, 0);                   // tap 0, row 0
        *reinterpret_cast<uint4*>(sb + 2 * pbh + line_hoff(H - 1, lane)) = make_uint4(0, 0, 0, 0);     // tap 2, row H-1
    }
    __syncwarp();
}
// generic-proxy writes to a stage are ordered before the TMA writes that refill it
__device__ __forceinline__ void line_release_stage(uint64_t* empty_bar, int lane) {
    fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(empty_bar);
}

// one scan step of a vertical direction: operands of image row `row` of the stage, accumulator row i
template <typename ST, int NC, int P>
__device__ __forceinline__ void line_fwd_vstep(const LineCtx& cx, const ST* row, uint32_t pbe, int i, bool acc,
                                               float (&h)[P]) {
    float w0[P], w1[P], w2[P], uu[P];
    LineRaw<ST, P> la, xx;
    line_ld<ST, P>(row, w0);
    line_ld<ST, P>(row + pbe, w1);
    line_ld<ST, P>(row + 2 * pbe, w2);
    line_ld_raw<ST, P>(row + (3 + cx.c) * pbe, la);
    line_ld<ST, P>(row + (3 + NC + cx.c) * pbe, uu);
    line_ld_raw<ST, P>(row + (3 + 2 * NC + cx.c) * pbe, xx);
    float yv[P];
    if (acc) tm_ld<P>(cx.tb + i * P, yv);
    const float hl = __shfl_up_sync(0xffffffffu, h[P - 1], 1);     // lane 0 / the last lane: multiplied by a zeroed tap
    const float hr = __shfl_down_sync(0xffffffffu, h[0], 1);
    float hn[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const float l = k == 0 ? hl : h[k - 1];
        const float r = k == P - 1 ? hr : h[k + 1];
        hn[k] = fmaf(w0[k], l, fmaf(w2[k], r, line_fma_raw<ST>(la.w, xx.w, k, w1[k] * h[k])));
    }
#pragma unroll
    for (int k = 0; k < P; ++k) h[k] = hn[k];
    if (acc) {
        tm_wait_ld<P>(yv);
#pragma unroll
        for (int k = 0; k < P; ++k) yv[k] = fmaf(uu[k], h[k], yv[k]);
    } else {
#pragma unroll
        for (int k = 0; k < P; ++k) yv[k] = uu[k] * h[k];
    }
    tm_st<P>(cx.tb + i * P, yv);
}

// a vertical direction (d = 0: T->B, d = 1: B->T): steps [0, first) store into the plane; with `both` the two directions
// then meet and steps [first, H) add to what the other one left
template <typename ST, int NC, int P>
__device__ __forceinline__ void line_fwd_vrun(const LineCtx& cx, int first, bool both, float (&h)[P]) {
    constexpr int S = kLineSteps, NS = kLineStages, ES = sizeof(ST);
    const int H = cx.H, W = cx.W, lane = cx.lane, d = cx.d;
    const int lp = lane < W / P ? lane : 0;
    const uint32_t pbe = cx.pb / ES;
    for (int seg = 0; seg < (both ? 2 : 1); ++seg) {
    const bool acc = seg == 1;
    const int s_end = seg ? H : first;
    int s = seg ? first : 0;
    if (seg) tm_pair_sync(1 + cx.c);
    while (s < s_end) {
        const int blk = s / S, r0 = s % S;
        const int r1 = min(S, r0 + (s_end - s));
        const int cur = cx.it + blk, stg = cur % NS;
        unsigned char* sb = cx.ring + (size_t)stg * cx.stage_bytes;
        if (r0 == 0) {
            mbar_wait(&cx.full[stg], (cur / NS) & 1);
            if (LINE_EXP == 3 && lane == 0 && blockIdx.x == 0 && d == 0 && cx.c == 0) reinterpret_cast<unsigned long long*>(cx.dbg)[64 + cur] = gtime();
            line_zero_edge_taps_v<ST>(sb, cx.pb, W, lane);
        }
        const ST* base = reinterpret_cast<const ST*>(sb) + P * lp;
        const int i0 = d ? H - 1 - blk * S : blk * S;          // image row of step r = 0 of this stage
        if (LINE_EXP == 1 || LINE_EXP == 3) {
        } else if (r0 == 0 && r1 == S && acc) {
#pragma unroll
            for (int r = 0; r < S; ++r)
                line_fwd_vstep<ST, NC, P>(cx, base + (d ? S - 1 - r : r) * W, pbe, d ? i0 - r : i0 + r, true, h);
        } else if (r0 == 0 && r1 == S) {
#pragma unroll
            for (int r = 0; r < S; ++r)
                line_fwd_vstep<ST, NC, P>(cx, base + (d ? S - 1 - r : r) * W, pbe, d ? i0 - r : i0 + r, false, h);
        } else {
            for (int r = r0; r < r1; ++r)
                line_fwd_vstep<ST, NC, P>(cx, base + (d ? S - 1 - r : r) * W, pbe, d ? i0 - r : i0 + r, acc, h);
        }
        s += r1 - r0;
        if (r1 == S || s == H) line_release_stage(&cx.empty[stg], lane);
    }
    }
}

// one column stage (2 * 16 / ES columns: rows of 32 bytes) of one channel; REV: R->L (columns descending).
// Lane b owns rows b + 32k.
template <typename ST, int NC, int P, bool REV>
__device__ __forceinline__ void line_fwd_hstage(const LineCtx& cx, const unsigned char* sb, int blk, bool both, int first,
                                                bool touched, float (&h)[P]) {
    constexpr int ES = sizeof(ST), K = 16 / ES, NCH = 2, S = NCH * K;
    const int H = cx.H, W = cx.W, lane = cx.lane, c = cx.c;
    const uint32_t pb = cx.pbh;
    const int src_up = (lane + 31) & 31, src_dn = (lane + 1) & 31;
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        const int s0 = blk * S + n * K;                      // first scan step of this 16-byte piece
        if (s0 >= W) return;
        const int cn = REV ? NCH - 1 - n : n;                // piece inside the 32-byte row (columns ascend in memory)
        uint32_t rw[6][P][4];                                // raw 16-byte pieces: taps, lambda, u, x
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const int row = lane + 32 * k;
            const unsigned char* p16 = sb + line_hoff(row < H ? row : 0, cn);
            lds_vec<16>(p16, rw[0][k]);
            lds_vec<16>(p16 + pb, rw[1][k]);
            lds_vec<16>(p16 + 2 * pb, rw[2][k]);
            lds_vec<16>(p16 + (size_t)(3 + c) * pb, rw[3][k]);
            lds_vec<16>(p16 + (size_t)(3 + NC + c) * pb, rw[4][k]);
            lds_vec<16>(p16 + (size_t)(3 + 2 * NC + c) * pb, rw[5][k]);
        }
#pragma unroll
        for (int t4 = 0; t4 < K; t4 += 4) {
            const int s = s0 + t4;                           // four steps = four adjacent columns
            if (both && s == first) tm_pair_sync(1 + c);
            const bool acc = touched || (both && s >= first);
            const int j0 = REV ? W - 4 - s : s;              // lowest column of the group
            float yv[P][4];
            if (acc) {
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    if (32 * k < H) tm_ld<4>(cx.tb + k * 32 * P + j0, yv[k]);      // slots past the plane own no columns
                    else yv[k][0] = yv[k][1] = yv[k][2] = yv[k][3] = 0.f;
                }
            }
#pragma unroll
            for (int tt = 0; tt < 4; ++tt) {
                const int e = REV ? K - 1 - (t4 + tt) : t4 + tt;       // element inside the 16-byte chunk
                const int ye = REV ? 3 - tt : tt;
                // the row above (b + 32k - 1) is slot k of lane b-1, or slot k-1 of lane 31 for lane 0: lane 31 only
                // serves lane 0, so it sends the slot below; likewise lane 0 serves lane 31 with the slot above
                float up[P], dn[P];
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const float su = (k > 0 && lane == 31) ? h[k > 0 ? k - 1 : 0] : h[k];
                    const float sd = (k < P - 1 && lane == 0) ? h[k < P - 1 ? k + 1 : k] : h[k];
                    up[k] = __shfl_sync(0xffffffffu, su, src_up);
                    dn[k] = __shfl_sync(0xffffffffu, sd, src_dn);
                }
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const float a0 = line_elem<ST>(rw[0][k], e), a1 = line_elem<ST>(rw[1][k], e);
                    const float a2 = line_elem<ST>(rw[2][k], e);
                    h[k] = fmaf(a0, up[k], fmaf(a2, dn[k], line_fma_raw<ST>(rw[3][k], rw[5][k], e, a1 * h[k])));
                }
                if (tt == 0 && acc) {
#pragma unroll
                    for (int k = 0; k < P; ++k) if (32 * k < H) tm_wait_ld<4>(yv[k]);
                }
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const float uu = line_elem<ST>(rw[4][k], e);
                    yv[k][ye] = acc ? fmaf(uu, h[k], yv[k][ye]) : uu * h[k];
                }
            }
#pragma unroll
            for (int k = 0; k < P; ++k) if (32 * k < H) tm_st<4>(cx.tb + k * 32 * P + j0, yv[k]);
        }
    }
}

template <typename ST, int NC, int P>
__global__ void __launch_bounds__(320, 1)
line_fwd_kernel(const __grid_constant__ CUtensorMap mxv, const __grid_constant__ CUtensorMap mwv,
                const __grid_constant__ CUtensorMap mlv, const __grid_constant__ CUtensorMap muv,
                const __grid_constant__ CUtensorMap mxh, const __grid_constant__ CUtensorMap mwh,
                const __grid_constant__ CUtensorMap mlh, const __grid_constant__ CUtensorMap muh,
                const LineFwdParams prm) {
    constexpr int ES = sizeof(ST);
    constexpr int K = 16 / ES;                     // scan steps per 16-byte column chunk
    constexpr int S = kLineSteps;
    constexpr int NS = kLineStages;
    constexpr int NPL = 3 + 3 * NC;                // operand planes per stage: taps, lambda, u, x
    constexpr int NT = NC < 2 ? NC : 2;            // transposition tiles (channels c and c + 2 take turns)

    extern __shared__ __align__(128) unsigned char smem[];
    const int H = prm.H, W = prm.W;
    const uint32_t stage_bytes = NPL * prm.pb_bytes;
    const uint32_t hstage_bytes = NPL * prm.pbh_bytes;
    unsigned char* const ring = smem;              // row stages [2][NS]; later the same bytes as 3 column stages
    float* const tiles = reinterpret_cast<float*>(ring + prm.ring_bytes);
    const size_t tile_floats = (size_t)32 * prm.pitch;
    uint64_t* const bars = reinterpret_cast<uint64_t*>(tiles + NT * tile_floats);
    uint64_t* const full = bars;                   // [2][NS]
    uint64_t* const empty = bars + 2 * NS;         // [2][NS]
    uint64_t* const tfree = bars + 4 * NS;         // [2]: transposition tile t is free again
    // column stages: 3 slots shared by L->R and R->L.  A slot alternates between the directions, and an mbarrier wait
    // by parity must see EVERY phase of its barrier (a waiter that skips one takes the phase before for the one it
    // wants), so each direction has its own "full" barrier per slot: its k-th use of a slot is phase k there.  The
    // producer alone waits on the "empty" barriers, and it sees every phase.
    uint64_t* const fullh = bars + 4 * NS + 2;     // [2 directions][3 slots]
    uint64_t* const emptyh = bars + 4 * NS + 8;    // [3 slots]
    uint64_t* const vdone = bars + 4 * NS + 11;    // every scan-line warp has left the row stages
    uint32_t* const tm_slot = reinterpret_cast<uint32_t*>(bars + 4 * NS + 12);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int subs = prm.cg / NC;
    const int item = blockIdx.x;
    const int sub = item % subs;
    const int g = (item / subs) % prm.G;
    const int b = item / (subs * prm.G);
    const int c0 = g * prm.cg + sub * NC;          // first channel of this CTA
    const unsigned mask = prm.mask;

    if (threadIdx.x == 0) {
        for (int i = 0; i < 2 * NS; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NC); }
        mbar_init(&tfree[0], 1); mbar_init(&tfree[1], 1);
        for (int i = 0; i < 6; ++i) mbar_init(&fullh[i], 1);
        for (int i = 0; i < 3; ++i) mbar_init(&emptyh[i], NC);
        mbar_init(vdone, 2 * NC);
        mbar_init_fence();
    }
    if (warp == 8) tm_alloc(tm_slot, prm.tm_cols);
    tm_fence_before();
    __syncthreads();
    tm_fence_after();
    const uint32_t tm_base = *tm_slot;

    constexpr int SH = 2 * K;                      // scan steps per column stage
    const int nblk_v = (H + S - 1) / S, nblk_h = (W + SH - 1) / SH;

    if (warp >= 8) {
        // ------------------------------------------------------------------ producers
        // this lane's box: first plane inside its tensor, first plane slot inside the stage
        int plane = 0, slot = 0;
        const CUtensorMap* map = nullptr;
        const unsigned char* gsrc = nullptr;       // the lane's tensor, for row stages brought by 1-D bulk copies
        bool issue = false;
        auto roles = [&](int dir, int ph) {
            const int q = prm.slab[dir];
            const int pw = ((q * prm.B + b) * prm.G + g) * 3, pc = (q * prm.B + b) * prm.C + c0, px = b * prm.C + c0;
            map = nullptr; gsrc = nullptr;
            if (prm.multi) {                       // 4 boxes per stage, each with all planes of one operand
                issue = lane < 4;
                if (lane == 0) { plane = pw; slot = 0; map = ph ? &mwh : &mwv; }
                else if (lane == 1) { plane = pc; slot = 3; map = ph ? &mlh : &mlv; }
                else if (lane == 2) { plane = pc; slot = 3 + NC; map = ph ? &muh : &muv; }
                else if (lane == 3) { plane = px; slot = 3 + 2 * NC; map = ph ? &mxh : &mxv; }
            } else {
                issue = lane < NPL;
                slot = lane;
                if (lane < 3) { plane = pw + lane; map = ph ? &mwh : &mwv; gsrc = (const unsigned char*)prm.w3; }
                else if (lane < 3 + NC) { plane = pc + (lane - 3); map = ph ? &mlh : &mlv; gsrc = (const unsigned char*)prm.lam; }
                else if (lane < 3 + 2 * NC) { plane = pc + (lane - 3 - NC); map = ph ? &muh : &muv; gsrc = (const unsigned char*)prm.u; }
                else if (lane < NPL) { plane = px + (lane - 3 - 2 * NC); map = ph ? &mxh : &mxv; gsrc = (const unsigned char*)prm.x; }
                if (gsrc) gsrc += (size_t)plane * H * W * ES;
            }
        };
        // ---- row stages of T->B (warp 8) / B->T (warp 9): a ring of NS stages each
        const int d = warp - 8;
        if (mask >> d & 1u) {
            roles(d, 0);
            const uint32_t tx = (uint32_t)(NPL * S * ES) * (uint32_t)W;
            for (int it = 0; it < nblk_v; ++it) {
                const int stg = it % NS;
                if (it >= NS) mbar_wait(&empty[d * NS + stg], ((it / NS) - 1) & 1);
                uint64_t* fb = &full[d * NS + stg];
                const int s0 = d ? H - (it + 1) * S : it * S;        // first row of the stage (may be < 0)
                const bool rows1d = !prm.multi;                      // row stages of single planes: contiguous in HBM
                const int r_lo = s0 < 0 ? 0 : s0, r_hi = s0 + S > H ? H : s0 + S;
                const uint32_t rbytes = (uint32_t)(r_hi - r_lo) * W * ES;
                if (lane == 0) { if (LINE_EXP == 2) mbar_arrive(fb); else mbar_arrive_expect_tx(fb, rows1d ? NPL * rbytes : tx); }
                __syncwarp();
                if (issue && LINE_EXP != 2) {
                    unsigned char* dst = ring + (size_t)(d * NS + stg) * stage_bytes + (size_t)slot * prm.pb_bytes;
                    if (rows1d) bulk_load_1d(dst + (size_t)(r_lo - s0) * W * ES, gsrc + (size_t)r_lo * W * ES, rbytes, fb);
                    else tma_load_3d(dst, map, 0, s0, plane, fb);
                }
            }
        }
        // ---- column stages (rows of 32 bytes) of L->R and R->L: ONE ring of 3 stages over the same bytes, filled by
        // warp 8 in the order L->R 0, R->L 0, L->R 1, ... once every scan-line warp has left the row stages
        if (warp == 8 && (mask & 12u)) {
            mbar_wait(vdone, 0);
            const bool both = (mask & 12u) == 12u;
            const int nst = both ? 2 * nblk_h : nblk_h;
            const uint32_t tx = (uint32_t)NPL * 32u * (uint32_t)H;
            int cur_dir = -1;
            for (int n = 0; n < nst; ++n) {
                const int dd = both ? (n & 1) : ((mask >> 3) & 1u ? ((mask >> 2) & 1u ? 0 : 1) : 0);
                const int blk = both ? n >> 1 : n;
                if (2 + dd != cur_dir) { cur_dir = 2 + dd; roles(cur_dir, 1); }
                const int stg = n % 3;
                if (n >= 3) mbar_wait(&emptyh[stg], ((n / 3) - 1) & 1);
                uint64_t* fb = &fullh[dd * 3 + stg];
                if (lane == 0) { if (LINE_EXP == 2) mbar_arrive(fb); else mbar_arrive_expect_tx(fb, tx); }
                __syncwarp();
                if (issue && LINE_EXP != 2) {
                    unsigned char* dst = ring + (size_t)stg * hstage_bytes + (size_t)slot * prm.pbh_bytes;
                    const int j0 = dd ? W - (blk + 1) * SH : blk * SH;   // first column of the stage (may be < 0)
                    tma_load_3d(dst, map, j0, 0, plane, fb);
                }
            }
        }
    } else if ((warp & 3) < NC) {
        // ------------------------------------------------------------------ scan line of channel c, direction slot d
        LineCtx cx;
        cx.H = H; cx.W = W; cx.lane = lane; cx.c = warp & 3; cx.d = warp >> 2;
        cx.ring = ring + (size_t)cx.d * NS * stage_bytes;
        cx.full = full + cx.d * NS; cx.empty = empty + cx.d * NS;
        cx.pb = prm.pb_bytes; cx.stage_bytes = stage_bytes; cx.pbh = prm.pbh_bytes;
        cx.tb = tm_base + ((uint32_t)(32 * cx.c) << 16);
        cx.it = 0; cx.dbg = prm.y;
        const int c = cx.c, d = cx.d, ch = c0 + c;
        const size_t Lmax = H > W ? H : W;
        const bool any_v = (mask & 3u) != 0, any_h = (mask & 12u) != 0;

        // ---- T->B (d = 0) / B->T (d = 1)
        if (mask >> d & 1u) {
            const bool both = (mask & 3u) == 3u;
            float h[P];
#pragma unroll
            for (int k = 0; k < P; ++k) h[k] = 0.f;
            if (prm.h0 && lane < W / P) {
                const ST* hp = reinterpret_cast<const ST*>(prm.h0) +
                               ((size_t)(prm.slab[d] * prm.B + b) * prm.C + ch) * Lmax + P * lane;
#pragma unroll
                for (int k = 0; k < P; ++k) h[k] = ld_f(hp + k);
            }
            const int Hh = (H + 1) / 2;
            const int first = both ? (d == 0 ? Hh : H - Hh) : H;     // steps on the half this direction touches first
            line_fwd_vrun<ST, NC, P>(cx, first, both, h);
            cx.it += nblk_v;
        } else if ((mask & 3u) == 3u) {
            tm_pair_sync(1 + c);
        }
        tm_pair_sync(1 + c);                       // the vertical sums of this channel are complete
        if (lane == 0) mbar_arrive(vdone);         // this warp has left the row stages (their bytes become column stages)

        // ---- the plane turns into the row-owner layout
        if (any_v && any_h) {
            if (d == 0) {
                if (c >= 2) mbar_wait(&tfree[c - 2], 0);
                line_transpose<P>(cx.tb, tiles + (size_t)(c & 1) * tile_floats, prm.pitch, H, W, lane);
                if (c < 2 && lane == 0) mbar_arrive(&tfree[c]);
            }
            tm_pair_sync(1 + c);
        }

        // ---- L->R (d = 0) / R->L (d = 1)
        if (mask >> (2 + d) & 1u) {
            const bool both = (mask & 12u) == 12u;
            float h[P];
#pragma unroll
            for (int k = 0; k < P; ++k) h[k] = 0.f;
            if (prm.h0) {
                const ST* hp = reinterpret_cast<const ST*>(prm.h0) +
                               ((size_t)(prm.slab[2 + d] * prm.B + b) * prm.C + ch) * Lmax;
#pragma unroll
                for (int k = 0; k < P; ++k) if (lane + 32 * k < H) h[k] = ld_f(hp + lane + 32 * k);
            }
            const int Wh = (W / 2 + 3) / 4 * 4;                        // swap point, a multiple of 4 columns
            const int first = both ? (d == 0 ? Wh : W - Wh) : W;
            for (int blk = 0; blk < nblk_h; ++blk) {
                const int n = both ? 2 * blk + d : blk, stg = n % 3;      // place in the shared ring of column stages
                mbar_wait(&fullh[d * 3 + stg], (blk / 3) & 1);      // this direction's (blk / 3)-th use of the slot
                unsigned char* sb = ring + (size_t)stg * hstage_bytes;
                line_zero_edge_taps_h(sb, cx.pbh, H, lane);
                if (LINE_EXP == 1 || LINE_EXP == 3) {}
                else if (d) line_fwd_hstage<ST, NC, P, true>(cx, sb, blk, both, first, any_v, h);
                else line_fwd_hstage<ST, NC, P, false>(cx, sb, blk, both, first, any_v, h);
                line_release_stage(&emptyh[stg], lane);
            }
            if (both && first >= W) tm_pair_sync(1 + c);
        } else if ((mask & 12u) == 12u) {
            tm_pair_sync(1 + c);
        }
        tm_pair_sync(1 + c);                       // the plane of this channel is complete

        // ---- the finished plane leaves: one RNE per element
        ST* yg = reinterpret_cast<ST*>(prm.y) + ((size_t)b * prm.C + ch) * H * W;
        if (LINE_EXP == 3) {
        } else if (any_h) {                               // row-owner layout: 16-byte pieces of this lane's rows
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const int i = lane + 32 * k;
                if (32 * k >= H) continue;
                for (int jc = d; jc * K < W; jc += 2) {
                    float f[K];
                    tm_ld<K>(cx.tb + k * 32 * P + jc * K, f);
                    tm_wait_ld<K>(f);
                    uint32_t r[4];
                    Store<ST>::template pack<16>(f, r);
                    if (i < H) *reinterpret_cast<uint4*>(yg + (size_t)i * W + jc * K) = make_uint4(r[0], r[1], r[2], r[3]);
                }
            }
        } else {                                   // column-owner layout: a warp writes whole rows
            for (int i = d; i < H; i += 2) {
                float f[P];
                tm_ld<P>(cx.tb + i * P, f);
                tm_wait_ld<P>(f);
                if (lane < W / P) {
#pragma unroll
                    for (int k = 0; k < P; ++k) st_f(yg + (size_t)i * W + P * lane + k, f[k]);
                }
            }
        }
    }
    tm_fence_before();
    __syncthreads();
    if (warp == 8) tm_dealloc(tm_base, prm.tm_cols);
}

}  // namespace

// ---- host side ---------------------------------------------------------------------------------------------------
template <typename ST, int NC, int P>
static int line_fwd_run(const FwdArgs<ST>& a, cudaStream_t st) {
    constexpr int ES = sizeof(ST);
    constexpr int K = 16 / ES;
    constexpr int S = kLineSteps;
    constexpr int NT = NC < 2 ? NC : 2;
    const Shape& sh = a.sh;
    const int H = sh.H, W = sh.W, L = sh.Lmax();
    LineFwdParams prm{};
    prm.B = sh.B; prm.C = sh.C; prm.H = H; prm.W = W; prm.G = sh.G; prm.cg = sh.cg();
    prm.mask = sh.mask;
    int q = 0;
    for (int d = 0; d < 4; ++d) prm.slab[d] = (sh.mask >> d & 1u) ? q++ : -1;
    prm.pitch = line_pitch(W);
    // TMA destinations are 128-byte aligned.  Square planes whose stage planes are a multiple of 128 bytes take one box per
    // operand (the planes of a box land back to back); other shapes take one box per plane at a padded pitch.
    prm.multi = ((S * W * ES) % 128 == 0 && H % 8 == 0) ? 1 : 0;
#ifdef LINE_NOMULTI
    prm.multi = 0;
#endif
    prm.pb_bytes = (uint32_t)((S * W * ES + 127) / 128 * 128);
    prm.pbh_bytes = (uint32_t)((H * 32 + 255) / 256 * 256);        // SWIZZLE_32B repeats every 256 bytes
    const size_t ring_v = (size_t)2 * kLineStages * (3 + 3 * NC) * prm.pb_bytes, ring_h = (size_t)3 * (3 + 3 * NC) * prm.pbh_bytes;
    prm.ring_bytes = (uint32_t)(((ring_v > ring_h ? ring_v : ring_h) + 1023) / 1024 * 1024);
    uint32_t cols = 32;
    while (cols < (uint32_t)((H + 31) / 32 * 32 * P)) cols *= 2;
    prm.tm_cols = cols;
    prm.h0 = a.h0; prm.y = a.y;
    prm.x = a.x; prm.w3 = a.w3; prm.lam = a.lam; prm.u = a.u;
    const size_t smem = (size_t)prm.ring_bytes + (size_t)NT * 32 * prm.pitch * 4 + (4 * kLineStages + 12) * 8 + 16;
    if (smem > (size_t)kMaxSmemOptin) return GSPN_EUNSUPPORTED;

    const int D = sh.D();
    struct Src { const void* p; uint64_t planes; };
    const Src src[4] = {{a.x, (uint64_t)sh.B * sh.C}, {a.w3, (uint64_t)D * sh.B * sh.G * 3},
                        {a.lam, (uint64_t)D * sh.B * sh.C}, {a.u, (uint64_t)D * sh.B * sh.C}};
    // The eight tensor maps depend on the operand addresses and the shape only: the last set of this host thread is kept
    // (a cached launch descriptor, include/gspn.h) so that repeated calls on the same buffers skip the driver's encoder.
    struct MapCache { const void* p[4]; int B, C, H, W, G, multi; CUtensorMap m[8]; bool valid; };
    static thread_local MapCache mc{};
    const bool hit = mc.valid && mc.p[0] == a.x && mc.p[1] == a.w3 && mc.p[2] == a.lam && mc.p[3] == a.u && mc.B == sh.B &&
                     mc.C == sh.C && mc.H == H && mc.W == W && mc.G == (int)(sh.G * 16 + NC) && mc.multi == prm.multi * 8 + D;
    CUtensorMap* const m = mc.m;
    if (!hit) {
        mc.valid = false;
        const uint64_t row_b = (uint64_t)W * ES, plane_b = (uint64_t)H * W * ES;
        for (int t = 0; t < 4; ++t) {
            const uint64_t dv[3] = {(uint64_t)W, (uint64_t)H, src[t].planes};
            const uint64_t sv[2] = {row_b, plane_b};
            const uint32_t np = prm.multi ? (t == 1 ? 3u : (uint32_t)NC) : 1u;      // planes per box
            const uint32_t bv[3] = {(uint32_t)W, (uint32_t)S, np};
            if (!encode_tensor_map(&m[t], ES, const_cast<void*>(src[t].p), 3, dv, sv, bv)) return GSPN_ECUDA;
            // column stages: a box is 32 bytes wide and the whole plane height; SWIZZLE_32B keeps the lanes' 16-byte
            // reads (one row per lane) free of bank conflicts
            const uint32_t bh[3] = {(uint32_t)(2 * K), (uint32_t)H, np};
            if (!encode_tensor_map(&m[4 + t], ES, const_cast<void*>(src[t].p), 3, dv, sv, bh, 1)) return GSPN_ECUDA;
        }
        mc.p[0] = a.x; mc.p[1] = a.w3; mc.p[2] = a.lam; mc.p[3] = a.u;
        mc.B = sh.B; mc.C = sh.C; mc.H = H; mc.W = W; mc.G = (int)(sh.G * 16 + NC); mc.multi = prm.multi * 8 + D;
        mc.valid = true;
    }
    auto kern = line_fwd_kernel<ST, NC, P>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("line fwd: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    const int items = sh.B * sh.G * (sh.cg() / NC);
    GSPN_LAUNCH(kern, items, 320, smem, st, m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("line fwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST, int P>
static int line_fwd_nc(const FwdArgs<ST>& a, cudaStream_t st) {
    const int cg = a.sh.cg();
    int rc = GSPN_EUNSUPPORTED;
    if (cg % 4 == 0) rc = line_fwd_run<ST, 4, P>(a, st);
    if (rc == GSPN_EUNSUPPORTED && cg % 2 == 0) rc = line_fwd_run<ST, 2, P>(a, st);
    if (rc == GSPN_EUNSUPPORTED) rc = line_fwd_run<ST, 1, P>(a, st);
    return rc;
}

template <typename ST>
int line_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    const Shape& sh = a.sh;
    const int H = sh.H, W = sh.W;
    if ((W * ES) % 16 != 0) { set_error("line fwd: rows of %d B are not 16-byte aligned", W * ES); return GSPN_EUNSUPPORTED; }
    if (sh.Lmax() > 128) { set_error("line fwd: lines of %d positions exceed 4 per lane", sh.Lmax()); return GSPN_EUNSUPPORTED; }
    const int P = sh.Lmax() <= 32 ? 1 : sh.Lmax() <= 64 ? 2 : 4;      // W % 4 == 0 follows from the row alignment
    int rc = P == 1 ? line_fwd_nc<ST, 1>(a, st) : P == 2 ? line_fwd_nc<ST, 2>(a, st) : line_fwd_nc<ST, 4>(a, st);
    if (rc == GSPN_EUNSUPPORTED) set_error("line fwd: the operand ring of %dx%d exceeds shared memory", H, W);
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "line_fwd"; }
    return rc;
}

template int line_fwd_launch<float>(const FwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int line_fwd_launch<__nv_bfloat16>(const FwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
