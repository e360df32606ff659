// gspn_line_fwd.cu -- forward scan for 16-byte-aligned rows (the 2K config 128x128, the classification stage 56x56,
// the tiny config): ONE launch, all four directions, y written once.
//
// CTA = NC channels of one (b, group) unit.  Warps 0, 1: producers (one per direction of the current axis pair);
// warp 2 + 2c + d: the scan line of channel c in direction d of the pair (T->B / B->T first, then L->R / R->L).
// A lane owns P adjacent positions of the line: h stays in registers, the two neighbours outside the lane's run
// come by one shuffle each per step.  Operands arrive in stages of kLineSteps scan steps (gspn_line.cuh) through a
// two-stage TMA ring per direction; the taps of a stage are shared by the NC channel warps (Eq. 5).
// y = sum_d u_d h_d is accumulated in ONE fp32 plane per channel in shared memory: the two directions of an axis
// start at opposite ends, each owns its half of the plane until they meet at a named barrier and swap halves, so
// every element has one writer at a time; the half a direction touches first on an untouched plane is stored, not
// read.  One RNE per output element when the finished plane leaves (Eq. 2, 9).
#include "gspn_line.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {
namespace {

struct LineFwdParams {
    int B, C, H, W, G, cg;
    unsigned mask;
    int slab[4];          // slab index of each direction inside w3 / lambda / u (ascending bit order)
    int HP, WP;           // H / P, W / P
    int pitch;            // floats per accumulator row
    uint32_t pb_bytes;    // bytes of one operand plane inside a stage
    const void* h0;
    void* y;
};

template <typename ST, int P>
__device__ __forceinline__ void line_step(float (&h)[P], const float (&w0)[P], const float (&w1)[P],
                                          const float (&w2)[P], const float (&lx)[P], bool first_lane,
                                          bool last_lane) {
    float hl = __shfl_up_sync(0xffffffffu, h[P - 1], 1);
    float hr = __shfl_down_sync(0xffffffffu, h[0], 1);
    if (first_lane) hl = 0.f;
    if (last_lane) hr = 0.f;
    float hn[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const float l = k == 0 ? hl : h[k - 1];
        const float r = k == P - 1 ? hr : h[k + 1];
        hn[k] = fmaf(w0[k], l, fmaf(w1[k], h[k], fmaf(w2[k], r, lx[k])));
    }
#pragma unroll
    for (int k = 0; k < P; ++k) h[k] = hn[k];
}

// one horizontal stage (kLineSteps columns) of one channel: REV = R->L (columns descending)
template <typename ST, int NC, int P, bool REV>
__device__ __forceinline__ void line_fwd_hstage(const unsigned char* sb, int blk, int H, int W, int HP, int lp, int lane,
                                                bool active, bool first_lane, bool last_lane, int c, uint32_t pb,
                                                int pitch, float* Yc, bool both, int first, bool touched,
                                                float (&h)[P]) {
    constexpr int ES = sizeof(ST);
    constexpr int K = 16 / ES;
    constexpr int S = kLineSteps;
    constexpr int NCH = S / K;
    #pragma unroll
                    for (int n = 0; n < NCH; ++n) {
                        const int s0 = blk * S + n * K;                    // first scan step of this chunk
                        if (s0 >= W) return;
                        const int cn = REV ? NCH - 1 - n : n;                // chunk inside the stage (ascending columns)
                        uint32_t rw[6][P][4];                              // raw 16-byte pieces: taps, lambda, u, x
    #pragma unroll
                        for (int k = 0; k < P; ++k) {
                            const unsigned char* p16 = sb + ((size_t)cn * H + k * HP + lp) * 16;
                            lds_vec<16>(p16, rw[0][k]);
                            lds_vec<16>(p16 + pb, rw[1][k]);
                            lds_vec<16>(p16 + 2 * pb, rw[2][k]);
                            lds_vec<16>(p16 + (size_t)(3 + c) * pb, rw[3][k]);
                            lds_vec<16>(p16 + (size_t)(3 + NC + c) * pb, rw[4][k]);
                            lds_vec<16>(p16 + (size_t)(3 + 2 * NC + c) * pb, rw[5][k]);
                        }
    #pragma unroll
                        for (int t4 = 0; t4 < K; t4 += 4) {
                            const int s = s0 + t4;                         // four steps = four adjacent columns
                            if (both && s == first) named_bar_sync(1 + c, 64);
                            const bool acc = touched || (both && s >= first);
                            const int j0 = REV ? W - 4 - s : s;              // lowest column of the group
                            float yv[P][4];
                            if (acc && active) {
    #pragma unroll
                                for (int k = 0; k < P; ++k) ldf<4>(Yc + (size_t)(k * HP + lane) * pitch + j0, yv[k]);
                            } else {
    #pragma unroll
                                for (int k = 0; k < P; ++k) yv[k][0] = yv[k][1] = yv[k][2] = yv[k][3] = 0.f;
                            }
    #pragma unroll
                            for (int tt = 0; tt < 4; ++tt) {
                                constexpr int dummy = 0; (void)dummy; const int e = REV ? K - 1 - (t4 + tt) : t4 + tt;   // element inside the 16-byte chunk
                                float a0[P], a1[P], a2[P], al[P], au[P];
    #pragma unroll
                                for (int k = 0; k < P; ++k) {
                                    a0[k] = line_elem<ST>(rw[0][k], e);
                                    a1[k] = line_elem<ST>(rw[1][k], e);
                                    a2[k] = line_elem<ST>(rw[2][k], e);
                                    al[k] = line_elem<ST>(rw[3][k], e) * line_elem<ST>(rw[5][k], e);
                                    au[k] = line_elem<ST>(rw[4][k], e);
                                }
                                if (first_lane) a0[0] = 0.f;
                                if (last_lane) a2[P - 1] = 0.f;
                                line_step<ST, P>(h, a0, a1, a2, al, first_lane, last_lane);
                                const int ye = REV ? 3 - tt : tt;
    #pragma unroll
                                for (int k = 0; k < P; ++k) yv[k][ye] = fmaf(au[k], h[k], yv[k][ye]);
                            }
                            if (active) {
    #pragma unroll
                                for (int k = 0; k < P; ++k) stf<4>(Yc + (size_t)(k * HP + lane) * pitch + j0, yv[k]);
                            }
                        }
                    }
}

template <typename ST, int NC, int P>
__global__ void __launch_bounds__((2 + 2 * NC) * 32, 1)
line_fwd_kernel(const __grid_constant__ CUtensorMap mxv, const __grid_constant__ CUtensorMap mwv,
                const __grid_constant__ CUtensorMap mlv, const __grid_constant__ CUtensorMap muv,
                const __grid_constant__ CUtensorMap mxh, const __grid_constant__ CUtensorMap mwh,
                const __grid_constant__ CUtensorMap mlh, const __grid_constant__ CUtensorMap muh,
                const LineFwdParams prm) {
    constexpr int ES = sizeof(ST);
    constexpr int K = 16 / ES;                     // scan steps per 16-byte column chunk
    constexpr int S = kLineSteps;
    constexpr int NCH = S / K;                     // column chunks per horizontal stage
    constexpr int NS = kLineStages;
    constexpr int NPL = 3 + 3 * NC;                // operand planes per stage: taps, lambda, u, x

    extern __shared__ __align__(128) unsigned char smem[];
    const int H = prm.H, W = prm.W;
    const size_t y_bytes = (size_t)NC * H * prm.pitch * 4;
    float* const Y = reinterpret_cast<float*>(smem);
    unsigned char* const ring = smem + (y_bytes + 127) / 128 * 128;
    const uint32_t stage_bytes = NPL * prm.pb_bytes;
    uint64_t* const bars = reinterpret_cast<uint64_t*>(ring + (size_t)2 * NS * stage_bytes);
    uint64_t* const full = bars;                   // [2][NS]
    uint64_t* const empty = bars + 2 * NS;         // [2][NS]

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
        mbar_init_fence();
    }
    __syncthreads();

    const int nblk_v = (H + S - 1) / S, nblk_h = (W + S - 1) / S;

    if (warp < 2) {
        // ------------------------------------------------------------------ producer of direction pair member d
        const int d = warp;
        int it = 0;
        for (int ph = 0; ph < 2; ++ph) {
            const int dir = 2 * ph + d;
            if (!(mask >> dir & 1u)) continue;
            const int q = prm.slab[dir];
            // plane index of this lane's operand inside its tensor
            int plane = 0;
            const CUtensorMap* map = nullptr;
            if (lane < 3) {
                plane = ((q * prm.B + b) * prm.G + g) * 3 + lane;
                map = ph ? &mwh : &mwv;
            } else if (lane < 3 + NC) {
                plane = (q * prm.B + b) * prm.C + c0 + (lane - 3);
                map = ph ? &mlh : &mlv;
            } else if (lane < 3 + 2 * NC) {
                plane = (q * prm.B + b) * prm.C + c0 + (lane - 3 - NC);
                map = ph ? &muh : &muv;
            } else if (lane < NPL) {
                plane = b * prm.C + c0 + (lane - 3 - 2 * NC);
                map = ph ? &mxh : &mxv;
            }
            const int nblk = ph ? nblk_h : nblk_v;
            const int Ls = ph ? W : H;
            for (int blk = 0; blk < nblk; ++blk, ++it) {
                const int stg = it % NS;
                if (it >= NS) mbar_wait(&empty[d * NS + stg], ((it / NS) - 1) & 1);
                uint64_t* fb = &full[d * NS + stg];
                if (lane == 0) mbar_arrive_expect_tx(fb, (uint32_t)(NPL * S * ES) * (uint32_t)(ph ? H : W));
                __syncwarp();
                if (lane < NPL) {
                    unsigned char* dst = ring + (size_t)(d * NS + stg) * stage_bytes + (size_t)lane * prm.pb_bytes;
                    const int s0 = d ? Ls - (blk + 1) * S : blk * S;      // first row / column of the stage (may be < 0)
                    if (ph == 0) tma_load_3d(dst, map, 0, s0, plane, fb);
                    else tma_load_5d(dst, map, 0, 0, 0, s0 / K, plane, fb);
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- scan line of channel c, pair member d
    const int c = (warp - 2) >> 1, d = (warp - 2) & 1;
    const int ch = c0 + c;
    float* const Yc = Y + (size_t)c * H * prm.pitch;
    const int pitch = prm.pitch;
    const uint32_t pb = prm.pb_bytes;
    int it = 0;
    bool touched = false;                         // the accumulator plane holds data

    // ---- T->B (d = 0) / B->T (d = 1): lanes own columns
    {
        const int dir = d;
        const bool present = mask >> dir & 1u;
        const bool both = (mask & 3u) == 3u;
        if (present) {
            const int q = prm.slab[dir];
            const bool active = lane < prm.WP;
            const int lp = active ? lane : 0;
            const bool first_lane = lane == 0, last_lane = lane == prm.WP - 1;
            float h[P];
#pragma unroll
            for (int k = 0; k < P; ++k) h[k] = 0.f;
            if (prm.h0 && active) {
                const ST* hp = reinterpret_cast<const ST*>(prm.h0) +
                               ((size_t)(q * prm.B + b) * prm.C + ch) * (H > W ? H : W) + P * lane;
#pragma unroll
                for (int k = 0; k < P; ++k) h[k] = ld_f(hp + k);
            }
            const int Hh = (H + 1) / 2;
            const int first = both ? (d == 0 ? Hh : H - Hh) : H;      // steps on the half this direction touches first
            for (int s = 0; s < H; ++s) {
                const int blk = s / S, r = s % S;
                const int cur = it + blk, stg = cur % NS;
                if (both && s == first) named_bar_sync(1 + c, 64);
                if (r == 0) mbar_wait(&full[d * NS + stg], (cur / NS) & 1);
                const int i = d ? H - 1 - s : s;
                const int rl = d ? S - 1 - r : r;
                const ST* row = reinterpret_cast<const ST*>(ring + (size_t)(d * NS + stg) * stage_bytes) + rl * W + P * lp;
                const uint32_t pbe = pb / ES;
                float w0[P], w1[P], w2[P], la[P], uu[P], xx[P], lx[P];
                line_ld<ST, P>(row, w0);
                line_ld<ST, P>(row + pbe, w1);
                line_ld<ST, P>(row + 2 * pbe, w2);
                line_ld<ST, P>(row + (3 + c) * pbe, la);
                line_ld<ST, P>(row + (3 + NC + c) * pbe, uu);
                line_ld<ST, P>(row + (3 + 2 * NC + c) * pbe, xx);
                if (first_lane) w0[0] = 0.f;
                if (last_lane) w2[P - 1] = 0.f;
#pragma unroll
                for (int k = 0; k < P; ++k) lx[k] = la[k] * xx[k];
                line_step<ST, P>(h, w0, w1, w2, lx, first_lane, last_lane);
                if (active) {
                    float* yp = Yc + (size_t)line_phys_row<P>(i, prm.HP) * pitch + P * lane;
                    float yv[P];
                    if (both && s >= first) {
                        ldf<P>(yp, yv);
#pragma unroll
                        for (int k = 0; k < P; ++k) yv[k] = fmaf(uu[k], h[k], yv[k]);
                    } else {
#pragma unroll
                        for (int k = 0; k < P; ++k) yv[k] = uu[k] * h[k];
                    }
                    stf<P>(yp, yv);
                }
                if (r == S - 1 || s == H - 1) {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[d * NS + stg]);
                }
            }
            if (both && first >= H) named_bar_sync(1 + c, 64);
            it += nblk_v;
        }
        touched = (mask & 3u) != 0;
        named_bar_sync(1 + c, 64);                 // the vertical sums of this channel are complete
    }

    // ---- L->R (d = 0) / R->L (d = 1): lanes own rows, a stage holds NCH 16-byte column chunks
    {
        const int dir = 2 + d;
        const bool present = mask >> dir & 1u;
        const bool both = (mask & 12u) == 12u;
        if (present) {
            const int q = prm.slab[dir];
            const int HP = prm.HP;
            const bool active = lane < HP;
            const int lp = active ? lane : 0;
            const bool first_lane = lane == 0, last_lane = lane == HP - 1;
            float h[P];
#pragma unroll
            for (int k = 0; k < P; ++k) h[k] = 0.f;
            if (prm.h0 && active) {
                const ST* hp = reinterpret_cast<const ST*>(prm.h0) +
                               ((size_t)(q * prm.B + b) * prm.C + ch) * (H > W ? H : W) + P * lane;
#pragma unroll
                for (int k = 0; k < P; ++k) h[k] = ld_f(hp + k);
            }
            const int Wh = (W / 2 + 3) / 4 * 4;                        // swap point, a multiple of 4 columns
            const int first = both ? (d == 0 ? Wh : W - Wh) : W;
            for (int blk = 0; blk < nblk_h; ++blk) {
                const int cur = it + blk, stg = cur % NS;
                mbar_wait(&full[d * NS + stg], (cur / NS) & 1);
                const unsigned char* sb = ring + (size_t)(d * NS + stg) * stage_bytes;
                if (d) line_fwd_hstage<ST, NC, P, true>(sb, blk, H, W, HP, lp, lane, active, first_lane, last_lane, c, pb,
                                                         pitch, Yc, both, first, touched, h);
                else line_fwd_hstage<ST, NC, P, false>(sb, blk, H, W, HP, lp, lane, active, first_lane, last_lane, c, pb,
                                                        pitch, Yc, both, first, touched, h);
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[d * NS + stg]);
            }
            if (both && first >= W) named_bar_sync(1 + c, 64);
            it += nblk_h;
        }
        named_bar_sync(1 + c, 64);                 // the plane of this channel is complete
    }

    // ---- the finished plane leaves: one RNE per element, 16-byte stores
    {
        ST* yg = reinterpret_cast<ST*>(prm.y) + ((size_t)b * prm.C + ch) * H * W;
        const int wk = W / K, n16 = H * wk;
        for (int qd = d * 32 + lane; qd < n16; qd += 64) {
            const int i = qd / wk, jc = qd - i * wk;
            float f[K];
            ldf<K>(Yc + (size_t)line_phys_row<P>(i, prm.HP) * pitch + jc * K, f);
            uint32_t r[4];
            Store<ST>::template pack<16>(f, r);
            *reinterpret_cast<uint4*>(yg + (size_t)i * W + jc * K) = make_uint4(r[0], r[1], r[2], r[3]);
        }
    }
}

}  // namespace

// ---- host side ---------------------------------------------------------------------------------------------------
template <typename ST, int NC, int P>
static int line_fwd_run(const FwdArgs<ST>& a, cudaStream_t st) {
    constexpr int ES = sizeof(ST);
    constexpr int K = 16 / ES;
    constexpr int S = kLineSteps;
    const Shape& sh = a.sh;
    const int H = sh.H, W = sh.W, L = sh.Lmax();
    LineFwdParams prm{};
    prm.B = sh.B; prm.C = sh.C; prm.H = H; prm.W = W; prm.G = sh.G; prm.cg = sh.cg();
    prm.mask = sh.mask;
    int q = 0;
    for (int d = 0; d < 4; ++d) prm.slab[d] = (sh.mask >> d & 1u) ? q++ : -1;
    prm.HP = H / P; prm.WP = W / P;
    prm.pitch = line_pitch(W);
    prm.pb_bytes = (uint32_t)((S * L * ES + 127) / 128 * 128);   // TMA destinations are 128-byte aligned
    prm.h0 = a.h0; prm.y = a.y;
    const size_t y_bytes = ((size_t)NC * H * prm.pitch * 4 + 127) / 128 * 128;
    const size_t smem = y_bytes + (size_t)2 * kLineStages * (3 + 3 * NC) * prm.pb_bytes + 4 * kLineStages * 8;
    if (smem > (size_t)kMaxSmemOptin) return GSPN_EUNSUPPORTED;

    const int D = sh.D();
    struct Src { const void* p; uint64_t planes; };
    const Src src[4] = {{a.x, (uint64_t)sh.B * sh.C}, {a.w3, (uint64_t)D * sh.B * sh.G * 3},
                        {a.lam, (uint64_t)D * sh.B * sh.C}, {a.u, (uint64_t)D * sh.B * sh.C}};
    CUtensorMap m[8];
    const uint64_t row_b = (uint64_t)W * ES, plane_b = (uint64_t)H * W * ES;
    for (int t = 0; t < 4; ++t) {
        const uint64_t dv[3] = {(uint64_t)W, (uint64_t)H, src[t].planes};
        const uint64_t sv[2] = {row_b, plane_b};
        const uint32_t bv[3] = {(uint32_t)W, (uint32_t)S, 1u};
        if (!encode_tensor_map(&m[t], ES, const_cast<void*>(src[t].p), 3, dv, sv, bv)) return GSPN_ECUDA;
        // [16 B][row / P][row % P][column chunk][plane]
        const uint64_t dh[5] = {(uint64_t)K, (uint64_t)(H / P), (uint64_t)P, (uint64_t)(W / K), src[t].planes};
        const uint64_t shh[4] = {(uint64_t)P * row_b, row_b, 16u, plane_b};
        const uint32_t bh[5] = {(uint32_t)K, (uint32_t)(H / P), (uint32_t)P, (uint32_t)(S / K), 1u};
        if (!encode_tensor_map(&m[4 + t], ES, const_cast<void*>(src[t].p), 5, dh, shh, bh)) return GSPN_ECUDA;
    }
    auto kern = line_fwd_kernel<ST, NC, P>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("line fwd: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    const int items = sh.B * sh.G * (sh.cg() / NC);
    kern<<<items, (2 + 2 * NC) * 32, smem, st>>>(m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], prm);
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
    if (W % 4 != 0) { set_error("line fwd: W = %d is not a multiple of 4", W); return GSPN_EUNSUPPORTED; }
    int P = 0;
    for (int p : {1, 2, 4}) if (H % p == 0 && W % p == 0 && sh.Lmax() <= 32 * p) { P = p; break; }
    if (!P) { set_error("line fwd: %dx%d does not fit one warp per line with 1, 2 or 4 positions per lane", H, W); return GSPN_EUNSUPPORTED; }
    int rc = P == 1 ? line_fwd_nc<ST, 1>(a, st) : P == 2 ? line_fwd_nc<ST, 2>(a, st) : line_fwd_nc<ST, 4>(a, st);
    if (rc == GSPN_EUNSUPPORTED) set_error("line fwd: the accumulator plane and the operand ring of %dx%d exceed shared memory", H, W);
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "line_fwd"; }
    return rc;
}

template int line_fwd_launch<float>(const FwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int line_fwd_launch<__nv_bfloat16>(const FwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
