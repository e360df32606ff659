// gspn_fused_fwd.cu -- the fused forward scan of libgspn: all directions of
// dir_mask and their merge in ONE launch, x/lambda/u/w3 streamed once through shared memory by TMA,
// the hidden state h in registers for the whole recurrence (Eq. 1), y = sum_d u_d*h_d
// (Eq. 2 / Eq. 9) accumulated on chip in fp32 and written once.
//
// "Tile" variant (rows 16-byte aligned: W*sizeof(ST) % 16 == 0).  One CTA owns `cpc` channels of one
// (b, group) unit.  Every direction has its own ring of TMA stages, each stage holding the operands
// of the next K = 16/sizeof(ST) scan steps of all cpc channels:
//     vertical   (T->B, B->T): K image rows   [K][W]        per plane  (3-D tensor map  W,H,plane)
//     horizontal (L->R, R->L): K image columns [R][L][16 B] per plane  (4-D tensor map  W,L,R,plane:
//                              row i = R*l + k is stored at [k][l], so lane l reads its R rows with
//                              conflict-free 16-byte loads -- the transposed-tile path)
// A warp runs one chain = (direction, channel): a lane holds CPT = CPTB/sizeof(ST) adjacent cross
// positions (vertical) or R adjacent rows (horizontal) of h, neighbours inside a lane are registers
// and across lanes one shuffle each way per step.  Four producer warps (one elected lane each) feed
// the four rings.  The two vertical chains of a channel share the fp32 plane Yv, the two horizontal
// ones Yh: the chain that reaches a line first stores, the second one adds; one mbarrier hand-shake
// per pair at half time separates the two phases, so no atomics are needed.  After the last step the
// CTA adds Yv + Yh, rounds once (RNE) and writes y with 16-byte stores.
#include <initializer_list>
#include <type_traits>

#include "gspn_fused.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

struct FwdTileParams {
    Shape sh;
    int cpc;            // channels per CTA
    int ns;             // ring stages per direction
    int Wp;             // row pitch of Yh in floats
    int L;              // lanes of a horizontal chain (H / R)
    int nst[4];         // stages per direction, 0 = direction not in dir_mask
    int q[4];           // slab index of each direction
    uint32_t off_yv, off_yh;        // byte offsets inside dynamic shared memory
    uint32_t off_ring[4];
    uint32_t stage_bytes[2];        // [0] vertical, [1] horizontal ring stage (128-byte multiples)
    uint32_t boxw_bytes[2], boxc_bytes[2];   // slot of the w3 box / of a cpc-plane box (128-byte multiples)
    uint32_t tx_bytes[2];           // bytes TMA delivers per stage
    void* y;
    const void* h0;
};

constexpr int kMaxStages = 8;
constexpr int kBarBytes = 1024;     // full[4][8], empty[4][8], pair[2][8]

// dir 0 T->B, 1 B->T, 2 L->R, 3 R->L
template <typename ST, int CPTB, int R>
__global__ void __launch_bounds__((R >= 4 || CPTB == 16) ? 384 : 640, 1)
fwd_tile_kernel(const __grid_constant__ CUtensorMap mxv, const __grid_constant__ CUtensorMap mlv,
                const __grid_constant__ CUtensorMap muv, const __grid_constant__ CUtensorMap mwv,
                const __grid_constant__ CUtensorMap mxh, const __grid_constant__ CUtensorMap mlh,
                const __grid_constant__ CUtensorMap muh, const __grid_constant__ CUtensorMap mwh,
                const FwdTileParams p) {
    constexpr int ES = Store<ST>::ES;
    constexpr int K = 16 / ES;              // scan steps per stage
    constexpr int CPT = CPTB / ES;          // cross positions per lane, vertical chains
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);            // [4][kMaxStages]
    uint64_t* empty = full + 4 * kMaxStages;                       // [4][kMaxStages]
    uint64_t* pairb = empty + 4 * kMaxStages;                      // [2][8]
    float* Yv = reinterpret_cast<float*>(smem + p.off_yv);
    float* Yh = reinterpret_cast<float*>(smem + p.off_yh);

    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, cpc = p.cpc, NS = p.ns;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int slices = sh.cg() / cpc;
    const int item = blockIdx.x;
    const int b = item / (sh.G * slices);
    const int g = (item / slices) % sh.G;
    const int c0 = g * sh.cg() + (item % slices) * cpc;           // first channel of this CTA
    const bool vact = (sh.mask & 3u) != 0, hact = (sh.mask & 12u) != 0;

    if (threadIdx.x == 0) {
        for (int d = 0; d < 4; ++d)
            for (int s = 0; s < NS; ++s) { mbar_init(&full[d * kMaxStages + s], 1); mbar_init(&empty[d * kMaxStages + s], cpc); }
        for (int t = 0; t < 16; ++t) mbar_init(&pairb[t], 2);
        mbar_init_fence();
    }
    __syncthreads();

    if (warp < 4) {
        // ---------------- producer of direction `warp` ------------------------------------------
        const int d = warp;
        if (lane == 0 && p.nst[d] > 0) {
            const int vh = d >> 1;
            const CUtensorMap* mw = vh ? &mwh : &mwv;
            const CUtensorMap* ml = vh ? &mlh : &mlv;
            const CUtensorMap* mu = vh ? &muh : &muv;
            const CUtensorMap* mx = vh ? &mxh : &mxv;
            tma_prefetch_desc(mw); tma_prefetch_desc(ml); tma_prefetch_desc(mu); tma_prefetch_desc(mx);
            const int pw = ((p.q[d] * sh.B + b) * sh.G + g) * 3;
            const int pc = (p.q[d] * sh.B + b) * sh.C + c0;
            const int px = b * sh.C + c0;
            uint8_t* ring = smem + p.off_ring[d];
            const int Ls = vh ? W : H;
            for (int t = 0; t < p.nst[d]; ++t) {
                const int slot = t % NS, it = t / NS;
                mbar_wait(&empty[d * kMaxStages + slot], (it & 1) ^ 1);
                uint64_t* fb = &full[d * kMaxStages + slot];
                mbar_arrive_expect_tx(fb, p.tx_bytes[vh]);
                uint8_t* dst = ring + (size_t)slot * p.stage_bytes[vh];
                const int s0 = (d & 1) ? Ls - K * (t + 1) : K * t;    // first line of the stage (may be < 0: zero filled)
                if (!vh) {
                    tma_load_3d(dst, mw, 0, s0, pw, fb);
                    tma_load_3d(dst + p.boxw_bytes[0], ml, 0, s0, pc, fb);
                    tma_load_3d(dst + p.boxw_bytes[0] + p.boxc_bytes[0], mu, 0, s0, pc, fb);
                    tma_load_3d(dst + p.boxw_bytes[0] + 2 * p.boxc_bytes[0], mx, 0, s0, px, fb);
                } else {
                    tma_load_4d(dst, mw, s0, 0, 0, pw, fb);
                    tma_load_4d(dst + p.boxw_bytes[1], ml, s0, 0, 0, pc, fb);
                    tma_load_4d(dst + p.boxw_bytes[1] + p.boxc_bytes[1], mu, s0, 0, 0, pc, fb);
                    tma_load_4d(dst + p.boxw_bytes[1] + 2 * p.boxc_bytes[1], mx, s0, 0, 0, px, fb);
                }
            }
        }
    } else {
        // ---------------- one chain per warp: (direction d, channel ch) -------------------------
        const int cw = warp - 4;
        const int d = cw / cpc, ch = cw % cpc;
        if (d < 4 && p.nst[d] > 0) {
            const int vh = d >> 1;
            const bool rev = d & 1;
            const bool partner = (sh.mask >> (d ^ 1)) & 1u;
            uint64_t* pb = &pairb[vh * 8 + ch];
            const uint8_t* ring = smem + p.off_ring[d];
            const size_t h0off = ((size_t)(p.q[d] * sh.B + b) * sh.C + c0 + ch) * sh.Lmax();
            const ST* h0p = p.h0 ? reinterpret_cast<const ST*>(p.h0) + h0off : nullptr;
            bool synced = false;
            if (!vh) {
                // ======== vertical chain: lane holds columns [CPT*lane, CPT*lane + CPT) =========
                const int LPC = W / CPT;
                const bool act = lane < LPC;
                const uint32_t TP = (uint32_t)K * W * ES;                 // bytes of one plane tile
                float h[CPT];
#pragma unroll
                for (int e = 0; e < CPT; ++e) h[e] = (h0p && act) ? ld_f(h0p + CPT * lane + e) : 0.f;
                const int rstar = (H - 1) / 2;
                const int sync_step = rev ? H - 1 - rstar : rstar + 1;    // first step that adds instead of stores
                float* yplane = Yv + (size_t)ch * H * W + CPT * lane;
                const uint32_t lane_off = (uint32_t)lane * CPTB;
                for (int t = 0; t < p.nst[d]; ++t) {
                    const int slot = t % NS, it = t / NS;
                    mbar_wait(&full[d * kMaxStages + slot], it & 1);
                    const uint8_t* tile = ring + (size_t)slot * p.stage_bytes[0];
                    const uint8_t* tl = tile + p.boxw_bytes[0] + (size_t)ch * TP;
                    const uint8_t* tu = tl + p.boxc_bytes[0];
                    const uint8_t* tx = tu + p.boxc_bytes[0];
#pragma unroll
                    for (int j = 0; j < K; ++j) {
                        const int s = t * K + j;
                        if (s >= H) break;
                        if (partner && s == sync_step) {
                            __syncwarp();
                            if (lane == 0) mbar_arrive(pb);
                            mbar_wait(pb, 0);
                            synced = true;
                        }
                        const int rr = rev ? K - 1 - j : j;
                        const int i = rev ? H - 1 - s : s;
                        const uint32_t off = (uint32_t)rr * W * ES + lane_off;
                        float w0[CPT], w1[CPT], w2[CPT], lm[CPT], uu[CPT], xx[CPT];
                        if (act) {
                            uint32_t r[CPTB / 4];
                            lds_vec<CPTB>(tile + off, r);          Store<ST>::template unpack<CPTB>(r, w0);
                            lds_vec<CPTB>(tile + TP + off, r);     Store<ST>::template unpack<CPTB>(r, w1);
                            lds_vec<CPTB>(tile + 2 * TP + off, r); Store<ST>::template unpack<CPTB>(r, w2);
                            lds_vec<CPTB>(tl + off, r);            Store<ST>::template unpack<CPTB>(r, lm);
                            lds_vec<CPTB>(tu + off, r);            Store<ST>::template unpack<CPTB>(r, uu);
                            lds_vec<CPTB>(tx + off, r);            Store<ST>::template unpack<CPTB>(r, xx);
                        } else {
#pragma unroll
                            for (int e = 0; e < CPT; ++e) { w0[e] = w1[e] = w2[e] = lm[e] = uu[e] = xx[e] = 0.f; }
                        }
                        float hl = __shfl_up_sync(0xffffffffu, h[CPT - 1], 1);
                        float hr = __shfl_down_sync(0xffffffffu, h[0], 1);
                        if (lane == 0) { hl = 0.f; w0[0] = 0.f; }                  // out-of-grid tap: never used
                        if (lane == LPC - 1) { hr = 0.f; w2[CPT - 1] = 0.f; }
                        float hn[CPT], yv[CPT];
#pragma unroll
                        for (int e = 0; e < CPT; ++e) {
                            const float left = e ? h[e - 1] : hl;
                            const float right = e < CPT - 1 ? h[e + 1] : hr;
                            float acc = lm[e] * xx[e];
                            acc = fmaf(w0[e], left, acc);
                            acc = fmaf(w1[e], h[e], acc);
                            acc = fmaf(w2[e], right, acc);
                            hn[e] = acc;
                            yv[e] = uu[e] * acc;
                        }
                        if (act) {
                            float* yr = yplane + (size_t)i * W;
                            if (partner && s >= sync_step) {
                                float old[CPT];
                                ldf<CPT>(yr, old);
#pragma unroll
                                for (int e = 0; e < CPT; ++e) yv[e] += old[e];
                            }
                            stf<CPT>(yr, yv);
                        }
#pragma unroll
                        for (int e = 0; e < CPT; ++e) h[e] = hn[e];
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[d * kMaxStages + slot]);
                }
            } else {
                // ======== horizontal chain: lane holds rows [R*lane, R*lane + R) ================
                const int L = p.L;
                const bool act = lane < L;
                const uint32_t TP = (uint32_t)H * 16;                     // bytes of one plane tile [R][L][16]
                float h[R];
#pragma unroll
                for (int k = 0; k < R; ++k) h[k] = (h0p && act) ? ld_f(h0p + R * lane + k) : 0.f;
                const int NC = p.nst[d];
                const int ncs = (NC + 1) / 2;
                const int sync_stage = rev ? NC - ncs : ncs;              // first stage that adds instead of stores
                const int Wp = p.Wp;
                float* yplane = Yh + (size_t)ch * H * Wp;
                for (int t = 0; t < NC; ++t) {
                    const int slot = t % NS, it = t / NS;
                    mbar_wait(&full[d * kMaxStages + slot], it & 1);
                    const uint8_t* tile = ring + (size_t)slot * p.stage_bytes[1];
                    const uint8_t* tl = tile + p.boxw_bytes[1] + (size_t)ch * TP;
                    const uint8_t* tu = tl + p.boxc_bytes[1];
                    const uint8_t* tx = tu + p.boxc_bytes[1];
                    uint32_t rw0[R][4], rw1[R][4], rw2[R][4], rl[R][4], ru[R][4], rx[R][4];
#pragma unroll
                    for (int k = 0; k < R; ++k) {
                        const uint32_t off = (uint32_t)(k * L + lane) * 16;
                        if (act) {
                            lds_vec<16>(tile + off, rw0[k]);
                            lds_vec<16>(tile + TP + off, rw1[k]);
                            lds_vec<16>(tile + 2 * TP + off, rw2[k]);
                            lds_vec<16>(tl + off, rl[k]);
                            lds_vec<16>(tu + off, ru[k]);
                            lds_vec<16>(tx + off, rx[k]);
                        } else {
#pragma unroll
                            for (int v = 0; v < 4; ++v) rw0[k][v] = rw1[k][v] = rw2[k][v] = rl[k][v] = ru[k][v] = rx[k][v] = 0u;
                        }
                    }
                    float yh[R][K];
                    const bool first = lane == 0, last = lane == L - 1;
                    auto steps = [&](auto revc) {
                        constexpr bool REV = decltype(revc)::value;
#pragma unroll
                        for (int j = 0; j < K; ++j) {
                            constexpr int dummy = 0; (void)dummy;
                            const int e = REV ? K - 1 - j : j;            // element of the 16-byte chunk (compile time)
                            auto pick = [&](const uint32_t (&r)[4]) -> float {
                                if constexpr (ES == 4) return __uint_as_float(r[e]);
                                else return __uint_as_float((e & 1) ? (r[e >> 1] & 0xffff0000u) : (r[e >> 1] << 16));
                            };
                            float up = __shfl_up_sync(0xffffffffu, h[R - 1], 1);
                            float dn = __shfl_down_sync(0xffffffffu, h[0], 1);
                            if (first) up = 0.f;
                            if (last) dn = 0.f;
                            float hn[R];
#pragma unroll
                            for (int k = 0; k < R; ++k) {
                                const float a = k ? h[k - 1] : up;
                                const float c = k < R - 1 ? h[k + 1] : dn;
                                float t0 = pick(rw0[k]), t2 = pick(rw2[k]);
                                if (k == 0 && first) t0 = 0.f;             // out-of-grid tap: never used
                                if (k == R - 1 && last) t2 = 0.f;
                                float acc = pick(rl[k]) * pick(rx[k]);
                                acc = fmaf(t0, a, acc);
                                acc = fmaf(pick(rw1[k]), h[k], acc);
                                acc = fmaf(t2, c, acc);
                                hn[k] = acc;
                                yh[k][e] = pick(ru[k]) * acc;
                            }
#pragma unroll
                            for (int k = 0; k < R; ++k) h[k] = hn[k];
                        }
                    };
                    if (rev) steps(std::true_type{}); else steps(std::false_type{});
                    if (partner && t == sync_stage) {
                        __syncwarp();
                        if (lane == 0) mbar_arrive(pb);
                        mbar_wait(pb, 0);
                        synced = true;
                    }
                    if (act) {
                        const int col0 = rev ? W - K * (t + 1) : K * t;
                        const bool rmw = partner && t >= sync_stage;
#pragma unroll
                        for (int k = 0; k < R; ++k) {
                            float* yr = yplane + (size_t)(k * L + lane) * Wp + col0;
                            if (rmw) {
                                float old[K];
                                ldf<K>(yr, old);
#pragma unroll
                                for (int e = 0; e < K; ++e) yh[k][e] += old[e];
                            }
                            stf<K>(yr, yh[k]);
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[d * kMaxStages + slot]);
                }
            }
            if (partner && !synced) {          // never reached an adding step: still release the partner
                __syncwarp();
                if (lane == 0) mbar_arrive(pb);
            }
        }
    }
    __syncthreads();

    // ---------------- merge: y = Yv + Yh, one RNE, 16-byte stores --------------------------------
    {
        const int nvr = W / K;                                   // 16-byte vectors per row
        const int total = cpc * H * nvr;
        ST* yg = reinterpret_cast<ST*>(p.y) + ((size_t)b * sh.C + c0) * H * W;
        const int L = p.L;
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            const int v = idx % nvr;
            const int i = (idx / nvr) % H;
            const int ch = idx / (nvr * H);
            float acc[K];
#pragma unroll
            for (int e = 0; e < K; ++e) acc[e] = 0.f;
            if (vact) {
                float t[K];
                ldf<K>(Yv + ((size_t)ch * H + i) * W + v * K, t);
#pragma unroll
                for (int e = 0; e < K; ++e) acc[e] += t[e];
            }
            if (hact) {
                float t[K];
                const int slot = (i % R) * L + i / R;
                ldf<K>(Yh + ((size_t)ch * H + slot) * p.Wp + v * K, t);
#pragma unroll
                for (int e = 0; e < K; ++e) acc[e] += t[e];
            }
            uint32_t r[4];
            Store<ST>::template pack<16>(acc, r);
            *reinterpret_cast<uint4*>(yg + ((size_t)ch * H + i) * W + v * K) = make_uint4(r[0], r[1], r[2], r[3]);
        }
    }
}

// ---- host side -----------------------------------------------------------------------------------
static uint32_t rb128(size_t v) { return (uint32_t)((v + 127) / 128 * 128); }

struct TilePlan {
    int cptb, R, cpc, ns, Wp, L;
    size_t smem;
    FwdTileParams prm;
};

// smem use of the tile variant for (cpc, ns); fills the offsets of prm
static size_t tile_layout(const Shape& sh, int es, int cpc, int ns, int Wp, FwdTileParams* prm) {
    const int K = 16 / es;
    const bool vact = sh.mask & 3u, hact = sh.mask & 12u;
    size_t off = kBarBytes;
    prm->off_yv = (uint32_t)off;
    if (vact) off += (size_t)cpc * sh.H * sh.W * 4;
    off = (off + 127) / 128 * 128;
    prm->off_yh = (uint32_t)off;
    if (hact) off += (size_t)cpc * sh.H * Wp * 4;
    off = (off + 1023) / 1024 * 1024;
    const size_t tp[2] = {(size_t)K * sh.W * es, (size_t)sh.H * 16};
    for (int vh = 0; vh < 2; ++vh) {
        prm->boxw_bytes[vh] = rb128(3 * tp[vh]);
        prm->boxc_bytes[vh] = rb128(cpc * tp[vh]);
        prm->stage_bytes[vh] = prm->boxw_bytes[vh] + 3 * prm->boxc_bytes[vh];
        prm->tx_bytes[vh] = (uint32_t)(3 * tp[vh] + 3 * cpc * tp[vh]);
    }
    for (int d = 0; d < 4; ++d) {
        prm->off_ring[d] = (uint32_t)off;
        if (sh.mask >> d & 1u) off += (size_t)ns * prm->stage_bytes[d >> 1];
    }
    return off;
}

template <typename ST, int CPTB, int R>
static int launch_tile(const FwdArgs<ST>& a, const TilePlan& pl, cudaStream_t st) {
    constexpr int ES = sizeof(ST);
    constexpr int K = 16 / ES;
    const Shape& sh = a.sh;
    const int H = sh.H, W = sh.W, D = sh.D(), cpc = pl.cpc;
    CUtensorMap m[8];
    const uint64_t plane_b = (uint64_t)H * W * ES, row_b = (uint64_t)W * ES;
    struct Src { const void* p; uint64_t planes; uint32_t np; } src[4] = {
        {a.x, (uint64_t)sh.B * sh.C, (uint32_t)cpc},
        {a.lam, (uint64_t)D * sh.B * sh.C, (uint32_t)cpc},
        {a.u, (uint64_t)D * sh.B * sh.C, (uint32_t)cpc},
        {a.w3, (uint64_t)D * sh.B * sh.G * 3, 3u}};
    for (int t = 0; t < 4; ++t) {
        const uint64_t dv[3] = {(uint64_t)W, (uint64_t)H, src[t].planes};
        const uint64_t sv[2] = {row_b, plane_b};
        const uint32_t bv[3] = {(uint32_t)W, (uint32_t)K, src[t].np};
        if (!encode_tensor_map(&m[t], ES, const_cast<void*>(src[t].p), 3, dv, sv, bv)) return GSPN_ECUDA;
        const uint64_t dh[4] = {(uint64_t)W, (uint64_t)pl.L, (uint64_t)R, src[t].planes};
        const uint64_t shh[3] = {(uint64_t)R * row_b, row_b, plane_b};
        const uint32_t bh[4] = {(uint32_t)K, (uint32_t)pl.L, (uint32_t)R, src[t].np};
        if (!encode_tensor_map(&m[4 + t], ES, const_cast<void*>(src[t].p), 4, dh, shh, bh)) return GSPN_ECUDA;
    }
    auto kern = fwd_tile_kernel<ST, CPTB, R>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("fused fwd: cudaFuncSetAttribute(%zu B): %s", pl.smem, cudaGetErrorString(e)); return GSPN_ECUDA; }
    const int items = sh.B * sh.G * (sh.cg() / cpc);
    const int threads = (4 + 4 * cpc) * 32;
    GSPN_LAUNCH(kern, items, threads, pl.smem, st, m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], pl.prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("fused fwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int fused_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    constexpr int K = 16 / ES;
    const Shape& sh = a.sh;
    const int H = sh.H, W = sh.W;
    if ((W * ES) % 16 != 0) { set_error("fused fwd (tile): rows of %d B are not 16-byte aligned", W * ES); return GSPN_EUNSUPPORTED; }
    if (W > 256) { set_error("fused fwd (tile): W = %d > 256", W); return GSPN_EUNSUPPORTED; }
    TilePlan pl{};
    pl.cptb = W * ES <= 128 ? 4 : (W * ES <= 256 ? 8 : 16);
    if (W * ES / pl.cptb > 32) { set_error("fused fwd (tile): rows of %d B exceed one warp", W * ES); return GSPN_EUNSUPPORTED; }
    pl.R = 0;
    for (int r : {1, 2, 4}) if (H % r == 0 && H / r <= 32) { pl.R = r; break; }
    if (!pl.R) { set_error("fused fwd (tile): H = %d has no row blocking R in {1,2,4} with H/R <= 32", H); return GSPN_EUNSUPPORTED; }
    pl.L = H / pl.R;
    pl.Wp = ((W / 4) % 2 == 0) ? W + 4 : W;          // (Wp/4) odd: conflict-free 16-byte row accesses by lanes
    const int max_warps = ((pl.R >= 4 || pl.cptb == 16) ? 384 : 640) / 32;
    const int max_cpc = (max_warps - 4) / 4;
    pl.cpc = 0;
    for (int c = sh.cg() < max_cpc ? sh.cg() : max_cpc; c >= 1; --c) {
        if (sh.cg() % c) continue;
        if (tile_layout(sh, ES, c, 2, pl.Wp, &pl.prm) <= (size_t)kMaxSmemOptin) { pl.cpc = c; break; }
    }
    if (!pl.cpc) { set_error("fused fwd (tile): a %dx%d plane does not fit in shared memory", H, W); return GSPN_EUNSUPPORTED; }
    pl.ns = 2;
    while (pl.ns < 4 && tile_layout(sh, ES, pl.cpc, pl.ns + 1, pl.Wp, &pl.prm) <= (size_t)kMaxSmemOptin) ++pl.ns;
    pl.smem = tile_layout(sh, ES, pl.cpc, pl.ns, pl.Wp, &pl.prm);
    FwdTileParams& p = pl.prm;
    p.sh = sh; p.cpc = pl.cpc; p.ns = pl.ns; p.Wp = pl.Wp; p.L = pl.L;
    p.y = a.y; p.h0 = a.h0;
    int q = 0;
    for (int d = 0; d < 4; ++d) {
        p.nst[d] = 0; p.q[d] = 0;
        if (sh.mask >> d & 1u) {
            const int Ls = d < 2 ? H : W;
            p.nst[d] = (Ls + K - 1) / K;
            p.q[d] = q++;
        }
    }
    int rc = GSPN_EUNSUPPORTED;
#define GSPN_TILE_CASE(CB, RR) if (pl.cptb == CB && pl.R == RR) rc = launch_tile<ST, CB, RR>(a, pl, st);
    GSPN_TILE_CASE(4, 1) GSPN_TILE_CASE(4, 2) GSPN_TILE_CASE(4, 4)
    GSPN_TILE_CASE(8, 1) GSPN_TILE_CASE(8, 2) GSPN_TILE_CASE(8, 4)
    GSPN_TILE_CASE(16, 1) GSPN_TILE_CASE(16, 2) GSPN_TILE_CASE(16, 4)
#undef GSPN_TILE_CASE
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "fused_fwd_tile"; }
    return rc;
}

template int fused_fwd_launch<float>(const FwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int fused_fwd_launch<__nv_bfloat16>(const FwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
