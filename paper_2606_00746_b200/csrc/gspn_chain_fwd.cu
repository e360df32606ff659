// gspn_chain_fwd.cu -- fused forward scan of libgspn, "chain" design: ONE
// launch, every direction of dir_mask and the merge over directions, for any H, W <= 128 and storage
// type (rows and planes need not be 16-byte aligned).
//
// One CTA owns NC channels of one (b, group) unit; one WARP runs the recurrence of one channel
//     h[s] = w[s] h[s-1] + lambda[s]*x[s]            (Eq. 1 with Eq. 5's shared taps)
// with h in registers (P consecutive cross positions per lane), neighbours by warp shuffle and no
// block barrier on the serial path, and adds u[s]*h[s] (Eq. 2) into the channel's fp32
// plane Y on chip.  The directions run one after another, so Y has a single writer; after the last
// direction y = Y is rounded once (RNE) and stored with coalesced rows (Eq. 9's merge).
// Because forward has no reduction across the channels of a group, NC is chosen small (1 or 2): the CTA
// then needs little shared memory and several CTAs share an SM, which is where the latency hiding of
// this serial recurrence comes from; the taps of a group are re-read by its CTAs through L2.
//
// Operands: gspn_chain.cuh (producer warps, ring of row blocks / chunk columns, 16-byte-aligned
// supersets of unaligned rows, FHFMA for lambda*x).
#include "gspn_chain.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

constexpr int kCfMaxNC = 4;                       // channels per CTA
constexpr int kCfNPW = 2;                         // producer warps
constexpr int kCfMaxPlanes = 3 + 3 * kCfMaxNC;    // w0 w1 w2, lambda[c], x[c], u[c]

struct ChainFwdParams {
    Shape sh;
    const void *x, *w3, *lam, *u, *h0;
    void* y;
    int NC;                         // channels (= chain warps) per CTA
    int NSV, NSH, NQ;               // ring slots (row blocks / chunk columns); chunk columns per row
    int Wp;                         // row pitch of the Y planes in floats
    uint32_t vslot, vstage, hrow, hplane;
    uint32_t off_tab, off_y, off_ring, total;
    int q[4];                       // slab index of each direction, -1 = not in dir_mask
    unsigned long long bytes_x, bytes_c, bytes_w;
};

enum { FW0 = 0, FW1, FW2, FLAM, FX, FU, FNUM };

// One direction of one channel.  VH = false: T->B / B->T (lanes own columns), true: L->R / R->L (lanes
// own rows); REV = the direction walks the image lines downwards.
template <typename ST, int P, int CBH, bool VH, bool REV>
__device__ __forceinline__ void chain_fwd_dir(const ChainFwdParams& p, uint8_t* smem, const int d, const int b,
                                              const int cg0, const int c, const int lane, uint32_t& pf) {
    using E = Elem<ST>;
    using raw_t = typename E::raw_t;
    constexpr int ES = sizeof(ST);
    constexpr int CB = CBH;                           // horizontal: bytes of a row per chunk column
    constexpr int BLK = VH ? CB / ES : kBlk;          // scan steps per block (= ring stage)
    constexpr unsigned FULLM = 0xffffffffu;
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, NC = p.NC;
    const int Ls = VH ? W : H, Lp = VH ? H : W, Lmax = sh.Lmax();
    const int NB = (Ls + BLK - 1) / BLK;
    const uint32_t rowB = (uint32_t)W * ES;
    const int qd = p.q[d];
    const ChPlane* tb = reinterpret_cast<const ChPlane*>(smem + p.off_tab) + d * kCfMaxPlanes;
    const uint32_t ring = smem_u32(smem + p.off_ring);
    const int sidx[FNUM] = {0, 1, 2, 3 + c, 3 + NC + c, 3 + 2 * NC + c};
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
    const uint32_t ys = smem_u32(smem + p.off_y) + (uint32_t)c * H * p.Wp * 4;    // this channel's fp32 Y plane

    uint32_t phs[FNUM], vb[FNUM], hb[FNUM][P], yh[P];
    if constexpr (!VH) {
#pragma unroll
        for (int k = 0; k < FNUM; ++k) { phs[k] = (uint32_t)(tb[sidx[k]].b0 & 15ull); vb[k] = 0; }
    } else {
#pragma unroll
        for (int e = 0; e < P; ++e) {
            const int row = min(P * lane + e, H - 1);          // rows past the plane re-read the last row
#pragma unroll
            for (int k = 0; k < FNUM; ++k)
                hb[k][e] = ring + sidx[k] * p.hplane + row * p.hrow +
                           (uint32_t)((tb[sidx[k]].b0 + (unsigned long long)row * rowB) % CB);
            yh[e] = ys + (uint32_t)row * p.Wp * 4;
        }
    }
    const uint8_t* const sbase = smem - smem_u32(smem);           // generic address of shared offset 0
    auto ldr = [&](int k, int tl, uint32_t so, int e) -> raw_t {
        if constexpr (!VH) return *reinterpret_cast<const raw_t*>(sbase + (vb[k] + tl * rowB + e * ES));
        else return *reinterpret_cast<const raw_t*>(sbase + (hb[k][e] + so + tl * ES));
    };

    float h[P];
#pragma unroll
    for (int e = 0; e < P; ++e) {
        h[e] = 0.f;
        if (p.h0 && ok[e])
            h[e] = ld_f(reinterpret_cast<const ST*>(p.h0) + (((size_t)qd * sh.B + b) * sh.C + cg0 + c) * Lmax + P * lane + e);
    }
    rs.begin_pass(REV);
    uint32_t hso = 0;
    for (int n = 0; n < NB; ++n) {
        const int bi = REV ? NB - 1 - n : n;
        const int nb = min(BLK, Ls - BLK * bi);
        rs.acquire(bi, REV);
        uint32_t so = 0;
        if constexpr (!VH) {
            const uint32_t stage = ring + (bi % p.NSV) * p.vstage;
            const uint32_t rb = ((uint32_t)(BLK * bi) * rowB) & 15u;
#pragma unroll
            for (int k = 0; k < FNUM; ++k)
                vb[k] = stage + sidx[k] * p.vslot + ((phs[k] + rb) & 15u) + lane * (P * ES);
        } else {
            // fold the block's chunk-slot offset into the row addresses once per block
            const uint32_t nso = (uint32_t)(bi % p.NSH) * CB;
#pragma unroll
            for (int e = 0; e < P; ++e)
#pragma unroll
                for (int k = 0; k < FNUM; ++k) hb[k][e] += nso - hso;
            hso = nso;
        }
        const uint32_t yv = ys + ((uint32_t)(BLK * bi) * p.Wp + P * lane) * 4;      // vertical: (line 4bi, first column)
#pragma unroll
        for (int t = 0; t < BLK; ++t) {
            const int tl = REV ? BLK - 1 - t : t;
            if (tl < nb) {
                raw_t w0r[P], w1r[P], w2r[P], lr[P], xr[P], ur[P];
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    w0r[e] = ldr(FW0, tl, so, e); w1r[e] = ldr(FW1, tl, so, e); w2r[e] = ldr(FW2, tl, so, e);
                    lr[e] = ldr(FLAM, tl, so, e); xr[e] = ldr(FX, tl, so, e); ur[e] = ldr(FU, tl, so, e);
                }
                const float hl = maskf(__shfl_up_sync(FULLM, h[P - 1], 1), m_first);
                const float hr = __shfl_down_sync(FULLM, h[0], 1);     // lane 31: masked through m_w2 / okm
                float hn[P];
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    const float w0f = e == 0 ? maskf(E::f(w0r[e]), m_first) : E::f(w0r[e]);
                    const float w2f = maskf(E::f(w2r[e]), m_w2[e]);
                    const float left = e ? h[e - 1] : hl;
                    const float right = e < P - 1 ? h[e + 1] : hr;
                    float acc = E::f(w1r[e]) * h[e];
                    acc = fmaf(w0f, left, acc);
                    acc = fmaf(w2f, right, acc);
                    acc = E::fma2(lr[e], xr[e], acc);
                    hn[e] = maskf(acc, okm[e]);                         // positions past the line stay +0
                }
                // Y += u*h: the step's reads first, then its writes (one shared-memory round trip per step
                // instead of a read -> write -> read chain per position)
                float yo[P];
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    h[e] = hn[e];
                    const uint32_t a = VH ? yh[e] + (BLK * bi + tl) * 4 : yv + (tl * p.Wp + e) * 4;
                    yo[e] = 0.f;
                    if (ok[e]) yo[e] = lds32(a);
                }
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    const uint32_t a = VH ? yh[e] + (BLK * bi + tl) * 4 : yv + (tl * p.Wp + e) * 4;
                    if (ok[e]) sts32(a, fmaf(E::f(ur[e]), hn[e], yo[e]));
                }
            }
        }
        rs.release(bi, REV, n == NB - 1);
    }
    pf = rs.pf;
}

// ---------------------------------------------------------------------------------------------------
template <typename ST, int P, int CBH>
__global__ void __launch_bounds__(32 * (kCfNPW + kCfMaxNC))
chain_fwd_kernel(const ChainFwdParams p) {
    constexpr int ES = sizeof(ST);
    constexpr int CB = CBH;                           // horizontal chunk columns: CB bytes of every row
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    uint64_t* empty = full + kChSlots;
    ChPlane* tab = reinterpret_cast<ChPlane*>(smem + p.off_tab);       // [4][kCfMaxPlanes]
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, NC = p.NC;
    const int np = 3 + 3 * NC;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int slices = sh.cg() / NC;
    const int b = blockIdx.x / (sh.G * slices);
    const int g = (blockIdx.x / slices) % sh.G;
    const int c0 = g * sh.cg() + (blockIdx.x % slices) * NC;            // first channel of this CTA
    const unsigned long long HW = (unsigned long long)H * W;
    const uint32_t rowB = (uint32_t)W * ES;

    // shared memory starts as zeros: Y accumulates from 0, lanes past a line's end read finite values
    for (uint32_t o = threadIdx.x * 16; o < p.total; o += blockDim.x * 16)
        *reinterpret_cast<uint4*>(smem + o) = make_uint4(0, 0, 0, 0);
    __syncthreads();
    for (int idx = threadIdx.x; idx < 4 * kCfMaxPlanes; idx += blockDim.x) {
        const int d = idx / kCfMaxPlanes, s = idx % kCfMaxPlanes;
        if (p.q[d] >= 0 && s < np) {
            const unsigned long long q = p.q[d];
            ChPlane e;
            if (s < 3) {
                e.base = (const uint8_t*)p.w3; e.tbytes = p.bytes_w;
                e.b0 = ((((q * sh.B + b) * sh.G + g) * 3 + s) * HW) * ES;
            } else {
                const int t = (s - 3) / NC, c = (s - 3) % NC;          // 0 lambda, 1 x, 2 u
                const unsigned long long slab = (((q * sh.B + b) * sh.C + c0 + c) * HW) * ES;
                const unsigned long long img = (((unsigned long long)b * sh.C + c0 + c) * HW) * ES;
                if (t == 0)      { e.base = (const uint8_t*)p.lam; e.tbytes = p.bytes_c; e.b0 = slab; }
                else if (t == 1) { e.base = (const uint8_t*)p.x;   e.tbytes = p.bytes_x; e.b0 = img; }
                else             { e.base = (const uint8_t*)p.u;   e.tbytes = p.bytes_c; e.b0 = slab; }
            }
            tab[idx] = e;
        }
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < kChSlots; ++s) { mbar_init(&full[s], kCfNPW * 33); mbar_init(&empty[s], NC); }
        mbar_init_fence();
    }
    fence_proxy_async();      // zeros (generic proxy) before bulk copies
    __syncthreads();

    if (warp < kCfNPW) {
        // ---------------- producer warp pw: planes pw, pw + NPW, ... of every stage ----------------------
        const int pw = warp;
        const uint32_t ring = smem_u32(smem + p.off_ring);
        uint8_t* ringp = smem + p.off_ring;
        uint32_t pe = 0;
        bool drained = false;
        uint32_t rowoff[4], rowdst[4];                                  // horizontal: rows lane, lane+32, ...
#pragma unroll
        for (int r = 0; r < 4; ++r) { rowoff[r] = (uint32_t)(lane + 32 * r) * rowB; rowdst[r] = (uint32_t)(lane + 32 * r) * p.hrow; }
        for (int d = 0; d < 4; ++d) {
            if (p.q[d] < 0) continue;
            const bool vh = d >> 1, desc = d & 1;
            const ChPlane* tb = tab + d * kCfMaxPlanes;
            {   // announce every operand plane of this direction to L2
                const int s = lane * kCfNPW + pw;
                if (s < np) l2_prefetch_plane(tb[s].base, tb[s].b0, tb[s].tbytes, HW * ES);
            }
            if (vh && !drained) {
                // row-block stages and chunk columns lay the ring out differently: every slot must be
                // released before the first chunk column is written
                for (int s = 0; s < kChSlots; ++s) mbar_wait(&empty[s], ((pe >> s) & 1u) ^ 1u);
                drained = true;
            }
            if (!vh) {
                const int NB = (H + kBlk - 1) / kBlk;
                const int s = lane * kCfNPW + pw;                     // this lane's plane
                ChPlane e{nullptr, 0, 0};
                if (s < np) e = tb[s];
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
                    if (s < np) {
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
                    for (int s = pw; s < np; s += kCfNPW) {
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
    } else if (warp < kCfNPW + NC) {
        const int c = warp - kCfNPW;
        uint32_t pf = 0;
        if (p.q[0] >= 0) chain_fwd_dir<ST, P, CBH, false, false>(p, smem, 0, b, c0, c, lane, pf);
        if (p.q[1] >= 0) chain_fwd_dir<ST, P, CBH, false, true>(p, smem, 1, b, c0, c, lane, pf);
        if (p.q[2] >= 0) chain_fwd_dir<ST, P, CBH, true, false>(p, smem, 2, b, c0, c, lane, pf);
        if (p.q[3] >= 0) chain_fwd_dir<ST, P, CBH, true, true>(p, smem, 3, b, c0, c, lane, pf);
    }
    __syncthreads();

    // ---------------- y = sum over directions, one RNE, coalesced rows ---------------------------------
    {
        const float* Y = reinterpret_cast<const float*>(smem + p.off_y);
        ST* yg = reinterpret_cast<ST*>(p.y) + ((size_t)b * sh.C + c0) * HW;
        const int nw = blockDim.x >> 5;
        if (p.Wp == W) {       // odd W: Y has the pitch of the image rows, the CTA's planes are one contiguous run
            const int total = NC * H * W;
            for (int idx = threadIdx.x; idx < total; idx += blockDim.x) st_f(yg + idx, Y[idx]);
        } else {
            for (int ci = warp; ci < NC * H; ci += nw)
                for (int j = lane; j < W; j += 32) st_f(yg + (size_t)ci * W + j, Y[(size_t)ci * p.Wp + j]);
        }
    }
}

// ---- host side -----------------------------------------------------------------------------------
static size_t chain_fwd_layout(const Shape& sh, int es, int P, int NC, int NSV, int NSH, int CB, ChainFwdParams* prm) {
    const int np = 3 + 3 * NC;
    const bool vact = sh.mask & 3u, hact = sh.mask & 12u;
    size_t off = 2 * kChSlots * sizeof(uint64_t);
    prm->off_tab = (uint32_t)off;
    off += (size_t)4 * kCfMaxPlanes * sizeof(ChPlane);
    off = (off + 127) / 128 * 128;
    prm->Wp = sh.W | 1;
    prm->off_y = (uint32_t)off;
    off += (size_t)NC * sh.H * prm->Wp * 4;
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
    off = (off + 15) / 16 * 16;
    prm->total = (uint32_t)off;
    return off;
}

template <typename ST, int P, int CBH>
static int launch_chain_fwd(const ChainFwdParams& prm, int items, int threads, cudaStream_t st) {
    auto kern = chain_fwd_kernel<ST, P, CBH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("chain fwd: cudaFuncSetAttribute(%u B): %s", prm.total, cudaGetErrorString(e)); return GSPN_ECUDA; }
    GSPN_LAUNCH(kern, items, threads, prm.total, st, prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("chain fwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int chain_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    const Shape& sh = a.sh;
    const int L = sh.Lmax(), cg = sh.cg();
    const int P = (L + 31) / 32;
    if (P > 4) { set_error("chain fwd: max(H,W) = %d > 128", L); return GSPN_EUNSUPPORTED; }
    // channels per CTA: the count (1, 2 or 4, dividing cg) that puts the most chain warps on one SM
    // (228 KB of shared memory per SM, 1 KB reserved per CTA, at most 32 CTAs)
    // horizontal chunk columns: 16 bytes of every row when rows are not 16-byte aligned (half the copy
    // requests; the rows' different byte phases spread the row-per-lane reads over the banks), else 8 bytes
    // (row slots an odd number of 8-byte units apart: 2-way instead of 16-way bank conflicts)
    const int CBH = ((size_t)sh.W * ES) % 16 ? 16 : (ES == 4 ? 16 : 8);
    const int NSH = CBH == 16 && ES == 2 ? 3 : 4;
    ChainFwdParams best{};
    int best_warps = 0;
    for (int NC = 1; NC <= kCfMaxNC; NC *= 2) {
        if (cg % NC) continue;
        ChainFwdParams prm{};
        const size_t need = chain_fwd_layout(sh, ES, P, NC, 4, NSH, CBH, &prm);
        if (need > (size_t)kMaxSmemOptin) continue;
        int ctas = (int)((size_t)228 * 1024 / (need + 1024));
        if (ctas > 32) ctas = 32;
        const int tpc = 32 * (kCfNPW + NC);
        if (ctas * tpc > 2048) ctas = 2048 / tpc;
        const int warps = ctas * NC;
        if (warps > best_warps) { best_warps = warps; best = prm; best.NC = NC; }
    }
    if (!best_warps) {
        set_error("chain fwd: a %dx%d plane does not fit in shared memory", sh.H, sh.W);
        return GSPN_EUNSUPPORTED;
    }
    ChainFwdParams& prm = best;
    prm.NSH = NSH;            // prm.NSV was set by the layout
    prm.sh = sh;
    prm.x = a.x; prm.w3 = a.w3; prm.lam = a.lam; prm.u = a.u; prm.h0 = a.h0; prm.y = a.y;
    prm.NQ = (CBH - ES + sh.W * ES + CBH - 1) / CBH;
    const unsigned long long n = (unsigned long long)sh.B * sh.C * sh.H * sh.W;
    prm.bytes_x = n * ES;
    prm.bytes_c = (unsigned long long)sh.D() * n * ES;
    prm.bytes_w = (unsigned long long)sh.D() * sh.B * sh.G * 3 * sh.H * sh.W * ES;
    int q = 0;
    for (int d = 0; d < 4; ++d) prm.q[d] = (sh.mask >> d & 1u) ? q++ : -1;
    const int threads = 32 * (kCfNPW + prm.NC), items = sh.B * sh.G * (cg / prm.NC);
    int rc = GSPN_EUNSUPPORTED;
    constexpr int CBW = ES == 4 ? 16 : 8;       // the narrow variant (fp32: 16 bytes = 4 columns either way)
#define GSPN_CF_CASE(PP)                                                                              \
    case PP:                                                                                          \
        rc = CBH == CBW ? launch_chain_fwd<ST, PP, CBW>(prm, items, threads, st)                      \
                        : launch_chain_fwd<ST, PP, 16>(prm, items, threads, st);                      \
        break;
    switch (P) { GSPN_CF_CASE(1) GSPN_CF_CASE(2) GSPN_CF_CASE(3) GSPN_CF_CASE(4) }
#undef GSPN_CF_CASE
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "chain_fwd"; }
    return rc;
}

template int chain_fwd_launch<float>(const FwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int chain_fwd_launch<__nv_bfloat16>(const FwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
