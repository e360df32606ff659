// gspn_flat_fwd.cu -- the universal fused forward scan of libgspn: every
// direction of dir_mask and the merge over directions in ONE launch, for any H, W and storage type
// (rows and planes need not be 16-byte aligned).  x, lambda, u, w3 are streamed once through shared
// memory (gspn_flat.cuh: bulk-copied row blocks for the vertical directions, cp.async-gathered chunk
// columns for the horizontal ones), the hidden state h of Eq. (1) lives in registers
// for the whole recurrence, y = sum_d u_d*h_d (Eq. 2 / Eq. 9) is accumulated on
// chip in fp32 and written once.
//
// Work split.  One CTA owns nch channels of one (b, group) unit.  Warps 0-3 are the producers of the
// four directions.  Every other warp runs one chain set = (direction d, CS channels): a lane owns P
// consecutive cross positions (columns for T->B / B->T, rows for L->R / R->L) of all CS channels, so
// the three taps of w3 (shared by the channels of a group, Eq. 5) are fetched and
// widened once per CS channels; neighbours inside a lane are registers, across lanes one shuffle each
// way per step and channel.  The two vertical chains of a channel share the fp32 plane Yv, the two
// horizontal ones Yh: whoever reaches a line first stores, the second adds, one mbarrier hand-shake
// per pair at half time.  After the last step the CTA adds Yv + Yh, rounds once (RNE) and stores y.
#include <type_traits>

#include "gspn_flat.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

constexpr int kFlatMaxStages = 8;
constexpr int kFlatBarBytes = 1024;      // full[4][8], empty[4][8], pair[2][8] = 80 mbarriers
constexpr int kFlatMaxPlanes = 16;       // 3 + 3*nch, nch <= 4

struct FlatFwdParams {
    Shape sh;
    const void *x, *w3, *lam, *u, *h0;
    void* y;
    int nch, ncs;                 // channels per CTA; chain sets per direction (nch / CS)
    int Kv, NSv, nstv;            // vertical: rows per stage, ring slots, stages
    int NSh, NQ, T;               // horizontal: ring slots, chunk columns, column blocks
    uint32_t vslot, vstage;       // bytes of one plane slot / of one stage of a vertical ring
    uint32_t hrow, hplane;        // bytes of one (plane,row) = (NSh+1)*16 / of one plane of a horizontal ring
    uint32_t off_yv, off_yh, off_tab, off_ring[4];
    int Wp;                       // row pitch of Yh in floats
    int q[4];                     // slab index of each direction, -1 = not in dir_mask
    unsigned long long bytes_x, bytes_c, bytes_w;
};

struct PlaneEnt {                 // table entry in shared memory: one operand plane of one direction
    const uint8_t* base;
    unsigned long long b0;        // first byte of the plane inside the tensor
    unsigned long long tbytes;
};

// dir 0 T->B, 1 B->T, 2 L->R, 3 R->L
template <typename ST, int P, int CS>
__global__ void __launch_bounds__(512, 1)
fwd_flat_kernel(const FlatFwdParams p) {
    constexpr int ES = sizeof(ST);
    constexpr int KC = 16 / ES;             // columns per horizontal block
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);            // [4][8]
    uint64_t* empty = full + 4 * kFlatMaxStages;                   // [4][8]
    uint64_t* pairb = empty + 4 * kFlatMaxStages;                  // [2][8]
    PlaneEnt* tab = reinterpret_cast<PlaneEnt*>(smem + p.off_tab); // [4][kFlatMaxPlanes]

    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, nch = p.nch, ncs = p.ncs;
    const int np = 3 + 3 * nch;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int slices = sh.cg() / nch;
    const int item = blockIdx.x;
    const int b = item / (sh.G * slices);
    const int g = (item / slices) % sh.G;
    const int c0 = g * sh.cg() + (item % slices) * nch;
    const bool vact = (sh.mask & 3u) != 0, hact = (sh.mask & 12u) != 0;
    const unsigned long long HW = (unsigned long long)H * W;

    if (threadIdx.x < 4 * kFlatMaxPlanes) {
        const int d = threadIdx.x / kFlatMaxPlanes, s = threadIdx.x % kFlatMaxPlanes;
        if (p.q[d] >= 0 && s < np) {
            const unsigned long long q = p.q[d];
            PlaneEnt e;
            if (s < 3) {
                e.base = (const uint8_t*)p.w3; e.tbytes = p.bytes_w;
                e.b0 = ((((q * sh.B + b) * sh.G + g) * 3 + s) * HW) * ES;
            } else if (s < 3 + 2 * nch) {
                const bool isu = s >= 3 + nch;
                e.base = (const uint8_t*)(isu ? p.u : p.lam); e.tbytes = p.bytes_c;
                e.b0 = (((q * sh.B + b) * sh.C + c0 + (s - 3 - (isu ? nch : 0))) * HW) * ES;
            } else {
                e.base = (const uint8_t*)p.x; e.tbytes = p.bytes_x;
                e.b0 = (((unsigned long long)b * sh.C + c0 + (s - 3 - 2 * nch)) * HW) * ES;
            }
            tab[d * kFlatMaxPlanes + s] = e;
        }
    }
    if (threadIdx.x == 0) {
        for (int d = 0; d < 4; ++d)
            for (int s = 0; s < kFlatMaxStages; ++s) {
                mbar_init(&full[d * kFlatMaxStages + s], d < 2 ? 1 : 33);
                mbar_init(&empty[d * kFlatMaxStages + s], ncs);
            }
        for (int t = 0; t < 16; ++t) mbar_init(&pairb[t], 2);
        mbar_init_fence();
    }
    __syncthreads();

    if (warp < 4) {
        const int d = warp;
        if (p.q[d] >= 0) {
            uint8_t* ring = smem + p.off_ring[d];
            if (d < 2) {
                // ---------------- vertical producer: one bulk copy per plane and stage ---------------
                PlaneEnt e{nullptr, 0, 0};
                if (lane < np) e = tab[d * kFlatMaxPlanes + lane];
                for (int t = 0; t < p.nstv; ++t) {
                    const int slot = t % p.NSv, it = t / p.NSv;
                    int r0, r1;
                    if (d == 0) { r0 = t * p.Kv; r1 = min(H, r0 + p.Kv); }
                    else        { r1 = H - t * p.Kv; r0 = max(0, r1 - p.Kv); }
                    mbar_wait(&empty[d * kFlatMaxStages + slot], (it & 1) ^ 1);
                    uint64_t* fb = &full[d * kFlatMaxStages + slot];
                    int nb = 0;
                    unsigned long long a0 = 0;
                    uint8_t* dst = ring + (size_t)slot * p.vstage + (size_t)lane * p.vslot;
                    if (lane < np) {
                        const unsigned long long byte0 = e.b0 + (unsigned long long)r0 * W * ES;
                        const unsigned long long byte1 = e.b0 + (unsigned long long)r1 * W * ES;
                        a0 = byte0 & ~15ull;
                        const unsigned long long lim = e.tbytes & ~15ull;
                        unsigned long long a1 = (byte1 + 15) & ~15ull;
                        if (a1 > lim) a1 = lim;
                        nb = a1 > a0 ? (int)(a1 - a0) : 0;
                        if (byte1 > a1) {     // bytes past the tensor's last whole chunk: ordinary loads
                            for (unsigned long long o = (a1 > byte0 ? a1 : byte0); o < byte1; o += ES)
                                *reinterpret_cast<ST*>(dst + (o - a0)) = *reinterpret_cast<const ST*>(e.base + o);
                        }
                    }
                    const int total = warp_sum(nb);
                    __syncwarp();
                    if (lane == 0) mbar_arrive_expect_tx(fb, (uint32_t)total);
                    __syncwarp();
                    if (nb > 0) bulk_load_1d(dst, e.base + a0, (uint32_t)nb, fb);
                }
            } else {
                // ---------------- horizontal producer: gather one chunk column per stage -------------
                const int NS = p.NSh;
                for (int n = 0; n < p.NQ; ++n) {
                    const int qn = d == 2 ? n : p.NQ - 1 - n;
                    const int slot = qn % NS, it = n / NS;
                    mbar_wait(&empty[d * kFlatMaxStages + slot], (it & 1) ^ 1);
                    uint64_t* fb = &full[d * kFlatMaxStages + slot];
                    int s = 0, i = lane;
                    while (i >= H) { i -= H; ++s; }
                    while (s < np) {
                        const PlaneEnt e = tab[d * kFlatMaxPlanes + s];
                        const unsigned long long rowb = e.b0 + (unsigned long long)i * W * ES;
                        const unsigned long long cb = ((rowb >> 4) + qn) << 4;
                        uint8_t* dst = ring + (size_t)s * p.hplane + (size_t)i * p.hrow + slot * 16;
                        if (cb + 16 <= e.tbytes) {
                            cp_async_16(dst, e.base + cb);
                            if (slot == 0) cp_async_16(dst + NS * 16, e.base + cb);
                        } else if (cb < e.tbytes) {
                            for (unsigned long long o = cb; o < e.tbytes; o += ES) {
                                const ST v = *reinterpret_cast<const ST*>(e.base + o);
                                *reinterpret_cast<ST*>(dst + (o - cb)) = v;
                                if (slot == 0) *reinterpret_cast<ST*>(dst + NS * 16 + (o - cb)) = v;
                            }
                        }
                        i += 32;
                        while (i >= H) { i -= H; ++s; }
                    }
                    cp_async_arrive_noinc(fb);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(fb);
                }
            }
        }
    } else {
        // ---------------- chain set (direction d, channels cs*CS .. cs*CS+CS-1 of the CTA) -----------
        const int cw = warp - 4;
        const int d = cw / ncs, cs = cw % ncs;
        if (d < 4 && p.q[d] >= 0) {
            const int vh = d >> 1;
            const bool rev = d & 1;
            const bool partner = (sh.mask >> (d ^ 1)) & 1u;
            uint64_t* pb = &pairb[vh * 8 + cs];
            const uint32_t ring = smem_u32(smem + p.off_ring[d]);
            const int Lp = vh ? H : W;                 // cross length
            const int Ls = vh ? W : H;                 // scan length
            const int chb = cs * CS;                   // first channel (inside the CTA) of this set
            // per-lane position bookkeeping
            bool ok[P];
#pragma unroll
            for (int e = 0; e < P; ++e) ok[e] = P * lane + e < Lp;
            const bool lane_first = lane == 0;
            const int last_lane = (Lp - 1) / P, last_e = (Lp - 1) % P;
            float h[CS][P];
#pragma unroll
            for (int c = 0; c < CS; ++c)
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    h[c][e] = 0.f;
                    if (p.h0 && ok[e]) {
                        const size_t o = ((size_t)(p.q[d] * sh.B + b) * sh.C + c0 + chb + c) * sh.Lmax() + P * lane + e;
                        h[c][e] = ld_f(reinterpret_cast<const ST*>(p.h0) + o);
                    }
                }
            // byte phases (mod 16) of the planes this set reads: w0,w1,w2, then lambda,u,x per channel
            const PlaneEnt* tb = tab + d * kFlatMaxPlanes;
            uint32_t ph[3 + 3 * CS];
            int sidx[3 + 3 * CS];
#pragma unroll
            for (int k = 0; k < 3; ++k) sidx[k] = k;
#pragma unroll
            for (int c = 0; c < CS; ++c) {
                sidx[3 + 3 * c] = 3 + chb + c;
                sidx[4 + 3 * c] = 3 + nch + chb + c;
                sidx[5 + 3 * c] = 3 + 2 * nch + chb + c;
            }
#pragma unroll
            for (int k = 0; k < 3 + 3 * CS; ++k) ph[k] = (uint32_t)(tb[sidx[k]].b0 & 15ull);

            // one recurrence step on widened operands; returns y contributions in yv
            auto step = [&](float (&w0)[P], float (&w1)[P], float (&w2)[P], float (&lm)[CS][P],
                            float (&uu)[CS][P], float (&xx)[CS][P], float (&yv)[CS][P]) {
                if (lane_first) w0[0] = 0.f;                         // out-of-grid tap: never used
#pragma unroll
                for (int e = 0; e < P; ++e) if (lane == last_lane && e == last_e) w2[e] = 0.f;
#pragma unroll
                for (int c = 0; c < CS; ++c) {
                    float hl = __shfl_up_sync(0xffffffffu, h[c][P - 1], 1);
                    float hr = __shfl_down_sync(0xffffffffu, h[c][0], 1);
                    if (lane_first) hl = 0.f;
                    if (lane == 31) hr = 0.f;
                    float hn[P];
#pragma unroll
                    for (int e = 0; e < P; ++e) {
                        const float left = e ? h[c][e - 1] : hl;
                        const float right = e < P - 1 ? h[c][e + 1] : hr;
                        float acc = lm[c][e] * xx[c][e];
                        acc = fmaf(w1[e], h[c][e], acc);
                        acc = fmaf(w0[e], left, acc);
                        acc = fmaf(w2[e], right, acc);
                        hn[e] = ok[e] ? acc : 0.f;                   // positions past the line stay 0
                        yv[c][e] = uu[c][e] * hn[e];
                    }
#pragma unroll
                    for (int e = 0; e < P; ++e) h[c][e] = hn[e];
                }
            };

            bool synced = false;
            if (!vh) {
                // ======== vertical: lane owns columns [P*lane, P*lane+P) ============================
                const uint32_t yv0 = smem_u32(smem + p.off_yv);
                const int rstar = (H - 1) / 2;
                const int sync_step = rev ? H - 1 - rstar : rstar + 1;   // first step that adds
                int s_glob = 0;
                for (int t = 0; t < p.nstv; ++t) {
                    const int slot = t % p.NSv, it = t / p.NSv;
                    int r0, r1;
                    if (!rev) { r0 = t * p.Kv; r1 = min(H, r0 + p.Kv); }
                    else      { r1 = H - t * p.Kv; r0 = max(0, r1 - p.Kv); }
                    mbar_wait(&full[d * kFlatMaxStages + slot], it & 1);
                    const uint32_t stage = ring + slot * p.vstage;
                    const uint32_t rb = (uint32_t)(((unsigned long long)r0 * W * ES) & 15ull);
                    uint32_t base[3 + 3 * CS];
#pragma unroll
                    for (int k = 0; k < 3 + 3 * CS; ++k)
                        base[k] = stage + sidx[k] * p.vslot + ((ph[k] + rb) & 15u) + lane * (P * ES);
                    const int nr = r1 - r0;
                    for (int jr = 0; jr < nr; ++jr, ++s_glob) {
                        const int r = rev ? nr - 1 - jr : jr;
                        const int i = r0 + r;
                        if (partner && s_glob == sync_step) {
                            __syncwarp();
                            if (lane == 0) mbar_arrive(pb);
                            mbar_wait(pb, 0);
                            synced = true;
                        }
                        const uint32_t ro = (uint32_t)r * W * ES;
                        float w0[P], w1[P], w2[P], lm[CS][P], uu[CS][P], xx[CS][P], yv[CS][P];
#pragma unroll
                        for (int e = 0; e < P; ++e) {
                            w0[e] = lds_f<ST>(base[0] + ro + e * ES);
                            w1[e] = lds_f<ST>(base[1] + ro + e * ES);
                            w2[e] = lds_f<ST>(base[2] + ro + e * ES);
                        }
#pragma unroll
                        for (int c = 0; c < CS; ++c)
#pragma unroll
                            for (int e = 0; e < P; ++e) {
                                lm[c][e] = lds_f<ST>(base[3 + 3 * c] + ro + e * ES);
                                uu[c][e] = lds_f<ST>(base[4 + 3 * c] + ro + e * ES);
                                xx[c][e] = lds_f<ST>(base[5 + 3 * c] + ro + e * ES);
                            }
                        step(w0, w1, w2, lm, uu, xx, yv);
                        const bool add = partner && s_glob >= sync_step;
#pragma unroll
                        for (int c = 0; c < CS; ++c) {
                            // Yv[ch][i][e][lane]: conflict-free for every P
                            const uint32_t ya = yv0 + ((((chb + c) * H + i) * P) * 32 + lane) * 4;
#pragma unroll
                            for (int e = 0; e < P; ++e) {
                                float v = yv[c][e];
                                if (add) v += lds_f32(ya + e * 128);
                                sts_f32(ya + e * 128, v);
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[d * kFlatMaxStages + slot]);
                }
            } else {
                // ======== horizontal: lane owns rows [P*lane, P*lane+P) =============================
                const uint32_t yh0 = smem_u32(smem + p.off_yh);
                const int NS = p.NSh, NQ = p.NQ, T = p.T;
                // address of (plane k, row e) inside the ring, at chunk slot 0, plus the row's byte phase
                uint32_t a0[3 + 3 * CS][P];
                uint32_t yrow[P];
#pragma unroll
                for (int e = 0; e < P; ++e) {
                    const int i = min(P * lane + e, H - 1);          // rows past the plane re-read the last row
                    const uint32_t rp = (uint32_t)(((unsigned long long)i * W * ES) & 15ull);
#pragma unroll
                    for (int k = 0; k < 3 + 3 * CS; ++k)
                        a0[k][e] = ring + sidx[k] * p.hplane + i * p.hrow + ((ph[k] + rp) & 15u);
                    yrow[e] = (uint32_t)i * p.Wp * 4;
                }
                const int ncs_blocks = (T + 1) / 2;
                const int sync_blk = rev ? T - ncs_blocks : ncs_blocks;   // first block (in processing order) that adds
                // stages are loaded in processing order n = 0..NQ-1 (chunk column n for L->R, NQ-1-n for R->L)
                int waited = 0;                                      // stages [0, waited) have been waited for
                auto wait_upto = [&](int n_last) {                   // make stages 0..n_last visible
                    for (; waited <= n_last && waited < NQ; ++waited) {
                        const int qn = rev ? NQ - 1 - waited : waited;
                        mbar_wait(&full[d * kFlatMaxStages + qn % NS], (waited / NS) & 1);
                    }
                };
                for (int tb_ = 0; tb_ < T; ++tb_) {
                    const int t = rev ? T - 1 - tb_ : tb_;           // column block [t*KC, t*KC+KC)
                    // needs chunk columns t and t+1: processing indices
                    const int need = rev ? NQ - 1 - t : min(t + 1, NQ - 1);
                    wait_upto(need);
                    if (partner && tb_ == sync_blk) {
                        __syncwarp();
                        if (lane == 0) mbar_arrive(pb);
                        mbar_wait(pb, 0);
                        synced = true;
                    }
                    const bool add = partner && tb_ >= sync_blk;
                    const uint32_t so = (uint32_t)(t % NS) * 16;
#pragma unroll
                    for (int jj_ = 0; jj_ < KC; ++jj_) {
                        const int jj = rev ? KC - 1 - jj_ : jj_;
                        const int j = t * KC + jj;
                        if (j < W) {
                            float w0[P], w1[P], w2[P], lm[CS][P], uu[CS][P], xx[CS][P], yv[CS][P];
#pragma unroll
                            for (int e = 0; e < P; ++e) {
                                w0[e] = lds_f<ST>(a0[0][e] + so + jj * ES);
                                w1[e] = lds_f<ST>(a0[1][e] + so + jj * ES);
                                w2[e] = lds_f<ST>(a0[2][e] + so + jj * ES);
                            }
#pragma unroll
                            for (int c = 0; c < CS; ++c)
#pragma unroll
                                for (int e = 0; e < P; ++e) {
                                    lm[c][e] = lds_f<ST>(a0[3 + 3 * c][e] + so + jj * ES);
                                    uu[c][e] = lds_f<ST>(a0[4 + 3 * c][e] + so + jj * ES);
                                    xx[c][e] = lds_f<ST>(a0[5 + 3 * c][e] + so + jj * ES);
                                }
                            step(w0, w1, w2, lm, uu, xx, yv);
#pragma unroll
                            for (int c = 0; c < CS; ++c) {
                                const uint32_t yc = yh0 + (uint32_t)((chb + c) * H) * p.Wp * 4 + j * 4;
#pragma unroll
                                for (int e = 0; e < P; ++e) {
                                    if (ok[e]) {
                                        float v = yv[c][e];
                                        if (add) v += lds_f32(yc + yrow[e]);
                                        sts_f32(yc + yrow[e], v);
                                    }
                                }
                            }
                        }
                    }
                    // chunk column no longer needed: t (L->R) or t+1 (R->L)
                    __syncwarp();
                    if (lane == 0) {
                        if (!rev) mbar_arrive(&empty[d * kFlatMaxStages + t % NS]);
                        else if (t + 1 < NQ) mbar_arrive(&empty[d * kFlatMaxStages + (t + 1) % NS]);
                    }
                }
                wait_upto(NQ - 1);      // every issued stage has landed before the CTA may exit
            }
            if (partner && !synced) {
                __syncwarp();
                if (lane == 0) mbar_arrive(pb);
            }
        }
    }
    __syncthreads();

    // ---------------- merge: y = Yv + Yh, one RNE, coalesced stores ---------------------------------
    {
        const float* Yv = reinterpret_cast<const float*>(smem + p.off_yv);
        const float* Yh = reinterpret_cast<const float*>(smem + p.off_yh);
        ST* yg = reinterpret_cast<ST*>(p.y) + ((size_t)b * sh.C + c0) * HW;
        const int total = nch * H * W;
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            const int j = idx % W;
            const int ci = idx / W;                     // ch*H + i
            float acc = 0.f;
            if (vact) acc += Yv[((size_t)ci * P + j % P) * 32 + j / P];
            if (hact) acc += Yh[(size_t)ci * p.Wp + j];
            st_f(yg + idx, acc);
        }
    }
}

// ---- host side -----------------------------------------------------------------------------------
struct FlatPlan {
    int P, CS;
    size_t smem;
    int threads;
    FlatFwdParams prm;
};

static size_t flat_layout(const Shape& sh, int es, int P, int nch, int Kv, int NSv, int NSh, FlatFwdParams* prm) {
    const bool vact = sh.mask & 3u, hact = sh.mask & 12u;
    const int np = 3 + 3 * nch;
    size_t off = kFlatBarBytes;
    prm->off_tab = (uint32_t)off;
    off += 4 * kFlatMaxPlanes * sizeof(PlaneEnt);
    off = (off + 127) / 128 * 128;
    prm->off_yv = (uint32_t)off;
    if (vact) off += (size_t)nch * sh.H * P * 32 * 4;
    off = (off + 127) / 128 * 128;
    prm->Wp = (sh.W % 2) ? sh.W : sh.W + 1;
    prm->off_yh = (uint32_t)off;
    if (hact) off += (size_t)nch * sh.H * prm->Wp * 4;
    off = (off + 127) / 128 * 128;
    const int over = 32 * P > sh.W ? 32 * P - sh.W : 0;   // lanes past the row end read (and discard) this much
    prm->vslot = (uint32_t)(((size_t)Kv * sh.W * es + 16 + (size_t)over * es + 15) / 16 * 16);
    prm->vstage = (uint32_t)(np * prm->vslot);
    prm->hrow = (uint32_t)((NSh + 1) * 16);
    prm->hplane = (uint32_t)(sh.H * prm->hrow);
    for (int d = 0; d < 4; ++d) {
        prm->off_ring[d] = (uint32_t)off;
        if (!(sh.mask >> d & 1u)) continue;
        if (d < 2) off += (size_t)NSv * prm->vstage;
        else off += (size_t)np * prm->hplane + 64;
        off = (off + 127) / 128 * 128;
    }
    return off;
}

template <typename ST, int P, int CS>
static int launch_flat(const FlatPlan& pl, int items, cudaStream_t st) {
    auto kern = fwd_flat_kernel<ST, P, CS>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("flat fwd: cudaFuncSetAttribute(%zu B): %s", pl.smem, cudaGetErrorString(e)); return GSPN_ECUDA; }
    GSPN_LAUNCH(kern, items, pl.threads, pl.smem, st, pl.prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("flat fwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int flat_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    const Shape& sh = a.sh;
    const int H = sh.H, W = sh.W, L = sh.Lmax();
    if (L > 256) { set_error("flat fwd: max(H,W) = %d > 256", L); return GSPN_EUNSUPPORTED; }
    FlatPlan pl{};
    const int pneed = (L + 31) / 32;
    pl.P = pneed <= 4 ? pneed : (pneed <= 6 ? 6 : 8);
    const int cg = sh.cg();
    // channels per CTA: as many (<= 4, dividing cg) as leave room for the rings
    const size_t budget = (size_t)kMaxSmemOptin;
    int best_nch = 0, best_cs = 1, bKv = 0, bNSv = 0, bNSh = 0;
    // first fit in priority order: a 4-slot horizontal ring (2 slots cannot prefetch), then as many
    // channels (<= 4, dividing cg) as fit, then deep vertical rings of ~6 KB stages
    for (int NSh = 4; NSh >= 2 && !best_nch; NSh -= 2)
        for (int nch = cg < 4 ? cg : 4; nch >= 1 && !best_nch; --nch) {
            if (cg % nch) continue;
            if (pl.P > 4 && nch > 2) continue;               // register budget of the wide variants
            const int np = 3 + 3 * nch;
            int Kv0 = (int)(6144 / ((size_t)np * W * ES));
            if (Kv0 < 1) Kv0 = 1;
            if (Kv0 > H) Kv0 = H;
            for (int NSv = 4; NSv >= 2 && !best_nch; --NSv)
                for (int Kv = Kv0; Kv >= 1; Kv = Kv / 2) {
                    FlatFwdParams tmp{};
                    if (flat_layout(sh, ES, pl.P, nch, Kv, NSv, NSh, &tmp) <= budget) {
                        best_nch = nch; bKv = Kv; bNSv = NSv; bNSh = NSh;
                        break;
                    }
                    if (Kv == 1) break;
                }
        }
    if (!best_nch) { set_error("flat fwd: a %dx%d plane does not fit in shared memory", H, W); return GSPN_EUNSUPPORTED; }
    best_cs = (best_nch % 2 == 0 && pl.P <= 4) ? 2 : 1;
    pl.CS = best_cs;
    FlatFwdParams& p = pl.prm;
    pl.smem = flat_layout(sh, ES, pl.P, best_nch, bKv, bNSv, bNSh, &p);
    p.sh = sh; p.x = a.x; p.w3 = a.w3; p.lam = a.lam; p.u = a.u; p.h0 = a.h0; p.y = a.y;
    p.nch = best_nch; p.ncs = best_nch / best_cs;
    p.Kv = bKv; p.NSv = bNSv; p.nstv = (H + bKv - 1) / bKv;
    p.NSh = bNSh;
    p.NQ = (16 - ES + W * ES - 1) / 16 + 1;
    p.T = (W * ES + 15) / 16;
    const unsigned long long n = (unsigned long long)sh.B * sh.C * H * W;
    p.bytes_x = n * ES;
    p.bytes_c = (unsigned long long)sh.D() * n * ES;
    p.bytes_w = (unsigned long long)sh.D() * sh.B * sh.G * 3 * H * W * ES;
    int q = 0;
    for (int d = 0; d < 4; ++d) p.q[d] = (sh.mask >> d & 1u) ? q++ : -1;
    pl.threads = (4 + 4 * p.ncs) * 32;
    const int items = sh.B * sh.G * (cg / best_nch);
    int rc = GSPN_EUNSUPPORTED;
#define GSPN_FLAT_CASE(PP, CC) if (pl.P == PP && pl.CS == CC) rc = launch_flat<ST, PP, CC>(pl, items, st);
    GSPN_FLAT_CASE(1, 1) GSPN_FLAT_CASE(1, 2) GSPN_FLAT_CASE(2, 1) GSPN_FLAT_CASE(2, 2)
    GSPN_FLAT_CASE(3, 1) GSPN_FLAT_CASE(3, 2) GSPN_FLAT_CASE(4, 1) GSPN_FLAT_CASE(4, 2)
    GSPN_FLAT_CASE(6, 1) GSPN_FLAT_CASE(8, 1)
#undef GSPN_FLAT_CASE
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "fused_fwd_flat"; }
    return rc;
}

template int flat_fwd_launch<float>(const FwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int flat_fwd_launch<__nv_bfloat16>(const FwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
