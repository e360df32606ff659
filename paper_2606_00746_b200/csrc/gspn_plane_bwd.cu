// gspn_plane_bwd.cu -- fused backward scan of libgspn for SMALL planes (lines of at
// most one warp, e.g. the 378-px config's 27x27): ONE launch, CTA per (b, group) unit, every operand plane of the
// unit and of all four directions on chip as a whole (one 1-D bulk copy each), no rings, no gathers.
//
// The adjoint recurrence (include/gspn.h "Backward scan"; derived from Eq. 1-2,
// the paper gives backward timings only).  One WARP owns one direction and all
// NC = C/G channels of the group, one cross position per lane:
//   pass 1 (scan order)    h[s] = w[s] h[s-1] + lambda[s]*x[s], every h[s] kept in shared memory (fp32)
//   pass 2 (reverse order) gh[s] = dy[s]*u[s] + carry;  du = dy*h[s];  dlambda = x*gh;  dx += lambda*gh;
//                          dw3[k] = sum_c gh_c * h_c[s-1, p+k-1]  (the channels of the group live in one lane:
//                          ascending order in registers, no atomics);  carry = w[s]^T gh  (each lane multiplies
//                          its own taps, the products travel by shuffle)
// du, dlambda and dw3 overwrite u, lambda and the taps IN PLACE in shared memory (a lane reads its element of
// step s before it writes it) and leave the chip as whole planes at the end.  dx accumulates in fp32: T->B / B->T
// share one plane set, L->R / R->L another; the two warps of an axis sweep it in opposite senses in pass 2, meet
// once at a named barrier in the middle and never touch a line at the same time (no atomics); dx = sum, one RNE.
#include "gspn_chain.cuh"
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

struct PlaneBwdParams {
    Shape sh;
    const void *x, *w3, *lam, *u, *h0, *dy;
    void *dx, *dlam, *du, *dw3, *dh0;
    int Wp;
    uint32_t off_dxv, off_dxh, off_x, off_dy, off_pl, off_hs, plslot, hsdir, total;
    int q[4];
    unsigned long long bytes_x, bytes_c, bytes_w;
};

struct PbPlane { const uint8_t* base; unsigned long long b0, tbytes; };

// operand plane k of direction slab qd: 0..2 taps, 3+c lambda, 3+NC+c u
template <int NC, int ES>
__device__ __forceinline__ PbPlane pb_plane(const PlaneBwdParams& p, int qd, int b, int g, int k) {
    const Shape& sh = p.sh;
    const unsigned long long HW = (unsigned long long)sh.H * sh.W, q = (unsigned long long)qd;
    PbPlane e;
    if (k < 3) {
        e.base = (const uint8_t*)p.w3; e.tbytes = p.bytes_w;
        e.b0 = ((((q * sh.B + b) * sh.G + g) * 3 + k) * HW) * ES;
    } else {
        const int t = (k - 3) / NC, c = (k - 3) % NC;
        e.base = (const uint8_t*)(t == 0 ? p.lam : p.u); e.tbytes = p.bytes_c;
        e.b0 = (((q * sh.B + b) * sh.C + g * NC + c) * HW) * ES;
    }
    return e;
}

// 16-byte-aligned superset of [byte0, byte0 + n) inside the tensor; bytes past the tensor's last whole 16-byte
// chunk come by ordinary loads.  Returns the bytes to bulk-copy from base + *a0_out to dst.
__device__ __forceinline__ int pb_window(uint8_t* dst, const uint8_t* base, unsigned long long byte0, unsigned long long n,
                                         unsigned long long tbytes, int es, unsigned long long* a0_out) {
    const unsigned long long byte1 = byte0 + n;
    const unsigned long long a0 = byte0 & ~15ull, lim = tbytes & ~15ull;
    unsigned long long a1 = (byte1 + 15) & ~15ull;
    if (a1 > lim) a1 = lim;
    if (byte1 > a1)
        for (unsigned long long o = (a1 > byte0 ? a1 : byte0); o < byte1; o += es) {
            if (es == 2) *reinterpret_cast<unsigned short*>(dst + (o - a0)) = *reinterpret_cast<const unsigned short*>(base + o);
            else *reinterpret_cast<float*>(dst + (o - a0)) = *reinterpret_cast<const float*>(base + o);
        }
    *a0_out = a0;
    return a1 > a0 ? (int)(a1 - a0) : 0;
}

// One direction, all NC channels of the unit, on one warp.  VH = false: T->B / B->T (lanes own columns), true:
// L->R / R->L (lanes own rows); REV = the direction walks the image lines downwards.
// PART 0: the warp does everything.  PART 1 / 2 (NC >= 2): pass 1 is split between the direction's main warp
// (channels [0, NC/2)) and a helper warp (channels [NC/2, NC)); they meet at a named barrier, then the main warp
// runs pass 2 for all channels (dw3 is a sum over the group's channels: one warp, fixed order).
template <typename ST, int NC, bool VH, bool REV, int PART = 0>
__device__ __forceinline__ void plane_bwd_dir(const PlaneBwdParams& p, uint8_t* smem, const int d, const int b,
                                              const int g, const int lane, const bool pair_sync) {
    using E = Elem<ST>;
    using raw_t = typename E::raw_t;
    constexpr int ES = sizeof(ST), NP = 3 + 2 * NC;
    constexpr unsigned FULLM = 0xffffffffu;
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W, qd = p.q[d];
    const int Ls = VH ? W : H, Lp = VH ? H : W, Lmax = sh.Lmax();
    const uint32_t rowB = (uint32_t)W * ES;
    const uint32_t step = VH ? (uint32_t)ES : rowB;               // bytes from one image line of the scan to the next
    const int c0 = g * NC;
    const bool ok = lane < Lp;
    const uint32_t okm = ok ? 0xffffffffu : 0u;
    const uint32_t m_first = lane == 0 ? 0u : 0xffffffffu, m_last = lane == Lp - 1 ? 0u : 0xffffffffu;
    const int pos = min(lane, Lp - 1);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);

    // element (line 0, own position) of every plane
    uint32_t A[NP], AX[NC], AY[NC], DXA[NC];
#pragma unroll
    for (int k = 0; k < NP; ++k) {
        const unsigned long long b0 = pb_plane<NC, ES>(p, qd, b, g, k).b0;
        A[k] = smem_u32(smem + p.off_pl) + (uint32_t)(d * NP + k) * p.plslot + (uint32_t)(b0 & 15ull) +
               (VH ? (uint32_t)pos * rowB : (uint32_t)pos * ES);
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const unsigned long long xb0 = (((unsigned long long)b * sh.C + c0 + c) * H * W) * ES;
        const uint32_t o = (uint32_t)(xb0 & 15ull) + (VH ? (uint32_t)pos * rowB : (uint32_t)pos * ES);
        AX[c] = smem_u32(smem + p.off_x) + c * p.plslot + o;
        AY[c] = smem_u32(smem + p.off_dy) + c * p.plslot + o;
        DXA[c] = smem_u32(smem + (VH ? p.off_dxh : p.off_dxv)) + (uint32_t)c * H * p.Wp * 4 +
                 (VH ? (uint32_t)pos * p.Wp * 4 : (uint32_t)pos * 4);
    }
    const uint32_t dxstep = VH ? 4u : (uint32_t)p.Wp * 4;
    // h store of this direction: slot 0 = h0 (or zeros), slot s+1 = h[s]; [c][slot][32 lanes] fp32
    const uint32_t HS = smem_u32(smem + p.off_hs) + (uint32_t)d * p.hsdir + lane * 4;
    const uint32_t hsc = (uint32_t)(Lmax + 1) * 128;              // bytes per channel

    mbar_wait(&bars[4], 0);                                       // x, dy
    mbar_wait(&bars[d], 0);                                       // this direction's planes

    // ---------------- pass 1: h in scan order ------------------------------------------------------------
    constexpr int C0 = PART == 2 ? NC / 2 : 0, C1 = PART == 1 ? NC / 2 : NC;      // this warp's channels in pass 1
    float h[NC];
#pragma unroll
    for (int c = C0; c < C1; ++c) {
        h[c] = 0.f;
        if (p.h0 && ok)
            h[c] = ld_f(reinterpret_cast<const ST*>(p.h0) + (((size_t)qd * sh.B + b) * sh.C + c0 + c) * Lmax + lane);
        sts32(HS + c * hsc, h[c]);
    }
#pragma unroll 2
    for (int s = 0; s < Ls; ++s) {
        const uint32_t lo = (uint32_t)(REV ? Ls - 1 - s : s) * step;
        const float w0 = maskf(E::f(E::lds(A[0] + lo)), m_first);       // out-of-grid taps are never used
        const float w1 = E::f(E::lds(A[1] + lo));
        const float w2 = maskf(E::f(E::lds(A[2] + lo)), m_last);
        raw_t lr[NC], xr[NC];
#pragma unroll
        for (int c = C0; c < C1; ++c) { lr[c] = E::lds(A[3 + c] + lo); xr[c] = E::lds(AX[c] + lo); }
#pragma unroll
        for (int c = C0; c < C1; ++c) {
            const float hl = __shfl_up_sync(FULLM, h[c], 1), hr = __shfl_down_sync(FULLM, h[c], 1);
            float acc = w1 * h[c];
            acc = fmaf(w0, hl, acc);
            acc = fmaf(w2, hr, acc);
            acc = E::fma2(lr[c], xr[c], acc);
            h[c] = maskf(acc, okm);                                      // positions past the line stay +0
            sts32(HS + c * hsc + (uint32_t)(s + 1) * 128, h[c]);
        }
    }
    __syncwarp();
    if constexpr (PART != 0) {
        named_bar_sync(3 + d, 64);      // both halves of h are in shared memory
        if constexpr (PART == 2) return;
    }

    // ---------------- pass 2: adjoint chain in reverse order ---------------------------------------------
    const bool w_du = p.du != nullptr, w_dl = p.dlam != nullptr, w_dw = p.dw3 != nullptr, w_dx = p.dx != nullptr;
    const int mid = Ls / 2;                // line where the two warps of an axis meet (image line index)
    float carry[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) carry[c] = 0.f;
#pragma unroll 2
    for (int s = Ls - 1; s >= 0; --s) {
        const int li = REV ? Ls - 1 - s : s;                             // image line of this step
        // REV walks the lines upwards in pass 2, !REV downwards: the downward warp waits before line `mid`
        if (!REV && pair_sync && li == mid) named_bar_sync(VH ? 2 : 1, 64);
        const uint32_t lo = (uint32_t)li * step;
        const float w0 = E::f(E::lds(A[0] + lo)), w1 = E::f(E::lds(A[1] + lo)), w2 = E::f(E::lds(A[2] + lo));
        float dw0 = 0.f, dw1 = 0.f, dw2 = 0.f;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const raw_t lr = E::lds(A[3 + c] + lo), ur = E::lds(A[3 + NC + c] + lo);
            const raw_t xr = E::lds(AX[c] + lo), dyr = E::lds(AY[c] + lo);
            const uint32_t hsa = HS + c * hsc + (uint32_t)s * 128;       // slot s = h[s-1], slot s+1 = h[s]
            const float hp = lds32(hsa), hs = lds32(hsa + 128);
            const float hpl = maskf(lds32(hsa - 4), m_first), hpr = maskf(lds32(hsa + 4), m_last);
            const uint32_t dxa = DXA[c] + (uint32_t)li * dxstep;
            float dxo = 0.f;
            if (w_dx && ok) dxo = lds32(dxa);
            const float gh = maskf(E::fma2(dyr, ur, carry[c]), okm);
            if (w_du && ok) E::sts(A[3 + NC + c] + lo, E::pack(E::f(dyr) * hs));
            if (w_dl && ok) E::sts(A[3 + c] + lo, E::pack(E::f(xr) * gh));
            if (w_dx && ok) sts32(dxa, fmaf(E::f(lr), gh, dxo));
            dw0 = fmaf(gh, hpl, dw0);
            dw1 = fmaf(gh, hp, dw1);
            dw2 = fmaf(gh, hpr, dw2);
            const float froml = maskf(__shfl_up_sync(FULLM, w2 * gh, 1), m_first);     // w2[s,p-1]*gh[p-1]
            const float fromr = maskf(__shfl_down_sync(FULLM, w0 * gh, 1), m_last);    // w0[s,p+1]*gh[p+1]
            carry[c] = maskf(fmaf(w1, gh, froml + fromr), okm);
        }
        if (w_dw && ok) {
            E::sts(A[0] + lo, E::pack(dw0));
            E::sts(A[1] + lo, E::pack(dw1));
            E::sts(A[2] + lo, E::pack(dw2));
        }
        if (REV && pair_sync && li == mid) named_bar_sync(VH ? 2 : 1, 64);
    }
    if (p.dh0 && lane < Lmax) {                                    // entries past the line are zeros
#pragma unroll
        for (int c = 0; c < NC; ++c)
            st_f(reinterpret_cast<ST*>(p.dh0) + (((size_t)qd * sh.B + b) * sh.C + c0 + c) * Lmax + lane, carry[c]);
    }
}

// ---------------------------------------------------------------------------------------------------
template <typename ST, int NC>
__global__ void __launch_bounds__(NC >= 2 ? 288 : 160)
plane_bwd_kernel(const PlaneBwdParams p) {
    constexpr int ES = sizeof(ST), NP = 3 + 2 * NC;
    constexpr bool HELP = NC >= 2;                                // helper warps 4..7 take half of pass 1
    constexpr int PW = HELP ? 8 : 4, NWARP = PW + 1;              // producer warp, warps of the CTA
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);           // [0..3] direction planes, [4] x and dy
    const Shape sh = p.sh;
    const int H = sh.H, W = sh.W;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int b = blockIdx.x / sh.G, g = blockIdx.x % sh.G;
    const int c0 = g * NC;
    const unsigned long long HW = (unsigned long long)H * W;

    {   // both dx plane sets accumulate from zero
        uint8_t* z = smem + p.off_dxv;
        const uint32_t nb = p.off_x - p.off_dxv;
        for (uint32_t o = threadIdx.x * 16; o < nb; o += blockDim.x * 16)
            *reinterpret_cast<uint4*>(z + o) = make_uint4(0, 0, 0, 0);
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < 4; ++s) mbar_init(&bars[s], NP);           // one arrival per operand plane
        mbar_init(&bars[4], 2 * NC);
        mbar_init_fence();
    }
    __syncthreads();

    const bool act[4] = {p.q[0] >= 0, p.q[1] >= 0, p.q[2] >= 0, p.q[3] >= 0};
    if (warp == PW) {
        // every plane has its own lane (x and dy first: every direction needs them); a lane announces its bytes on
        // the plane's barrier and issues the copy at once
        for (int i = lane; i < 2 * NC + 4 * NP; i += 32) {
            const int t = i < 2 * NC ? -1 : (i - 2 * NC) / NP, k = i < 2 * NC ? i : (i - 2 * NC) % NP;
            if (t >= 0 && !act[t]) continue;
            unsigned long long a0 = 0;
            const uint8_t* base;
            uint8_t* dst;
            int nbytes;
            if (t < 0) {
                const int c = k % NC;
                base = (const uint8_t*)(k < NC ? p.x : p.dy);
                dst = smem + (k < NC ? p.off_x : p.off_dy) + (size_t)c * p.plslot;
                nbytes = pb_window(dst, base, (((unsigned long long)b * sh.C + c0 + c) * HW) * ES, HW * ES, p.bytes_x, ES, &a0);
            } else {
                const PbPlane e = pb_plane<NC, ES>(p, p.q[t], b, g, k);
                base = e.base;
                dst = smem + p.off_pl + (size_t)(t * NP + k) * p.plslot;
                nbytes = pb_window(dst, base, e.b0, HW * ES, e.tbytes, ES, &a0);
            }
            uint64_t* fb = &bars[t < 0 ? 4 : t];
            mbar_arrive_expect_tx(fb, (uint32_t)nbytes);             // also publishes the tail bytes written above
            if (nbytes > 0) bulk_load_1d(dst, base + a0, (uint32_t)nbytes, fb);
        }
    } else {
        constexpr int PM = HELP ? 1 : 0;
        if (warp == 0 && act[0]) plane_bwd_dir<ST, NC, false, false, PM>(p, smem, 0, b, g, lane, act[1]);
        if (warp == 1 && act[1]) plane_bwd_dir<ST, NC, false, true, PM>(p, smem, 1, b, g, lane, act[0]);
        if (warp == 2 && act[2]) plane_bwd_dir<ST, NC, true, false, PM>(p, smem, 2, b, g, lane, act[3]);
        if (warp == 3 && act[3]) plane_bwd_dir<ST, NC, true, true, PM>(p, smem, 3, b, g, lane, act[2]);
        if constexpr (HELP) {
            if (warp == 4 && act[0]) plane_bwd_dir<ST, NC, false, false, 2>(p, smem, 0, b, g, lane, act[1]);
            if (warp == 5 && act[1]) plane_bwd_dir<ST, NC, false, true, 2>(p, smem, 1, b, g, lane, act[0]);
            if (warp == 6 && act[2]) plane_bwd_dir<ST, NC, true, false, 2>(p, smem, 2, b, g, lane, act[3]);
            if (warp == 7 && act[3]) plane_bwd_dir<ST, NC, true, true, 2>(p, smem, 3, b, g, lane, act[2]);
        }
        fence_proxy_async();    // the in-place outputs, before the bulk stores read them
    }
    __syncthreads();

    // ---------------- outputs leave the chip as whole planes ------------------------------------------------
    const int hw = H * W;
    if (p.dx) {
        const float* dv = reinterpret_cast<const float*>(smem + p.off_dxv);
        const float* dh = reinterpret_cast<const float*>(smem + p.off_dxh);
        ST* dxg = reinterpret_cast<ST*>(p.dx) + ((size_t)b * sh.C + c0) * HW;
        if (p.Wp == W) {
            for (int idx = threadIdx.x; idx < NC * hw; idx += 32 * NWARP) st_f(dxg + idx, dv[idx] + dh[idx]);
        } else {
            for (int ci = warp; ci < NC * H; ci += NWARP)
                for (int j = lane; j < W; j += 32)
                    st_f(dxg + (size_t)ci * W + j, dv[(size_t)ci * p.Wp + j] + dh[(size_t)ci * p.Wp + j]);
        }
    }
    // du / dlambda / dw3 lie where u / lambda / the taps lay, at the byte phase they have in HBM (same tensor
    // offsets): the 16-byte-aligned interior of a plane leaves by ONE bulk store, the few elements before and
    // after it by ordinary stores
    for (int pl = warp; pl < 4 * NP; pl += NWARP) {
        const int d = pl / NP, k = pl % NP;
        if (!act[d]) continue;
        ST* out = k < 3 ? reinterpret_cast<ST*>(p.dw3) : (k < 3 + NC ? reinterpret_cast<ST*>(p.dlam) : reinterpret_cast<ST*>(p.du));
        if (!out) continue;
        const unsigned long long b0 = pb_plane<NC, ES>(p, p.q[d], b, g, k).b0;
        const uint32_t phase = (uint32_t)(b0 & 15ull), hwb = (uint32_t)hw * ES;
        const uint32_t head = min((16u - phase) & 15u, hwb);                 // bytes before the aligned interior
        const uint32_t inner = (hwb - head) & ~15u;
        const uint8_t* src = smem + p.off_pl + (size_t)pl * p.plslot + phase;
        uint8_t* dst = reinterpret_cast<uint8_t*>(out) + b0;
        if (lane == 0 && inner > 0)
            bulk_store_1d(dst + head, src + head, inner);
        for (uint32_t o = lane * ES; o < head; o += 32 * ES)
            *reinterpret_cast<ST*>(dst + o) = *reinterpret_cast<const ST*>(src + o);
        for (uint32_t o = head + inner + lane * ES; o < hwb; o += 32 * ES)
            *reinterpret_cast<ST*>(dst + o) = *reinterpret_cast<const ST*>(src + o);
    }
    // shared memory must outlive the bulk stores' reads
    bulk_commit();
    bulk_wait_read<0>();
}

// ---- host side -----------------------------------------------------------------------------------
static size_t plane_bwd_layout(const Shape& sh, int es, int NC, PlaneBwdParams* prm) {
    const int np = 3 + 2 * NC;
    size_t off = 128;
    prm->Wp = sh.W | 1;
    const size_t dset = ((size_t)NC * sh.H * prm->Wp * 4 + 127) / 128 * 128;
    prm->off_dxv = (uint32_t)off;
    prm->off_dxh = (uint32_t)(off + dset);
    off += 2 * dset;
    prm->plslot = (uint32_t)(((size_t)sh.H * sh.W * es + 32 + 15) / 16 * 16);
    prm->off_x = (uint32_t)off;  off += (size_t)NC * prm->plslot;
    prm->off_dy = (uint32_t)off; off += (size_t)NC * prm->plslot;
    prm->off_pl = (uint32_t)off; off += (size_t)4 * np * prm->plslot;
    off = (off + 127) / 128 * 128;
    off += 128;                                                 // the halo read below the first h slot
    prm->off_hs = (uint32_t)off;
    prm->hsdir = (uint32_t)((size_t)NC * (sh.Lmax() + 1) * 128);
    off += (size_t)4 * prm->hsdir + 128;                        // + the halo read past the last h slot
    off = (off + 15) / 16 * 16;
    prm->total = (uint32_t)off;
    return off;
}

template <typename ST, int NC>
static int launch_plane_bwd(const PlaneBwdParams& prm, int items, cudaStream_t st) {
    auto kern = plane_bwd_kernel<ST, NC>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("plane bwd: cudaFuncSetAttribute(%u B): %s", prm.total, cudaGetErrorString(e)); return GSPN_ECUDA; }
    GSPN_LAUNCH(kern, items, NC >= 2 ? 288 : 160, prm.total, st, prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("plane bwd: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int plane_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST);
    const Shape& sh = a.sh;
    const int cg = sh.cg();
    if (sh.Lmax() > 32) { set_error("plane bwd: max(H,W) = %d > 32", sh.Lmax()); return GSPN_EUNSUPPORTED; }
    if (cg != 1 && cg != 2 && cg != 4) { set_error("plane bwd: C/G = %d (1, 2 or 4 channels per group)", cg); return GSPN_EUNSUPPORTED; }
    PlaneBwdParams prm{};
    if (plane_bwd_layout(sh, ES, cg, &prm) > (size_t)kMaxSmemOptin) {
        set_error("plane bwd: the planes of a %dx%d unit do not fit in shared memory", sh.H, sh.W);
        return GSPN_EUNSUPPORTED;
    }
    prm.sh = sh;
    prm.x = a.x; prm.w3 = a.w3; prm.lam = a.lam; prm.u = a.u; prm.h0 = a.h0; prm.dy = a.dy;
    prm.dx = a.dx; prm.dlam = a.dlam; prm.du = a.du; prm.dw3 = a.dw3; prm.dh0 = a.dh0;
    const unsigned long long n = (unsigned long long)sh.B * sh.C * sh.H * sh.W;
    prm.bytes_x = n * ES;
    prm.bytes_c = (unsigned long long)sh.D() * n * ES;
    prm.bytes_w = (unsigned long long)sh.D() * sh.B * sh.G * 3 * sh.H * sh.W * ES;
    int q = 0;
    for (int d = 0; d < 4; ++d) prm.q[d] = (sh.mask >> d & 1u) ? q++ : -1;
    const int items = sh.B * sh.G;
    int rc = cg == 4 ? launch_plane_bwd<ST, 4>(prm, items, st) : cg == 2 ? launch_plane_bwd<ST, 2>(prm, items, st)
                                                                         : launch_plane_bwd<ST, 1>(prm, items, st);
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "plane_bwd"; }
    return rc;
}

template int plane_bwd_launch<float>(const BwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int plane_bwd_launch<__nv_bfloat16>(const BwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
