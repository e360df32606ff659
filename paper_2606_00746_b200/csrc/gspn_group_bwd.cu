// gspn_group_bwd.cu -- fused backward scan of libgspn for one (b, group)
// unit per CTA, ONE launch: every direction of dir_mask, dx summed over directions on chip, dw3
// reduced over the group's channels on chip in fixed order (no atomics), h recomputed on chip.
//
// The adjoint recurrence (include/gspn.h "Backward scan"; derived from Eq. 1-2,
// the paper gives backward timings only).  Per direction:
//   sweep 1 (scan order)    h[s] = w[s] h[s-1] + lambda[s]*x[s]            -> kept in shared memory (fp32)
//   sweep 2 (reverse order) gh[s] = dy[s]*u[s] + carry;  du = dy*h[s];  dlambda = x*gh;
//                           dx += lambda*gh;  dw3[k] = sum_c gh_c * h_c[s-1, p+k-1];  carry = w[s]^T gh
//
// Thread (c, p) owns cross position p of channel c of the group; a scan step costs two block barriers
// (neighbour exchange of h or gh through a line buffer).  Operands never come from global memory on
// the serial path: the CTA streams TILES of T scan steps of every operand plane through shared memory
// with coalesced loads (rows for T->B/B->T, T-column row segments for L->R/R->L: the transposed tile),
// fetched into registers one tile ahead so the global latency overlaps the previous tile's steps.
// Outputs go through the same tiles: one RNE when a value enters the tile, coalesced stores after T steps.
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

constexpr int kGT = 8;              // scan steps per tile
constexpr int kGroupMaxThreads = 512;

// storage <-> fp32 for values that live in shared memory
__device__ __forceinline__ float to_f(float v) { return v; }
__device__ __forceinline__ float to_f(__nv_bfloat16 v) {
    return __uint_as_float(((uint32_t)__bfloat16_as_ushort(v)) << 16);
}
template <typename ST> __device__ __forceinline__ ST to_st(float v);
template <> __device__ __forceinline__ float to_st<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 to_st<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

template <int CG>
struct GroupGeom {
    static constexpr int NI = kGT / CG;              // tile elements per plane and thread: T*Lp / (CG*Lpad) <= T/CG
    static constexpr int NP_IN = 3 + 4 * CG;         // w3[3], lambda, x, u, dy
    static constexpr int NP_OUT = 3 + 2 * CG;        // dw3[3], dlambda, du
};

struct GroupBwdSmem {               // byte offsets inside dynamic shared memory
    uint32_t hall, dxs, tin, tout, line, gline, red, ptrs;
    uint32_t total;
    int Lpad;
};

template <typename ST, int CG>
__global__ void __launch_bounds__(kGroupMaxThreads, 1)
group_bwd_kernel(const BwdArgs<ST> a, const GroupBwdSmem L) {
    using Geo = GroupGeom<CG>;
    constexpr int NI = Geo::NI;
    extern __shared__ __align__(16) uint8_t smem[];
    const Shape sh = a.sh;
    const int H = sh.H, W = sh.W, plane = H * W, Lmax = sh.Lmax(), Lpad = L.Lpad;
    float* hall = reinterpret_cast<float*>(smem + L.hall);        // [CG][Ls*Lp]  h of the current direction
    float* dxs = reinterpret_cast<float*>(smem + L.dxs);          // [CG][H*W]    dx, image layout
    ST* tin = reinterpret_cast<ST*>(smem + L.tin);                // [NP_IN][T][Lmax]
    ST* tout = reinterpret_cast<ST*>(smem + L.tout);              // [NP_OUT][T][Lmax]
    float* line = reinterpret_cast<float*>(smem + L.line);        // [2][CG][Lmax+2]  h[s-1] / h[s], zero halo
    float* gline = reinterpret_cast<float*>(smem + L.gline);      // [CG][Lmax+2]     gh[s], zero halo
    float* red = reinterpret_cast<float*>(smem + L.red);          // [CG][3][Lmax]    dw3 terms of one step
    const ST** pin = reinterpret_cast<const ST**>(smem + L.ptrs);  // [NP_IN] operand planes of this direction
    ST** pout = reinterpret_cast<ST**>(smem + L.ptrs) + Geo::NP_IN; // [NP_OUT] (may hold nullptr)

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int c = tid / Lpad, p = tid % Lpad;
    const int b = blockIdx.x / sh.G, g = blockIdx.x % sh.G;
    const int ch0 = g * CG;                                       // first channel of the group (cg == CG)
    const int LW = Lmax + 2;

    for (int o = tid; o < CG * plane; o += nthr) dxs[o] = 0.f;

    int q = 0;
    for (int dir = 0; dir < 4; ++dir) {
        if (!(sh.mask >> dir & 1u)) continue;
        const int Ls = dir < 2 ? H : W, Lp = dir < 2 ? W : H;
        const bool act = p < Lp;
        const int TL = kGT * Lp;                                   // elements of one plane tile
        __syncthreads();                                           // previous direction done with pin/pout/line
        if (tid < Geo::NP_IN) {
            const size_t dbg = ((size_t)q * sh.B + b) * sh.G + g;
            const size_t dbc = ((size_t)q * sh.B + b) * sh.C + ch0;
            const size_t bc = (size_t)b * sh.C + ch0;
            const ST* ptr;
            if (tid < 3) ptr = a.w3 + (dbg * 3 + tid) * plane;
            else if (tid < 3 + CG) ptr = a.lam + (dbc + tid - 3) * plane;
            else if (tid < 3 + 2 * CG) ptr = a.x + (bc + tid - 3 - CG) * plane;
            else if (tid < 3 + 3 * CG) ptr = a.u + (dbc + tid - 3 - 2 * CG) * plane;
            else ptr = a.dy + (bc + tid - 3 - 3 * CG) * plane;
            pin[tid] = ptr;
        }
        if (tid < Geo::NP_OUT) {
            const size_t dbg = ((size_t)q * sh.B + b) * sh.G + g;
            const size_t dbc = ((size_t)q * sh.B + b) * sh.C + ch0;
            ST* ptr;
            if (tid < 3) ptr = a.dw3 ? a.dw3 + (dbg * 3 + tid) * plane : nullptr;
            else if (tid < 3 + CG) ptr = a.dlam ? a.dlam + (dbc + tid - 3) * plane : nullptr;
            else ptr = a.du ? a.du + (dbc + tid - 3 - CG) * plane : nullptr;
            pout[tid] = ptr;
        }
        for (int o = tid; o < 2 * CG * LW; o += nthr) line[o] = 0.f;
        for (int o = tid; o < CG * LW; o += nthr) gline[o] = 0.f;
        __syncthreads();
        const ST* h0p = a.h0 ? a.h0 + (((size_t)q * sh.B + b) * sh.C + ch0 + c) * Lmax : nullptr;
        if (act && h0p) line[c * LW + p + 1] = ld_f(h0p + p);

        // tile element e = tid + it*nthr of a plane <-> (t, pp): rows are contiguous for the vertical
        // directions, T-element row segments for the horizontal ones (coalesced either way)
        int et[NI], ep[NI];
        bool eok[NI];
#pragma unroll
        for (int it = 0; it < NI; ++it) {
            const int e = tid + it * nthr;
            eok[it] = e < TL;
            if (dir < 2) { et[it] = e / Lp; ep[it] = e % Lp; }
            else         { ep[it] = e / kGT; et[it] = e % kGT; }
        }
        // fetch the tile whose first step (in processing order) is s_first into registers
        auto fetch = [&](ST (&r)[Geo::NP_IN][NI], int np, int s_first, bool reverse) {
#pragma unroll
            for (int pl = 0; pl < Geo::NP_IN; ++pl) {
                if (pl < np) {
                    const ST* src = pin[pl];
#pragma unroll
                    for (int it = 0; it < NI; ++it) {
                        const int s = reverse ? s_first - et[it] : s_first + et[it];
                        if (eok[it] && s >= 0 && s < Ls) r[pl][it] = __ldg(src + img_off(dir, s, ep[it], H, W));
                    }
                }
            }
        };
        auto stash = [&](const ST (&r)[Geo::NP_IN][NI], int np) {      // registers -> tin[pl][t][pp]
#pragma unroll
            for (int pl = 0; pl < Geo::NP_IN; ++pl)
                if (pl < np) {
#pragma unroll
                    for (int it = 0; it < NI; ++it)
                        if (eok[it]) tin[(pl * kGT + et[it]) * Lmax + ep[it]] = r[pl][it];
                }
        };
        ST r[Geo::NP_IN][NI];

        // ================= sweep 1: h[s] for every step, kept in hall =================================
        {
            const int np1 = 3 + 2 * CG;
            float* cur = line;
            float* nxt = line + CG * LW;
            fetch(r, np1, 0, false);
            for (int s0 = 0; s0 < Ls; s0 += kGT) {
                stash(r, np1);
                __syncthreads();
                if (s0 + kGT < Ls) fetch(r, np1, s0 + kGT, false);
#pragma unroll 1
                for (int t = 0; t < kGT && s0 + t < Ls; ++t) {
                    if (act) {
                        const int to = t * Lmax + p;
                        float acc = to_f(tin[(3 + c) * kGT * Lmax + to]) * to_f(tin[(3 + CG + c) * kGT * Lmax + to]);
                        const float* hp = cur + c * LW + p;        // hp[0] = h[p-1], hp[1] = h[p], hp[2] = h[p+1]
                        if (p > 0)      acc = fmaf(to_f(tin[to]), hp[0], acc);
                        acc = fmaf(to_f(tin[kGT * Lmax + to]), hp[1], acc);
                        if (p < Lp - 1) acc = fmaf(to_f(tin[2 * kGT * Lmax + to]), hp[2], acc);
                        nxt[c * LW + p + 1] = acc;
                        hall[c * plane + (s0 + t) * Lp + p] = acc;
                    }
                    __syncthreads();
                    float* tmp = cur; cur = nxt; nxt = tmp;
                }
            }
        }
        // ================= sweep 2: reverse order ========================================================
        {
            const int np2 = Geo::NP_IN;
            float carry = 0.f;
            fetch(r, np2, Ls - 1, true);
            for (int s1 = Ls - 1; s1 >= 0; s1 -= kGT) {
                stash(r, np2);
                __syncthreads();
                if (s1 - kGT >= 0) fetch(r, np2, s1 - kGT, true);
#pragma unroll 1
                for (int t = 0; t < kGT && s1 - t >= 0; ++t) {
                    const int s = s1 - t;
                    if (act) {
                        const int to = t * Lmax + p;
                        const float gy = to_f(tin[(3 + 3 * CG + c) * kGT * Lmax + to]);
                        const float gh = fmaf(gy, to_f(tin[(3 + 2 * CG + c) * kGT * Lmax + to]), carry);
                        const float hs = hall[c * plane + s * Lp + p];
                        tout[(3 + CG + c) * kGT * Lmax + to] = to_st<ST>(gy * hs);                                  // du
                        tout[(3 + c) * kGT * Lmax + to] = to_st<ST>(to_f(tin[(3 + CG + c) * kGT * Lmax + to]) * gh);  // dlambda
                        const int o = img_off(dir, s, p, H, W);
                        dxs[c * plane + o] = fmaf(to_f(tin[(3 + c) * kGT * Lmax + to]), gh, dxs[c * plane + o]);
                        // dw3 terms gh * h[s-1, p+k-1]
                        float hm = 0.f, h0v = 0.f, hp1 = 0.f;
                        if (s > 0) {
                            const float* hr = hall + c * plane + (s - 1) * Lp + p;
                            if (p > 0) hm = hr[-1];
                            h0v = hr[0];
                            if (p < Lp - 1) hp1 = hr[1];
                        } else if (h0p) {
                            if (p > 0) hm = ld_f(h0p + p - 1);
                            h0v = ld_f(h0p + p);
                            if (p < Lp - 1) hp1 = ld_f(h0p + p + 1);
                        }
                        red[(c * 3 + 0) * Lmax + p] = gh * hm;
                        red[(c * 3 + 1) * Lmax + p] = gh * h0v;
                        red[(c * 3 + 2) * Lmax + p] = gh * hp1;
                        gline[c * LW + p + 1] = gh;
                    }
                    __syncthreads();
                    if (act) {
                        // carry = w[s]^T gh: position p receives from p-1 (its tap k=2), p (k=1), p+1 (k=0)
                        const int to = t * Lmax + p;
                        const float* gp = gline + c * LW + p;
                        float acc = 0.f;
                        if (p > 0)      acc = fmaf(to_f(tin[2 * kGT * Lmax + to - 1]), gp[0], acc);
                        acc = fmaf(to_f(tin[kGT * Lmax + to]), gp[1], acc);
                        if (p < Lp - 1) acc = fmaf(to_f(tin[to + 1]), gp[2], acc);
                        carry = acc;
                        // dw3[k] of this step: channels summed in ascending order by the thread of channel k
                        for (int k = c; k < 3; k += CG) {
                            float sum = 0.f;
#pragma unroll
                            for (int cc = 0; cc < CG; ++cc) sum += red[(cc * 3 + k) * Lmax + p];
                            tout[k * kGT * Lmax + to] = to_st<ST>(sum);
                        }
                    }
                    __syncthreads();
                }
                // outputs of this tile -> global, same coalesced mapping as the loads
#pragma unroll
                for (int pl = 0; pl < Geo::NP_OUT; ++pl) {
                    ST* dst = pout[pl];
                    if (dst) {
#pragma unroll
                        for (int it = 0; it < NI; ++it) {
                            const int s = s1 - et[it];
                            if (eok[it] && s >= 0)
                                dst[img_off(dir, s, ep[it], H, W)] = tout[(pl * kGT + et[it]) * Lmax + ep[it]];
                        }
                    }
                }
            }
            if (a.dh0) {
                ST* d0 = a.dh0 + (((size_t)q * sh.B + b) * sh.C + ch0 + c) * Lmax;
                if (act) st_f(d0 + p, carry);
                else if (c < CG && p < Lmax) st_f(d0 + p, 0.f);
            }
        }
        ++q;
    }
    __syncthreads();
    if (a.dx) {
        ST* dxp = a.dx + ((size_t)b * sh.C + ch0) * plane;
        for (int o = tid; o < CG * plane; o += nthr) st_f(dxp + o, dxs[o]);
    }
}


// ---- host side -----------------------------------------------------------------------------------
template <typename ST, int CG>
static int launch_group(const BwdArgs<ST>& a, cudaStream_t st) {
    using Geo = GroupGeom<CG>;
    const Shape& sh = a.sh;
    const int Lmax = sh.Lmax();
    GroupBwdSmem L{};
    L.Lpad = (Lmax + 31) / 32 * 32;
    const int threads = CG * L.Lpad;
    if (threads > kGroupMaxThreads) {
        set_error("fused bwd (group): %d channels x %d positions exceed %d threads", CG, L.Lpad, kGroupMaxThreads);
        return GSPN_EUNSUPPORTED;
    }
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off = (off + bytes + 15) / 16 * 16; return (uint32_t)o; };
    L.hall = take((size_t)CG * sh.plane() * 4);
    L.dxs = take((size_t)CG * sh.plane() * 4);
    L.tin = take((size_t)Geo::NP_IN * kGT * Lmax * sizeof(ST));
    L.tout = take((size_t)Geo::NP_OUT * kGT * Lmax * sizeof(ST));
    L.line = take((size_t)2 * CG * (Lmax + 2) * 4);
    L.gline = take((size_t)CG * (Lmax + 2) * 4);
    L.red = take((size_t)CG * 3 * Lmax * 4);
    L.ptrs = take((size_t)(Geo::NP_IN + Geo::NP_OUT) * sizeof(void*));
    L.total = (uint32_t)off;
    if (off > (size_t)kMaxSmemOptin) {
        set_error("fused bwd (group): %d channels of a %dx%d plane need %zu B of shared memory (> %d)", CG, sh.H, sh.W,
                  off, kMaxSmemOptin);
        return GSPN_EUNSUPPORTED;
    }
    auto kern = group_bwd_kernel<ST, CG>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) { set_error("fused bwd (group): cudaFuncSetAttribute(%zu B): %s", off, cudaGetErrorString(e)); return GSPN_ECUDA; }
    GSPN_LAUNCH(kern, sh.B * sh.G, threads, off, st, a, L);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("fused bwd (group): launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int fused_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    int rc;
    switch (a.sh.cg()) {
    case 1: rc = launch_group<ST, 1>(a, st); break;
    case 2: rc = launch_group<ST, 2>(a, st); break;
    case 4: rc = launch_group<ST, 4>(a, st); break;
    default:
        set_error("fused bwd (group): C/G = %d channels per group (supported: 1, 2, 4)", a.sh.cg());
        return GSPN_EUNSUPPORTED;
    }
    if (rc == GSPN_OK) { li->launches = 1; li->variant = "fused_bwd_group"; }
    return rc;
}

template int fused_bwd_launch<float>(const BwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int fused_bwd_launch<__nv_bfloat16>(const BwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
