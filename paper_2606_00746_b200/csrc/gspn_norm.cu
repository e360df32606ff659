// gspn_norm.cu -- fused row-stochastic normalisation of the raw tap logits (Eq. 3) and its
// adjoint: SURVEY.md 8 row f1.  One pass does what the paper's fused kernel does ("sigmoid
// activation, local reduction, clamping, and division"):
//     s_k = sigmoid(wt_k),  S = sum of s_k over the taps whose neighbour is inside the grid (N(j) of Eq. 3),
//     w_k = s_k / max(S, eps) for k in N(j), 0 for the out-of-grid taps.
// wt, w3: [D,B,G,3,H,W] in storage type ST, arithmetic in fp32, one RNE per output.  The cross axis (the one the
// three taps index) is j for T->B / B->T and i for L->R / R->L.
//
// HBM-bound elementwise work: every thread owns V consecutive pixels of one (direction, b, group) plane triple.
// V*sizeof(ST) = 16 bytes (vector loads / stores) when the planes are 16-byte aligned (H*W*sizeof(ST) % 16 == 0),
// else V = 1 (coalesced 2/4-byte accesses: planes of odd H*W in bf16 start at 2-byte phases, and the three taps
// of a pixel then sit at different phases, so no vector width fits all of them).
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

struct NormParams {
    const void *wt, *dw3;
    void* out;
    int H, W;
    unsigned HW, tiles, BG;               // tiles = CTAs per plane triple, BG = plane triples per direction slab
    unsigned long long magicW, magicT;    // ceil(2^64 / W), ceil(2^64 / tiles): n / d = umul64hi(n, magic) for n < 2^32
    unsigned dirs;                        // direction of slab q in bits [2q, 2q+2)
    float eps;
};

// n / d for a 32-bit n with magic = ceil(2^64 / d), d >= 2 (exact: the error term n*(d*magic - 2^64)/(d*2^64) < 2^-32)
__device__ __forceinline__ unsigned nrm_div(unsigned n, unsigned long long magic) {
    return (unsigned)__umul64hi((unsigned long long)n, magic);
}
__device__ __forceinline__ float nrm_ex2(float v) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}
// a = 1 + exp(-v) with the exponent capped at `cap` (in units of log2: cap * log2(e))
__device__ __forceinline__ float nrm_one_plus_exp_neg(float v, float cap_log2) {
    return 1.f + nrm_ex2(fminf(v * -1.4426950408889634f, cap_log2));
}
__device__ __forceinline__ float nrm_rcp(float v) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}
// s = sigmoid(v) and 1 - s = e*s with e = exp(-v) (no cancellation for large v; the argument is capped so
// that e stays finite: sigmoid(-80) = 1.8e-35 either way)
__device__ __forceinline__ float nrm_sigmoid(float v, float& one_minus_s) {
    const float e = nrm_ex2(fminf(v * -1.4426950408889634f, 115.41560327f));       // exp(min(-v, 80))
    const float s = nrm_rcp(1.f + e);
    one_minus_s = e * s;
    return s;
}

template <typename ST, int V> struct NrmVec;
template <> struct NrmVec<float, 1> {
    static __device__ __forceinline__ void ld(const float* p, float (&f)[1]) { f[0] = __ldg(p); }
    static __device__ __forceinline__ void st(float* p, const float (&f)[1]) { *p = f[0]; }
};
template <> struct NrmVec<float, 4> {
    static __device__ __forceinline__ void ld(const float* p, float (&f)[4]) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(p));
        f[0] = v.x; f[1] = v.y; f[2] = v.z; f[3] = v.w;
    }
    static __device__ __forceinline__ void st(float* p, const float (&f)[4]) {
        *reinterpret_cast<float4*>(p) = make_float4(f[0], f[1], f[2], f[3]);
    }
};
template <> struct NrmVec<__nv_bfloat16, 1> {
    static __device__ __forceinline__ void ld(const __nv_bfloat16* p, float (&f)[1]) { f[0] = ld_f(p); }
    static __device__ __forceinline__ void st(__nv_bfloat16* p, const float (&f)[1]) { *p = __float2bfloat16_rn(f[0]); }
};
template <> struct NrmVec<__nv_bfloat16, 8> {
    static __device__ __forceinline__ void ld(const __nv_bfloat16* p, float (&f)[8]) {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
        const uint32_t r[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            f[2 * t] = __uint_as_float(r[t] << 16);
            f[2 * t + 1] = __uint_as_float(r[t] & 0xffff0000u);
        }
    }
    static __device__ __forceinline__ void st(__nv_bfloat16* p, const float (&f)[8]) {
        uint32_t r[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * t], f[2 * t + 1]);
            r[t] = *reinterpret_cast<uint32_t*>(&h);
        }
        *reinterpret_cast<uint4*>(p) = make_uint4(r[0], r[1], r[2], r[3]);
    }
};

// BWD = false: out = w3 = Eq. 3 of wt.  BWD = true: out = dwt, the adjoint at wt applied to dw3:
//   dwt_k = s_k (1 - s_k) * (dw_k - sum_{k' in N} dw_k' w_k') / S   (clamp inactive; dw_k / eps where S <= eps)
// A thread owns PPT groups of V consecutive pixels, 256*V pixels apart (the scalar path amortises its index and
// address arithmetic over PPT = 4 pixels; all loads are issued before the first store).
template <typename ST, int V, int PPT, bool BWD>
__global__ void __launch_bounds__(256)
norm_kernel(const NormParams p) {
    // grid: x = (b, g) plane triple * tiles + tile, y = direction slab q
    const unsigned bg = p.tiles > 1 ? nrm_div(blockIdx.x, p.magicT) : blockIdx.x;
    const unsigned pfirst = ((blockIdx.x - bg * p.tiles) * (256u * PPT) + threadIdx.x) * V;
    if (pfirst >= p.HW) return;
    const int dir = (p.dirs >> (2 * blockIdx.y)) & 3u;
    const size_t base = ((size_t)blockIdx.y * p.BG + bg) * 3 * p.HW + pfirst;
    const ST* __restrict__ wtp = reinterpret_cast<const ST*>(p.wt) + base;
    const ST* __restrict__ dwp = reinterpret_cast<const ST*>(p.dw3) + base;
    ST* __restrict__ outp = reinterpret_cast<ST*>(p.out) + base;
    const unsigned W = (unsigned)p.W;
    const unsigned Lm1 = dir < 2 ? W - 1 : (unsigned)p.H - 1;

    float aa[PPT][3][V], gg[PPT][3][V];
#pragma unroll
    for (int m = 0; m < PPT; ++m)
        if (pfirst + m * 256u * V < p.HW) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                NrmVec<ST, V>::ld(wtp + (size_t)k * p.HW + m * 256u * V, aa[m][k]);
                if constexpr (BWD) NrmVec<ST, V>::ld(dwp + (size_t)k * p.HW + m * 256u * V, gg[m][k]);
            }
        }
#pragma unroll
    for (int m = 0; m < PPT; ++m) {
    const unsigned p0 = pfirst + m * 256u * V;
    if (p0 >= p.HW) break;
    float (&a)[3][V] = aa[m];
    float (&g)[3][V] = gg[m];
    ST* out = outp + m * 256u * V;
    // cross position of the first pixel: j for the vertical directions, i for the horizontal ones
    unsigned i = W > 1 ? nrm_div(p0, p.magicW) : p0;
    unsigned j = p0 - i * W;
    float o[3][V];
#pragma unroll
    for (int t = 0; t < V; ++t) {
        const unsigned pos = dir < 2 ? j : i;
        const bool v0 = pos != 0, v2 = pos != Lm1;
        if constexpr (!BWD) {
            // One reciprocal instead of four: with a_k = 1 + exp(-wt_k) = 1/s_k,
            //   w_k = s_k / S = (product of the other two a) / (a1 a2 [k=0 in N] + a0 a2 + a0 a1 [k=2 in N]).
            // exp's argument is capped at 43 so the products stay finite (a tap below sigmoid(-43) = 2e-19 then
            // errs by < 1e-13 absolutely).  Valid where the clamp cannot bind: a_1 <= 3e5 gives S >= s_1 >= 3.3e-6
            // > eps; the other pixels take the literal sigmoid / sum / clamp / divide path below.
            constexpr float kCap = 62.0358872f;                                     // 43 * log2(e)
            const float a0 = nrm_one_plus_exp_neg(a[0][t], kCap), a1 = nrm_one_plus_exp_neg(a[1][t], kCap),
                        a2 = nrm_one_plus_exp_neg(a[2][t], kCap);
            if (a1 <= 3e5f) {                                                      // the centre tap is always in N(j)
                const float t0 = v0 ? a1 * a2 : 0.f, t2 = v2 ? a0 * a1 : 0.f, t1 = a0 * a2;
                const float r = nrm_rcp(t0 + t1 + t2);
                o[0][t] = t0 * r; o[1][t] = t1 * r; o[2][t] = t2 * r;
                if (++j == W) { j = 0; ++i; }
                continue;
            }
        }
        float c0, c1, c2;                                       // 1 - s_k
        const float s0 = nrm_sigmoid(a[0][t], c0), s1 = nrm_sigmoid(a[1][t], c1), s2 = nrm_sigmoid(a[2][t], c2);
        const float S = (v0 ? s0 : 0.f) + s1 + (v2 ? s2 : 0.f);
        const bool clamped = !(S > p.eps);
        const float rS = nrm_rcp(clamped ? p.eps : S);
        if constexpr (!BWD) {
            o[0][t] = v0 ? s0 * rS : 0.f;
            o[1][t] = s1 * rS;
            o[2][t] = v2 ? s2 * rS : 0.f;
        } else {
            float dot = 0.f;
            if (!clamped) {
                dot = g[1][t] * (s1 * rS);
                if (v0) dot = fmaf(g[0][t], s0 * rS, dot);
                if (v2) dot = fmaf(g[2][t], s2 * rS, dot);
            }
            o[0][t] = v0 ? s0 * c0 * ((g[0][t] - dot) * rS) : 0.f;
            o[1][t] = s1 * c1 * ((g[1][t] - dot) * rS);
            o[2][t] = v2 ? s2 * c2 * ((g[2][t] - dot) * rS) : 0.f;
        }
        if (++j == W) { j = 0; ++i; }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) NrmVec<ST, V>::st(out + (size_t)k * p.HW, o[k]);
    }
}

// ---- host side -----------------------------------------------------------------------------------
template <typename ST, int V, bool BWD>
static int launch_norm(NormParams prm, int D, int BG, cudaStream_t st) {
    constexpr int PPT = V == 1 ? 4 : 1;
    const unsigned per_cta = 256u * V * PPT;
    prm.tiles = (prm.HW + per_cta - 1) / per_cta;
    prm.magicT = prm.tiles > 1 ? ~0ull / prm.tiles + 1 : 0;
    prm.BG = (unsigned)BG;
    const unsigned long long ctas = (unsigned long long)prm.tiles * (unsigned)BG;
    if (ctas > 0x7fffffffull) { set_error("normalize: %llu CTAs exceed the grid limit", ctas); return GSPN_EUNSUPPORTED; }
    norm_kernel<ST, V, PPT, BWD><<<dim3((unsigned)ctas, (unsigned)D), 256, 0, st>>>(prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("normalize: launch failed: %s", cudaGetErrorString(e)); return GSPN_ECUDA; }
    return GSPN_OK;
}

template <typename ST>
int norm_launch(const ST* wt, const ST* dw3, ST* out, int B, int G, int H, int W, unsigned mask,
                cudaStream_t st, LaunchInfo* li) {
    constexpr int ES = sizeof(ST), VV = 16 / ES;
    NormParams prm{};
    prm.wt = wt; prm.dw3 = dw3; prm.out = out;
    prm.H = H; prm.W = W; prm.HW = (unsigned)H * (unsigned)W;
    prm.eps = GSPN_NORM_EPS;
    prm.magicW = W > 1 ? ~0ull / (unsigned)W + 1 : 0;
    int D = 0;
    for (int d = 0; d < 4; ++d) if (mask >> d & 1u) prm.dirs |= (unsigned)d << (2 * D++);
    const bool vec = ((size_t)H * W * ES) % 16 == 0;
    int rc;
    if (dw3) rc = vec ? launch_norm<ST, VV, true>(prm, D, B * G, st) : launch_norm<ST, 1, true>(prm, D, B * G, st);
    else     rc = vec ? launch_norm<ST, VV, false>(prm, D, B * G, st) : launch_norm<ST, 1, false>(prm, D, B * G, st);
    if (rc == GSPN_OK) {
        li->launches = 1;
        li->variant = dw3 ? (vec ? "normalize_bwd_vec" : "normalize_bwd_scalar") : (vec ? "normalize_fwd_vec" : "normalize_fwd_scalar");
    }
    return rc;
}

template int norm_launch<float>(const float*, const float*, float*, int, int, int, int, unsigned, cudaStream_t, LaunchInfo*);
template int norm_launch<__nv_bfloat16>(const __nv_bfloat16*, const __nv_bfloat16*, __nv_bfloat16*, int, int, int, int, unsigned,
                                        cudaStream_t, LaunchInfo*);

}  // namespace gspn
