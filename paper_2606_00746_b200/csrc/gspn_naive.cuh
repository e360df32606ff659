// gspn_naive.cuh -- device code of the naive kernels (see gspn_naive.cu for what they are for).  Kept in a header of its
// own so that the launchers (gspn_naive.cu) hold everything that needs the CUDA runtime: this file uses only what
// gspn_common.cuh declares, threadIdx / blockIdx / blockDim, __syncthreads and dynamic shared memory.
#pragma once

#include "gspn_common.cuh"

namespace gspn {

// ---- Eq. 3 in the load path (Shape::logits(); include/gspn.h gspn_normalize_fwd) --------------------
// s_k = sigmoid(l_k), S = sum over the taps whose neighbour is inside the grid, w_k = s_k / max(S, eps), 0 outside.
constexpr float kNormEps = 1e-6f;      // GSPN_NORM_EPS of include/gspn.h (reading R17)
struct Nrm3 {
    float s[3], oms[3], w[3], S;       // sigmoid, 1 - sigmoid (as e * s: no cancellation), normalised tap, in-grid sum
    bool v[3];
};
__device__ __forceinline__ Nrm3 nrm3(float l0, float l1, float l2, bool v0, bool v2) {
    Nrm3 r;
    const float l[3] = {l0, l1, l2};
    r.v[0] = v0; r.v[1] = true; r.v[2] = v2;
    r.S = 0.f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float e = expf(fminf(-l[k], 80.f));      // capped so that e stays finite: sigmoid(-80) = 1.8e-35 either way
        r.s[k] = 1.f / (1.f + e);
        r.oms[k] = e * r.s[k];
        if (r.v[k]) r.S += r.s[k];
    }
    const float Sc = r.S > kNormEps ? r.S : kNormEps;
#pragma unroll
    for (int k = 0; k < 3; ++k) r.w[k] = r.v[k] ? r.s[k] / Sc : 0.f;
    return r;
}

// the three taps of the pixel at plane offset o, cross position p: the stored values (0 for a tap whose neighbour lies
// outside the grid: it is never read), or Eq. 3 of the stored logits
template <typename ST>
__device__ __forceinline__ void load_taps(const ST* wp, int plane, int o, int p, int Lp, bool logits, float& w0, float& w1,
                                          float& w2) {
    w0 = p > 0 ? ld_f(wp + o) : 0.f;
    w1 = ld_f(wp + plane + o);
    w2 = p < Lp - 1 ? ld_f(wp + 2 * plane + o) : 0.f;
    if (logits) {
        const Nrm3 r = nrm3(w0, w1, w2, p > 0, p < Lp - 1);
        w0 = r.w[0]; w1 = r.w[1]; w2 = r.w[2];
    }
}

// one directional forward pass of one plane; every thread of the CTA must call it.
//   hbuf : 2*(Lmax+2) floats, line s-1 / line s with a zero halo at both ends
//   hall : NULL or [H*W] floats, receives every hidden state in image layout
//   ysm  : NULL or [H*W] floats, y += u*h
constexpr int kChunk = 8;      // scan steps whose operands a thread fetches together (one global latency per chunk)

//   Lc   : lines per band of the scan axis (chunked scan, Shape::band; Lc = Ls is the global scan)
// step s enters a band (the state of the line before counts as zero) when its line, in image coordinates, is a band's
// first line for the ascending directions (0, 2) and a band's last line for the descending ones (1, 3)
__device__ __forceinline__ bool band_entry(int dir, int s, int Ls, int Lc) {
    return s > 0 && ((dir & 1) ? (Ls - 1 - s) % Lc == Lc - 1 : s % Lc == 0);
}

template <typename ST>
__device__ void naive_pass_fwd(int dir, const ST* xp, const ST* wp, const ST* lp, const ST* up,
                               const ST* h0p, float* hbuf, float* hall, float* ysm, int H, int W, int Lc, bool logits) {
    const int Ls = dir < 2 ? H : W, Lp = dir < 2 ? W : H;
    const int Lmax = H > W ? H : W;
    const int plane = H * W;
    const int p = threadIdx.x;
    float* cur = hbuf;
    float* nxt = hbuf + (Lmax + 2);
    for (int t = p; t < Lmax + 2; t += blockDim.x) { cur[t] = 0.f; nxt[t] = 0.f; }
    __syncthreads();
    if (p < Lp && h0p) cur[p + 1] = ld_f(h0p + p);
    __syncthreads();
    for (int s0 = 0; s0 < Ls; s0 += kChunk) {
        // operands of steps s0 .. s0+kChunk-1 of this thread's position: all loads in flight at once
        float lx[kChunk], w0[kChunk], w1[kChunk], w2[kChunk], uu[kChunk];
#pragma unroll
        for (int j = 0; j < kChunk; ++j) {
            lx[j] = w0[j] = w1[j] = w2[j] = uu[j] = 0.f;
            if (p < Lp && s0 + j < Ls) {
                const int o = img_off(dir, s0 + j, p, H, W);
                lx[j] = ld_f(lp + o) * ld_f(xp + o);
                load_taps<ST>(wp, plane, o, p, Lp, logits, w0[j], w1[j], w2[j]);
                if (ysm) uu[j] = ld_f(up + o);
            }
        }
#pragma unroll
        for (int j = 0; j < kChunk; ++j) {
            const int s = s0 + j;
            if (s < Ls) {                                   // uniform over the CTA
                if (p < Lp) {
                    const int o = img_off(dir, s, p, H, W);
                    float acc = lx[j];
                    if (!band_entry(dir, s, Ls, Lc)) {
                        if (p > 0)      acc = fmaf(w0[j], cur[p], acc);
                        acc = fmaf(w1[j], cur[p + 1], acc);
                        if (p < Lp - 1) acc = fmaf(w2[j], cur[p + 2], acc);
                    }
                    nxt[p + 1] = acc;
                    if (hall) hall[o] = acc;
                    if (ysm) ysm[o] = fmaf(uu[j], acc, ysm[o]);
                }
                __syncthreads();
                float* t = cur; cur = nxt; nxt = t;
            }
        }
    }
}

// plane index of the INPUT operands of direction slab q: a shared operand (Shape::shared) has one slab, read by every
// direction; h0 and every output keep one slab per direction
struct SlabIn {
    size_t w, l, u;       // w3 plane triple, lambda plane, u plane
    __device__ SlabIn(const Shape& sh, int q, int b, int c, int g) {
        const size_t qw = sh.shared & kSharedW3 ? 0 : q, ql = sh.shared & kSharedLam ? 0 : q, qu = sh.shared & kSharedU ? 0 : q;
        w = (qw * sh.B + b) * sh.G + g;
        l = (ql * sh.B + b) * sh.C + c;
        u = (qu * sh.B + b) * sh.C + c;
    }
};

// (__launch_bounds__(1024): a block is as wide as the longest line, up to 1024 threads, so a thread may hold at most 64
// registers; without the bound ptxas takes 86-120 and a launch with more than 544-736 threads fails.)
// ws: NULL, or (large planes) global fp32 scratch that takes the place of the plane-sized shared-memory
// arrays -- one slice per CTA, touched by that CTA only, every access of one element separated from the next by a
// __syncthreads; shared memory then holds the two lines only
template <typename ST>
__global__ void __launch_bounds__(1024) naive_fwd_kernel(FwdArgs<ST> a, float* ws) {
    extern __shared__ float smem[];
    const Shape sh = a.sh;
    const int H = sh.H, W = sh.W, plane = H * W, Lmax = sh.Lmax();
    float* ysm = ws ? ws + (size_t)blockIdx.x * plane : smem;
    float* hbuf = ws ? smem : smem + plane;
    const int bc = blockIdx.x, b = bc / sh.C, c = bc % sh.C, g = c / sh.cg();
    for (int o = threadIdx.x; o < plane; o += blockDim.x) ysm[o] = 0.f;
    __syncthreads();
    int q = 0;
    for (int dir = 0; dir < 4; ++dir) {
        if (!(sh.mask >> dir & 1)) continue;
        const size_t dbc = ((size_t)q * sh.B + b) * sh.C + c;
        const SlabIn in(sh, q, b, c, g);
        naive_pass_fwd<ST>(dir, a.x + (size_t)bc * plane, a.w3 + in.w * 3 * plane,
                           a.lam + in.l * plane, a.u + in.u * plane,
                           a.h0 ? a.h0 + dbc * Lmax : nullptr, hbuf, nullptr, ysm, H, W, sh.band(dir < 2 ? H : W), sh.logits());
        ++q;
    }
    __syncthreads();
    ST* yp = a.y + (size_t)bc * plane;
    for (int o = threadIdx.x; o < plane; o += blockDim.x) st_f(yp + o, ysm[o]);
}

// reverse pass of one direction of one plane.  hall holds the forward states of this direction.
//   dxs  : NULL or [H*W] floats, dx += lambda*gh
//   dws  : NULL or [3*H*W] floats, dw_k += gh * h[s-1, p+k-1]
//   ghs  : Lmax+2 floats scratch
template <typename ST>
__device__ void naive_pass_bwd(int dir, const ST* xp, const ST* wp, const ST* lp, const ST* up,
                               const ST* h0p, const ST* gyp, const float* hall, float* ghs,
                               float* dxs, float* dws, ST* dlp, ST* dup, ST* dh0p, int H, int W, int Lc, bool logits) {
    const int Ls = dir < 2 ? H : W, Lp = dir < 2 ? W : H;
    const int Lmax = H > W ? H : W;
    const int plane = H * W;
    const int p = threadIdx.x;
    for (int t = p; t < Lmax + 2; t += blockDim.x) ghs[t] = 0.f;
    float carry = 0.f;
    __syncthreads();
    for (int s1 = Ls - 1; s1 >= 0; s1 -= kChunk) {
        // operands of steps s1, s1-1, .. s1-kChunk+1: all loads in flight at once
        float gyv[kChunk], uv[kChunk], lv[kChunk], xv[kChunk], wl[kChunk], wc[kChunk], wr[kChunk];
#pragma unroll
        for (int j = 0; j < kChunk; ++j) {
            gyv[j] = uv[j] = lv[j] = xv[j] = wl[j] = wc[j] = wr[j] = 0.f;
            const int s = s1 - j;
            if (p < Lp && s >= 0) {
                const int o = img_off(dir, s, p, H, W);
                gyv[j] = ld_f(gyp + o); uv[j] = ld_f(up + o);
                lv[j] = ld_f(lp + o);   xv[j] = ld_f(xp + o);
                // taps of the carry w[s]^T gh: position p receives from p-1 (its tap k=2), p (k=1), p+1 (k=0)
                if (!logits) {
                    if (p > 0)      wl[j] = ld_f(wp + 2 * plane + img_off(dir, s, p - 1, H, W));
                    wc[j] = ld_f(wp + plane + o);
                    if (p < Lp - 1) wr[j] = ld_f(wp + img_off(dir, s, p + 1, H, W));
                } else {            // each of the three taps belongs to another pixel: Eq. 3 of that pixel's logits
                    float t0, t1, t2;
                    if (p > 0) { load_taps<ST>(wp, plane, img_off(dir, s, p - 1, H, W), p - 1, Lp, true, t0, t1, t2); wl[j] = t2; }
                    load_taps<ST>(wp, plane, o, p, Lp, true, t0, t1, t2); wc[j] = t1;
                    if (p < Lp - 1) { load_taps<ST>(wp, plane, img_off(dir, s, p + 1, H, W), p + 1, Lp, true, t0, t1, t2); wr[j] = t0; }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < kChunk; ++j) {
            const int s = s1 - j;
            if (s >= 0) {                                   // uniform over the CTA
                if (p < Lp) {
                    const int o = img_off(dir, s, p, H, W);
                    const float gy = gyv[j];
                    const float gh = fmaf(gy, uv[j], carry);
                    if (dup) st_f(dup + o, gy * hall[o]);
                    if (dxs) dxs[o] = fmaf(lv[j], gh, dxs[o]);
                    if (dlp) st_f(dlp + o, xv[j] * gh);
                    if (dws && !band_entry(dir, s, Ls, Lc)) {      // a band's first step multiplies a zero state: no dw3 term
#pragma unroll
                        for (int k = 0; k < 3; ++k) {
                            const int pn = p + k - 1;
                            if (pn < 0 || pn >= Lp) continue;
                            float hp;
                            if (s > 0) hp = hall[img_off(dir, s - 1, pn, H, W)];
                            else       hp = h0p ? ld_f(h0p + pn) : 0.f;
                            dws[k * plane + o] = fmaf(gh, hp, dws[k * plane + o]);
                        }
                    }
                    ghs[p + 1] = gh;
                }
                __syncthreads();
                if (p < Lp) {
                    float acc = 0.f;
                    if (p > 0)      acc = fmaf(wl[j], ghs[p], acc);
                    acc = fmaf(wc[j], ghs[p + 1], acc);
                    if (p < Lp - 1) acc = fmaf(wr[j], ghs[p + 2], acc);
                    carry = band_entry(dir, s, Ls, Lc) ? 0.f : acc;      // nothing flows back across a band's first step
                }
                __syncthreads();
            }
        }
    }
    if (dh0p) {
        if (p < Lp) st_f(dh0p + p, carry);
        else if (p < Lmax) st_f(dh0p + p, 0.f);
    }
}

// grid B*C: dx (summed over directions on chip), dlambda, du, dh0
template <typename ST>
__global__ void __launch_bounds__(1024) naive_bwd_main_kernel(BwdArgs<ST> a, float* ws) {
    extern __shared__ float smem[];
    const Shape sh = a.sh;
    const int H = sh.H, W = sh.W, plane = H * W, Lmax = sh.Lmax();
    float* hall = ws ? ws + (size_t)blockIdx.x * 2 * plane : smem;
    float* dxs = hall + plane;
    float* hbuf = ws ? smem : dxs + plane;
    float* ghs = hbuf + 2 * (Lmax + 2);
    const int bc = blockIdx.x, b = bc / sh.C, c = bc % sh.C, g = c / sh.cg();
    for (int o = threadIdx.x; o < plane; o += blockDim.x) dxs[o] = 0.f;
    __syncthreads();
    int q = 0;
    for (int dir = 0; dir < 4; ++dir) {
        if (!(sh.mask >> dir & 1)) continue;
        const size_t dbc = ((size_t)q * sh.B + b) * sh.C + c;
        const SlabIn in(sh, q, b, c, g);
        const ST* h0p = a.h0 ? a.h0 + dbc * Lmax : nullptr;
        const int Lc = sh.band(dir < 2 ? H : W);
        naive_pass_fwd<ST>(dir, a.x + (size_t)bc * plane, a.w3 + in.w * 3 * plane,
                           a.lam + in.l * plane, a.u + in.u * plane, h0p, hbuf, hall, nullptr, H, W, Lc, sh.logits());
        naive_pass_bwd<ST>(dir, a.x + (size_t)bc * plane, a.w3 + in.w * 3 * plane,
                           a.lam + in.l * plane, a.u + in.u * plane, h0p, a.dy + (size_t)bc * plane,
                           hall, ghs, a.dx ? dxs : nullptr, nullptr,
                           a.dlam ? a.dlam + dbc * plane : nullptr,
                           a.du ? a.du + dbc * plane : nullptr,
                           a.dh0 ? a.dh0 + dbc * Lmax : nullptr, H, W, Lc, sh.logits());
        __syncthreads();
        ++q;
    }
    if (a.dx) {
        ST* dxp = a.dx + (size_t)bc * plane;
        for (int o = threadIdx.x; o < plane; o += blockDim.x) st_f(dxp + o, dxs[o]);
    }
}

// grid D*B*G: dw3 of one (direction slab, b, group), channels accumulated in ascending order
template <typename ST>
__global__ void __launch_bounds__(1024) naive_bwd_dw_kernel(BwdArgs<ST> a, float* ws) {
    extern __shared__ float smem[];
    const Shape sh = a.sh;
    const int H = sh.H, W = sh.W, plane = H * W, Lmax = sh.Lmax(), cg = sh.cg();
    float* hall = ws ? ws + (size_t)blockIdx.x * 4 * plane : smem;
    float* dws = hall + plane;
    float* hbuf = ws ? smem : dws + 3 * plane;
    float* ghs = hbuf + 2 * (Lmax + 2);
    const int q = blockIdx.x / (sh.B * sh.G);
    const int bg = blockIdx.x % (sh.B * sh.G), b = bg / sh.G, g = bg % sh.G;
    int dir = 0;
    for (int d = 0, qq = 0; d < 4; ++d)
        if (sh.mask >> d & 1) { if (qq == q) dir = d; ++qq; }
    for (int o = threadIdx.x; o < 3 * plane; o += blockDim.x) dws[o] = 0.f;
    __syncthreads();
    const size_t dbg = ((size_t)q * sh.B + b) * sh.G + g;
    const int Lc = sh.band(dir < 2 ? H : W);
    for (int cc = 0; cc < cg; ++cc) {
        const int c = g * cg + cc;
        const size_t bc = (size_t)b * sh.C + c;
        const size_t dbc = ((size_t)q * sh.B + b) * sh.C + c;
        const SlabIn in(sh, q, b, c, g);
        const ST* h0p = a.h0 ? a.h0 + dbc * Lmax : nullptr;
        naive_pass_fwd<ST>(dir, a.x + bc * plane, a.w3 + in.w * 3 * plane, a.lam + in.l * plane,
                           a.u + in.u * plane, h0p, hbuf, hall, nullptr, H, W, Lc, sh.logits());
        naive_pass_bwd<ST>(dir, a.x + bc * plane, a.w3 + in.w * 3 * plane, a.lam + in.l * plane,
                           a.u + in.u * plane, h0p, a.dy + bc * plane, hall, ghs, nullptr, dws,
                           nullptr, nullptr, nullptr, H, W, Lc, sh.logits());
        __syncthreads();
    }
    ST* dwp = a.dw3 + dbg * 3 * plane;
    if (!sh.logits()) {
        for (int o = threadIdx.x; o < 3 * plane; o += blockDim.x) st_f(dwp + o, dws[o]);
        return;
    }
    // Eq. 3's adjoint on chip (include/gspn.h gspn_normalize_bwd): dws holds the gradient of the normalised taps; what is
    // stored is the gradient of the logits:  dwt_k = s_k (1 - s_k) (dw_k - sum_{k' in N} dw_k' w_k') / S,  dw_k / eps
    // in place of the bracket over S where the clamp is active, 0 for the out-of-grid taps.
    const ST* wp = a.w3 + SlabIn(sh, q, b, g * cg, g).w * 3 * plane;
    const int Lp = dir < 2 ? W : H;
    for (int o = threadIdx.x; o < plane; o += blockDim.x) {
        const int p = dir < 2 ? o % W : o / W;
        const bool v0 = p > 0, v2 = p < Lp - 1;
        const Nrm3 r = nrm3(v0 ? ld_f(wp + o) : 0.f, ld_f(wp + plane + o), v2 ? ld_f(wp + 2 * plane + o) : 0.f, v0, v2);
        const float g3[3] = {dws[o], dws[plane + o], dws[2 * plane + o]};
        const bool clamped = !(r.S > kNormEps);
        float dot = 0.f;
        if (!clamped) {
#pragma unroll
            for (int k = 0; k < 3; ++k)
                if (r.v[k]) dot = fmaf(g3[k], r.w[k], dot);
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            float ds = 0.f;
            if (r.v[k]) ds = clamped ? g3[k] / kNormEps : (g3[k] - dot) / r.S;
            st_f(dwp + k * plane + o, r.s[k] * r.oms[k] * ds);
        }
    }
}

}  // namespace gspn
