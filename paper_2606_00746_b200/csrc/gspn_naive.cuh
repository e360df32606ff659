// gspn_naive.cuh -- device code of the naive kernels (see gspn_naive.cu for what they are for).  Kept in a header of its
// own so that the launchers (gspn_naive.cu) hold everything that needs the CUDA runtime: this file uses only what
// gspn_common.cuh declares, threadIdx / blockIdx / blockDim, __syncthreads and dynamic shared memory.
#pragma once

#include "gspn_common.cuh"

namespace gspn {

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
                               const ST* h0p, float* hbuf, float* hall, float* ysm, int H, int W, int Lc) {
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
                if (p > 0) w0[j] = ld_f(wp + o);
                w1[j] = ld_f(wp + plane + o);
                if (p < Lp - 1) w2[j] = ld_f(wp + 2 * plane + o);
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

template <typename ST>
__global__ void naive_fwd_kernel(FwdArgs<ST> a) {
    extern __shared__ float smem[];
    const Shape sh = a.sh;
    const int H = sh.H, W = sh.W, plane = H * W, Lmax = sh.Lmax();
    float* ysm = smem;
    float* hbuf = smem + plane;
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
                           a.h0 ? a.h0 + dbc * Lmax : nullptr, hbuf, nullptr, ysm, H, W, sh.band(dir < 2 ? H : W));
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
                               float* dxs, float* dws, ST* dlp, ST* dup, ST* dh0p, int H, int W, int Lc) {
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
                if (p > 0)      wl[j] = ld_f(wp + 2 * plane + img_off(dir, s, p - 1, H, W));
                wc[j] = ld_f(wp + plane + o);
                if (p < Lp - 1) wr[j] = ld_f(wp + img_off(dir, s, p + 1, H, W));
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
__global__ void naive_bwd_main_kernel(BwdArgs<ST> a) {
    extern __shared__ float smem[];
    const Shape sh = a.sh;
    const int H = sh.H, W = sh.W, plane = H * W, Lmax = sh.Lmax();
    float* hall = smem;
    float* dxs = smem + plane;
    float* hbuf = dxs + plane;
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
                           a.lam + in.l * plane, a.u + in.u * plane, h0p, hbuf, hall, nullptr, H, W, Lc);
        naive_pass_bwd<ST>(dir, a.x + (size_t)bc * plane, a.w3 + in.w * 3 * plane,
                           a.lam + in.l * plane, a.u + in.u * plane, h0p, a.dy + (size_t)bc * plane,
                           hall, ghs, a.dx ? dxs : nullptr, nullptr,
                           a.dlam ? a.dlam + dbc * plane : nullptr,
                           a.du ? a.du + dbc * plane : nullptr,
                           a.dh0 ? a.dh0 + dbc * Lmax : nullptr, H, W, Lc);
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
__global__ void naive_bwd_dw_kernel(BwdArgs<ST> a) {
    extern __shared__ float smem[];
    const Shape sh = a.sh;
    const int H = sh.H, W = sh.W, plane = H * W, Lmax = sh.Lmax(), cg = sh.cg();
    float* hall = smem;
    float* dws = smem + plane;
    float* hbuf = dws + 3 * plane;
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
                           a.u + in.u * plane, h0p, hbuf, hall, nullptr, H, W, Lc);
        naive_pass_bwd<ST>(dir, a.x + bc * plane, a.w3 + in.w * 3 * plane, a.lam + in.l * plane,
                           a.u + in.u * plane, h0p, a.dy + bc * plane, hall, ghs, nullptr, dws,
                           nullptr, nullptr, nullptr, H, W, Lc);
        __syncthreads();
    }
    ST* dwp = a.dw3 + dbg * 3 * plane;
    for (int o = threadIdx.x; o < 3 * plane; o += blockDim.x) st_f(dwp + o, dws[o]);
}

}  // namespace gspn
