/*
 * gspn_oracle.c -- plain, slow, obviously-correct CPU oracle for the GSPN 2D
 * line-scan propagation (arxiv/paper_2606_00746, "C-GSPN").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may build, link or call it.  It shares no code with the CUDA path under
 * paper_2606_00746_b200/csrc/ and neither includes the other.
 *
 * What it computes (the method is exact, so the oracle is the definition
 * written out):
 *   forward  h_i = w_i h_{i-1} + Diag(lambda_i) x_i        Eq. (1)/(5)
 *            y_i = u_i (.) h_i                               Eq. (2),
 *            tridiagonal w, three taps per pixel
 *            four directions, outputs summed                 PAPER.md:99, Eq. (9)
 *   backward the exact adjoint of the above (the paper reports backward
 *            timings only; derivation in gspn_oracle_impl.h)
 *   merge    y = sum_d m[d,c] * y_d                          Eq. (9)
 *   normalize w = sigmoid(wt) / sum_{N(j)} sigmoid(wt)        Eq. (3), PAPER.md:94-97 (and its adjoint)
 *
 * Precision: double ("truth").  A float build of the same loops, with fmaf in
 * one pinned order and -ffp-contract=off, exists as a diagnostic and as the
 * timed cpu_baseline; it is never the reference value of a parity test.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"):
 *   fwd : trinomial delta response (closed form), constant-row closed form,
 *         prefix-sum and first-order-IIR special cases (numpy cumsum /
 *         scipy.signal.lfilter), diagonal-shift orientation case, dense
 *         Eq. (4) matrix brute force on 4x4 and 3x5 grids,
 *         direction symmetries, group replication, stability bound
 *         (PAPER.md:94), linearity.
 *   bwd : central finite differences in fp64 for x, lambda, u, w3, h0,
 *         adjoint identity <scan(v),dy> = <v,dx>, dense-matrix transpose on
 *         4x4, group-sum identity for dw3.
 *   merge: numpy einsum on random data.
 *   normalize: rows sum to one, equal logits give 1/|N(j)|, softmax identity on two taps, scipy expit,
 *         finite differences and the adjoint identity for its backward, the clamp branch.
 * The paper prints no worked numeric example of Eq. (1), so there is no
 * paper-value fixture; every function above is pinned by the mathematics.
 *
 * Parallelism: an OpenMP "parallel for" over the independent (b, group) units
 * (each (chunk,b,c) slice is independent).  No blocking, no
 * SIMD intrinsics, no reordering.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define T double
#define FN(n) gspn_oracle_##n##_f64
#define FMA(a, b, c) ((a) * (b) + (c))
#include "gspn_oracle_impl.h"
#undef T
#undef FN
#undef FMA

#define T float
#define FN(n) gspn_oracle_##n##_f32
#define FMA(a, b, c) fmaf((a), (b), (c))
#include "gspn_oracle_impl.h"
#undef T
#undef FN
#undef FMA

/*
 * Merge of per-direction outputs (Eq. 9's Prop2D collects the four passes;
 * DESIGN.md reading R7): y[b,c,:,:] = sum_q m[q,c] * y_dirs[q,b,c,:,:],
 * q over the D slabs, m NULL = ones.
 */
int gspn_oracle_merge_f64(const double *y_dirs, const double *m, double *y,
                          int D, int B, int C, int H, int W)
{
    if (D < 1 || B < 1 || C < 1 || H < 1 || W < 1) return 1;
    const size_t plane = (size_t)H * W;
    for (int b = 0; b < B; ++b)
        for (int c = 0; c < C; ++c)
            for (size_t o = 0; o < plane; ++o) {
                double acc = 0.0;
                for (int q = 0; q < D; ++q)
                    acc += (m ? m[(size_t)q * C + c] : 1.0) *
                           y_dirs[(((size_t)q * B + b) * C + c) * plane + o];
                y[((size_t)b * C + c) * plane + o] = acc;
            }
    return 0;
}

/*
 * Row-stochastic normalisation of the raw tap logits, Eq. (3), in the order the paper's fused
 * kernel names ("sigmoid activation, local reduction, clamping, and division"):
 *     s_k   = 1 / (1 + exp(-wt_k))                       k = 0, 1, 2  (neighbour -1, 0, +1 on the cross axis)
 *     S     = sum over the taps k whose neighbour lies inside the grid (the set N(j) of Eq. 3)
 *     w_k   = s_k / max(S, eps)   for k in N(j),   0 for the out-of-grid taps
 * wt, w3: [D,B,G,3,H,W]; the cross axis is j for the vertical directions (mask bits 0, 1) and i for the
 * horizontal ones (bits 2, 3).  eps: the paper gives no clamp bound; reading R17 takes 1e-6.
 */
static int norm_valid(int dir, int k, int i, int j, int H, int W)
{
    const int p = dir < 2 ? j : i, L = dir < 2 ? W : H;      /* cross position and its extent */
    if (k == 0) return p > 0;
    if (k == 2) return p < L - 1;
    return 1;
}

int gspn_oracle_normalize_f64(const double *wt, double *w3, int B, int G, int H, int W,
                              unsigned mask, double eps)
{
    if (B < 1 || G < 1 || H < 1 || W < 1 || mask < 1 || mask > 15) return 1;
    const size_t plane = (size_t)H * W;
    int q = 0;
    for (int dir = 0; dir < 4; ++dir) {
        if (!(mask >> dir & 1u)) continue;
        for (int bg = 0; bg < B * G; ++bg) {
            const double *a = wt + ((size_t)q * B * G + bg) * 3 * plane;
            double *o = w3 + ((size_t)q * B * G + bg) * 3 * plane;
            for (int i = 0; i < H; ++i)
                for (int j = 0; j < W; ++j) {
                    double s[3], S = 0.0;
                    for (int k = 0; k < 3; ++k) {
                        s[k] = 1.0 / (1.0 + exp(-a[k * plane + (size_t)i * W + j]));
                        if (norm_valid(dir, k, i, j, H, W)) S += s[k];
                    }
                    const double Sc = S > eps ? S : eps;
                    for (int k = 0; k < 3; ++k)
                        o[k * plane + (size_t)i * W + j] = norm_valid(dir, k, i, j, H, W) ? s[k] / Sc : 0.0;
                }
        }
        ++q;
    }
    return 0;
}

/*
 * Adjoint of the above: dwt_k = s_k (1 - s_k) * dL/ds_k with, for k in N(j),
 *     dL/ds_k = (dw_k - sum_{k' in N(j)} dw_k' w_k') / S     where the clamp is inactive (S > eps)
 *     dL/ds_k = dw_k / eps                                    where it is active (the denominator is a constant)
 * and dwt_k = 0 for the out-of-grid taps (they do not reach any output).
 */
/* magnitude != 0: the sum of the absolute values of the terms instead (|dw| and a plus inside the bracket):
 * the scale rounding errors of dwt are relative to (tests/parity_util.py). */
int gspn_oracle_normalize_bwd_f64(const double *wt, const double *dw3, double *dwt, int B, int G, int H,
                                  int W, unsigned mask, double eps, int magnitude)
{
    if (B < 1 || G < 1 || H < 1 || W < 1 || mask < 1 || mask > 15) return 1;
    const size_t plane = (size_t)H * W;
    int q = 0;
    for (int dir = 0; dir < 4; ++dir) {
        if (!(mask >> dir & 1u)) continue;
        for (int bg = 0; bg < B * G; ++bg) {
            const size_t base = ((size_t)q * B * G + bg) * 3 * plane;
            for (int i = 0; i < H; ++i)
                for (int j = 0; j < W; ++j) {
                    const size_t o = base + (size_t)i * W + j;
                    double s[3], S = 0.0;
                    int v[3];
                    for (int k = 0; k < 3; ++k) {
                        s[k] = 1.0 / (1.0 + exp(-wt[o + k * plane]));
                        v[k] = norm_valid(dir, k, i, j, H, W);
                        if (v[k]) S += s[k];
                    }
                    double g[3];
                    for (int k = 0; k < 3; ++k) g[k] = magnitude ? fabs(dw3[o + k * plane]) : dw3[o + k * plane];
                    double dot = 0.0;                      /* sum_k' dw_k' w_k' over N(j) */
                    if (S > eps)
                        for (int k = 0; k < 3; ++k)
                            if (v[k]) dot += g[k] * (s[k] / S);
                    if (magnitude) dot = -dot;
                    for (int k = 0; k < 3; ++k) {
                        double ds = 0.0;
                        if (v[k]) ds = S > eps ? (g[k] - dot) / S : g[k] / eps;
                        dwt[o + k * plane] = s[k] * (1.0 - s[k]) * ds;
                    }
                }
        }
        ++q;
    }
    return 0;
}

/* threads the OpenMP loops above will use (1 when built without OpenMP) */
int gspn_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void gspn_oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
