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
