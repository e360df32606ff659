/*
 * gspn_oracle_impl.h -- body of the CPU oracle, included once per precision.
 *
 * TEST INFRASTRUCTURE ONLY.  See gspn_oracle.c for the header comment that
 * states who may call this and what it is pinned against.
 *
 * The including file defines
 *     T        the arithmetic type (double or float)
 *     FN(name) the name-mangling macro (gspn_oracle_<name>_f64 / _f32)
 *     FMA(a,b,c) a*b+c in T (plain expression for double; fmaf for float so
 *              that the float build has one pinned rounding order)
 *
 * Notation follows PAPER.md Sec. 3: x, lambda, u are
 * [B,C,H,W]; w is the row-stochastic tridiagonal matrix of Eq. (1)/(5), stored
 * as its three non-zero diagonals w3[.,k,i,j], k=0,1,2 <-> neighbour offset
 * -1,0,+1 along the NON-scan axis ("top-left, top-center, top-right",
 * PAPER.md:99).  One w per channel group g = c / (C/G) (Eq. 5, PAPER.md:131-134;
 * G=C gives Eq. 1's per-channel w, G=1 the paper's fully shared w).
 *
 * A direction is described by where scan step s and cross position p sit in
 * the image ("four complementary directional passes"):
 *     T->B : (i,j) = (s, p)        Ls = H, Lp = W
 *     B->T : (i,j) = (H-1-s, p)    Ls = H, Lp = W
 *     L->R : (i,j) = (p, s)        Ls = W, Lp = H
 *     R->L : (i,j) = (p, W-1-s)    Ls = W, Lp = H
 * Everything is evaluated in image coordinates; no tensor is flipped,
 * transposed or copied.
 */

/* image offset (within one [H,W] plane) of scan step s, cross position p */
static inline size_t FN(img)(int dir, int s, int p, int H, int W)
{
    switch (dir) {
    case 0:  return (size_t)s * W + p;               /* T->B */
    case 1:  return (size_t)(H - 1 - s) * W + p;     /* B->T */
    case 2:  return (size_t)p * W + s;               /* L->R */
    default: return (size_t)p * W + (W - 1 - s);     /* R->L */
    }
}

/*
 * One directional pass of Eq. (1)-(2) for one (b,c) plane.
 *   xp, lp, up : the plane's x, lambda_d, u_d          [H,W]
 *   wp         : the group's three tap planes of dir d [3,H,W]
 *   h0p        : initial state h_{-1}[p] (NULL = zeros; reading R1)
 *   hall       : out, every hidden state, indexed like the image [H,W]
 *   yp         : in/out, y += u_d * h_d   (Eq. 2 then the sum of Eq. 9's
 *                Prop2D over directions, reading R7)
 */
static void FN(pass_fwd)(int dir, const T *xp, const T *wp, const T *lp,
                         const T *up, const T *h0p, T *hall, T *yp,
                         int H, int W)
{
    const int Ls = (dir < 2) ? H : W;
    const int Lp = (dir < 2) ? W : H;
    const size_t plane = (size_t)H * W;
    T *hprev = (T *)malloc(sizeof(T) * (size_t)Lp);
    T *hcur = (T *)malloc(sizeof(T) * (size_t)Lp);
    for (int p = 0; p < Lp; ++p) hprev[p] = h0p ? h0p[p] : (T)0;
    for (int s = 0; s < Ls; ++s) {
        for (int p = 0; p < Lp; ++p) {
            const size_t o = FN(img)(dir, s, p, H, W);
            const T l = (p > 0) ? hprev[p - 1] : (T)0;      /* out-of-grid h = 0 */
            const T m = hprev[p];
            const T r = (p < Lp - 1) ? hprev[p + 1] : (T)0;
            T acc = lp[o] * xp[o];                          /* Diag(lambda) x   */
            if (p > 0)      acc = FMA(wp[0 * plane + o], l, acc);
            acc = FMA(wp[1 * plane + o], m, acc);
            if (p < Lp - 1) acc = FMA(wp[2 * plane + o], r, acc);
            hcur[p] = acc;                                  /* Eq. (1)          */
        }
        for (int p = 0; p < Lp; ++p) {
            const size_t o = FN(img)(dir, s, p, H, W);
            hall[o] = hcur[p];
            yp[o] = FMA(up[o], hcur[p], yp[o]);             /* Eq. (2), summed  */
            hprev[p] = hcur[p];
        }
    }
    free(hprev);
    free(hcur);
}

/*
 * Forward: y[b,c] = sum_{d in mask} u_d * scan_d(x)   in the fixed order
 * T->B, B->T, L->R, R->L.
 *   x [B,C,H,W]; w3 [D,B,G,3,H,W]; lambda,u [D,B,C,H,W];
 *   h0 NULL or [D,B,C,Lmax], Lmax = max(H,W) (first Lp entries used);
 *   y [B,C,H,W]; hsave NULL or [D,B,C,H,W].
 *   D = popcount(mask), slabs in ascending bit order.
 */
int FN(fwd)(const T *x, const T *w3, const T *lambda, const T *u, const T *h0,
            T *y, T *hsave, int B, int C, int H, int W, int G, unsigned mask)
{
    if (B < 1 || C < 1 || H < 1 || W < 1 || G < 1 || C % G || mask < 1 || mask > 15)
        return 1;
    const int cg = C / G;
    const int Lmax = H > W ? H : W;
    const size_t plane = (size_t)H * W;
    const long units = (long)B * G;
#pragma omp parallel for schedule(static)
    for (long ug = 0; ug < units; ++ug) {
        const int b = (int)(ug / G), g = (int)(ug % G);
        T *hall = (T *)malloc(sizeof(T) * plane);
        for (int cc = 0; cc < cg; ++cc) {
            const int c = g * cg + cc;
            const size_t bc = (size_t)b * C + c;
            T *yp = y + bc * plane;
            for (size_t o = 0; o < plane; ++o) yp[o] = (T)0;
            int q = 0;                                  /* slab index of dir */
            for (int dir = 0; dir < 4; ++dir) {
                if (!(mask >> dir & 1)) continue;
                const size_t dbc = ((size_t)q * B + b) * C + c;
                const size_t dbg = ((size_t)q * B + b) * G + g;
                FN(pass_fwd)(dir, x + bc * plane, w3 + dbg * 3 * plane,
                             lambda + dbc * plane, u + dbc * plane,
                             h0 ? h0 + dbc * Lmax : NULL,
                             hsave ? hsave + dbc * plane : hall, yp, H, W);
                ++q;
            }
        }
        free(hall);
    }
    return 0;
}

/*
 * Adjoint of one directional pass (reading R9; derived from
 * Eq. 1-2, the paper gives timings only).
 * With gy = dL/dy and h the states of the forward pass:
 *   gh[s]      = gy[s]*u[s] + w[s+1]^T gh[s+1]          (reverse recurrence)
 *   du[s]      = gy[s]*h[s]
 *   dlambda[s] = x[s]*gh[s]
 *   dx[s]     += lambda[s]*gh[s]                         (x shared by all dirs)
 *   dw_k[s][p]+= gh[s][p]*h[s-1][p+k-1]                  (summed over the group)
 *   dh0        = w[0]^T gh[0]
 */
static void FN(pass_bwd)(int dir, const T *xp, const T *wp, const T *lp,
                         const T *up, const T *h0p, const T *hall,
                         const T *gyp, T *dxp, T *dlp, T *dup, T *dwp,
                         T *dh0p, int H, int W)
{
    const int Ls = (dir < 2) ? H : W;
    const int Lp = (dir < 2) ? W : H;
    const size_t plane = (size_t)H * W;
    T *carry = (T *)malloc(sizeof(T) * (size_t)Lp);
    T *gh = (T *)malloc(sizeof(T) * (size_t)Lp);
    for (int p = 0; p < Lp; ++p) carry[p] = (T)0;
    for (int s = Ls - 1; s >= 0; --s) {
        for (int p = 0; p < Lp; ++p) {
            const size_t o = FN(img)(dir, s, p, H, W);
            gh[p] = FMA(gyp[o], up[o], carry[p]);
            dup[o] = gyp[o] * hall[o];
            dxp[o] = FMA(lp[o], gh[p], dxp[o]);
            dlp[o] = xp[o] * gh[p];
        }
        for (int p = 0; p < Lp; ++p) {
            const size_t o = FN(img)(dir, s, p, H, W);
            for (int k = 0; k < 3; ++k) {
                const int pn = p + k - 1;               /* neighbour in previous step */
                if (pn < 0 || pn >= Lp) continue;
                T hp;
                if (s > 0) hp = hall[FN(img)(dir, s - 1, pn, H, W)];
                else       hp = h0p ? h0p[pn] : (T)0;
                dwp[(size_t)k * plane + o] = FMA(gh[p], hp, dwp[(size_t)k * plane + o]);
            }
        }
        /* carry = w[s]^T gh : position q receives from p=q+1 (its k=0 tap),
         * p=q (k=1) and p=q-1 (k=2). */
        for (int qq = 0; qq < Lp; ++qq) {
            T acc = (T)0;
            if (qq > 0)
                acc = FMA(wp[2 * plane + FN(img)(dir, s, qq - 1, H, W)], gh[qq - 1], acc);
            acc = FMA(wp[1 * plane + FN(img)(dir, s, qq, H, W)], gh[qq], acc);
            if (qq < Lp - 1)
                acc = FMA(wp[0 * plane + FN(img)(dir, s, qq + 1, H, W)], gh[qq + 1], acc);
            carry[qq] = acc;
        }
    }
    if (dh0p) for (int p = 0; p < Lp; ++p) dh0p[p] = carry[p];
    free(carry);
    free(gh);
}

/*
 * Backward.  Inputs as in fwd plus dy [B,C,H,W].  Outputs (all required,
 * all fully overwritten): dx [B,C,H,W]; dlambda, du [D,B,C,H,W];
 * dw3 [D,B,G,3,H,W] (sum over the C/G channels of the group, channel order
 * ascending); dh0 [D,B,C,Lmax] (entries >= Lp set to 0).
 */
int FN(bwd)(const T *x, const T *w3, const T *lambda, const T *u, const T *h0,
            const T *dy, T *dx, T *dlambda, T *du, T *dw3, T *dh0,
            int B, int C, int H, int W, int G, unsigned mask)
{
    if (B < 1 || C < 1 || H < 1 || W < 1 || G < 1 || C % G || mask < 1 || mask > 15)
        return 1;
    const int cg = C / G;
    const int Lmax = H > W ? H : W;
    const size_t plane = (size_t)H * W;
    const long units = (long)B * G;
#pragma omp parallel for schedule(static)
    for (long ug = 0; ug < units; ++ug) {
        const int b = (int)(ug / G), g = (int)(ug % G);
        T *hall = (T *)malloc(sizeof(T) * plane);
        T *ytmp = (T *)malloc(sizeof(T) * plane);
        int q = 0;
        for (int cc = 0; cc < cg; ++cc) {
            const size_t bc = (size_t)b * C + (size_t)g * cg + cc;
            for (size_t o = 0; o < plane; ++o) dx[bc * plane + o] = (T)0;
        }
        for (int dir = 0; dir < 4; ++dir) {
            if (!(mask >> dir & 1)) continue;
            const size_t dbg = ((size_t)q * B + b) * G + g;
            T *dwp = dw3 + dbg * 3 * plane;
            for (size_t o = 0; o < 3 * plane; ++o) dwp[o] = (T)0;
            for (int cc = 0; cc < cg; ++cc) {
                const int c = g * cg + cc;
                const size_t bc = (size_t)b * C + c;
                const size_t dbc = ((size_t)q * B + b) * C + c;
                const T *h0p = h0 ? h0 + dbc * Lmax : NULL;
                for (size_t o = 0; o < plane; ++o) ytmp[o] = (T)0;
                FN(pass_fwd)(dir, x + bc * plane, w3 + dbg * 3 * plane,
                             lambda + dbc * plane, u + dbc * plane, h0p, hall,
                             ytmp, H, W);
                for (int p = 0; p < Lmax; ++p) dh0[dbc * Lmax + p] = (T)0;
                FN(pass_bwd)(dir, x + bc * plane, w3 + dbg * 3 * plane,
                             lambda + dbc * plane, u + dbc * plane, h0p, hall,
                             dy + bc * plane, dx + bc * plane,
                             dlambda + dbc * plane, du + dbc * plane, dwp,
                             dh0 + dbc * Lmax, H, W);
            }
            ++q;
        }
        free(hall);
        free(ytmp);
    }
    return 0;
}
