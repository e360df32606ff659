/*
 * gspn.h -- C ABI of libgspn: the GSPN 2D line-scan linear propagation
 * (arxiv/paper_2606_00746, "C-GSPN"), hand-written for NVIDIA B200 (sm_100a).
 *
 * The operator (Sec. 3, lines 82-99; Sec. 4.2 Eq. 5;
 * Eq. 9).  For every direction d in dir_mask, every image b,
 * every channel c with weight group g = c / (C/G):
 *
 *     h_d[s, p] = w3_d[g,0,s,p] * h_d[s-1, p-1]
 *               + w3_d[g,1,s,p] * h_d[s-1, p  ]
 *               + w3_d[g,2,s,p] * h_d[s-1, p+1]
 *               + lambda_d[c,s,p] * x[c,s,p]                  (Eq. 1 / Eq. 5)
 *     y[c]      = sum_d  u_d[c] (.) h_d[c]                    (Eq. 2, merged as in Eq. 9)
 *
 * where s is the scan step and p the position across the scan line:
 *     T->B : (i,j) = (s, p)            B->T : (i,j) = (H-1-s, p)
 *     L->R : (i,j) = (p, s)            R->L : (i,j) = (p, W-1-s)
 * Out-of-grid neighbours contribute 0 and their tap is never read.  h_d[-1] is
 * h0 (zeros when NULL).  Tap k = 0,1,2 is the neighbour at offset -1,0,+1 along
 * the NON-scan axis ("top-left, top-center, top-right").
 * Accumulation is always fp32; the hidden state h is never rounded to the
 * storage type; every output element is rounded once (RNE) when stored.
 *
 * Layouts (all dense, C-contiguous, image layout, D = popcount(dir_mask),
 * direction slabs in ascending bit order, Lmax = max(H,W)):
 *     x, y, dy, dx            [B, C, H, W]
 *     lambda, u, dlambda, du  [D, B, C, H, W]
 *     w3, dw3                 [D, B, G, 3, H, W]
 *     h0, dh0                 [D, B, C, Lmax]   (first Lp entries used; dh0's
 *                                               remaining entries are written 0)
 *     y_dirs (gspn_merge)     [D, B, C, H, W];  m [D, C] fp32
 *
 * Pointers and ownership.  Every pointer of the *device* entry points is a
 * DEVICE pointer owned by the caller; the library never allocates, frees or
 * retains device memory in those calls and keeps no state between calls.
 * `stream` is a cudaStream_t (NULL = the legacy default stream); the calls
 * enqueue work on it and return without synchronising.  Outputs are fully
 * overwritten, never accumulated into, and must not alias any input.  Base
 * pointers must be 16-byte aligned (GSPN_EALIGN otherwise).  The *_host entry
 * points take HOST pointers with the same layouts; they stage through device
 * memory obtained from the stream-ordered allocator, copy in, run the device
 * entry point, copy out, and synchronise the stream before returning.
 *
 * Errors.  Every call returns a status code, never throws, never exits.
 * gspn_last_error() returns a thread-local, NUL-terminated description of the
 * last non-OK status on the calling thread.
 *     GSPN_EINVAL        bad shape (B,C,H,W,G < 1, C % G != 0), dir_mask not in
 *                        [1,15], unknown dtype, NULL required pointer
 *     GSPN_EUNSUPPORTED  a line longer than 1024 positions (max(H,W) > 1024); a forced
 *                        kernel (gspn_args_t.impl) that does not hold the shape or option
 *     GSPN_EWORKSPACE    a plane whose fp32 accumulators exceed one SM's shared memory
 *                        needs gspn_args_t.workspace (gspn_workspace_bytes), which is
 *                        missing or too small; the plain calls pass none
 *     GSPN_EALIGN        a base pointer is not 16-byte aligned
 *     GSPN_ECUDA         a CUDA runtime call or launch failed
 * There is no CPU fallback: without a CUDA device every compute entry point
 * returns GSPN_ECUDA.
 */
#ifndef GSPN_H_
#define GSPN_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { GSPN_DIR_TB = 1, GSPN_DIR_BT = 2, GSPN_DIR_LR = 4, GSPN_DIR_RL = 8, GSPN_DIR_ALL = 15 };
enum { GSPN_F32 = 0, GSPN_BF16 = 1 };   /* storage type of every tensor; arithmetic is fp32 */
enum { GSPN_OK = 0, GSPN_EINVAL = 1, GSPN_EUNSUPPORTED = 2, GSPN_EALIGN = 3,
       GSPN_EWORKSPACE = 4, GSPN_ECUDA = 5 };
/* kernel selection for A/B measurements; GSPN_IMPL_AUTO is what users call */
enum { GSPN_IMPL_AUTO = 0, GSPN_IMPL_NAIVE = 1, GSPN_IMPL_FUSED = 2 /* 16-byte-aligned tile kernel */,
       GSPN_IMPL_FLAT = 3 /* any-shape fused kernel */,
       GSPN_IMPL_CHAIN = 4 /* warp-per-chain kernels (gspn_chain_*.cu) */,
       GSPN_IMPL_PAIR = 5 /* removed in round 2 (an A/B variant nothing selected): GSPN_EUNSUPPORTED; the value stays reserved */,
       GSPN_IMPL_PLANE = 6 /* small planes, forward and backward: whole operand planes on chip, 4 directions at once
                              (gspn_pair_fwd.cu plane_fwd, gspn_plane_bwd.cu) */,
       GSPN_IMPL_LINE = 7 /* 16-byte-aligned rows: warp per (channel, direction) line, several positions per lane,
                              one fp32 accumulator plane per channel (gspn_line_fwd.cu, gspn_line_bwd.cu) */ };

/*
 * Forward scan, Eq. (1),(2),(5),(9): the whole
 * Ls-step recurrence of every direction in dir_mask and the merge over
 * directions in ONE launch; x is read once, y written once.
 */
int gspn_scan_fwd(const void* x, const void* w3, const void* lambda, const void* u, void* y,
                  int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream);

/*
 * Backward scan: the exact adjoint of gspn_scan_fwd (the paper reports
 * backward timings only; derivation in DESIGN.md "Backward").
 * With gy = dy, per direction, in reverse scan order:
 *     gh[s]      = gy[s]*u[s] + w[s+1]^T gh[s+1]
 *     du[s]      = gy[s]*h[s]        dlambda[s] = x[s]*gh[s]
 *     dx[s]     += lambda[s]*gh[s]   (summed over directions)
 *     dw3[g,k,s,p] = sum_{c in g} gh_c[s,p] * h_c[s-1, p+k-1]
 *     dh0        = w[0]^T gh[0]
 * h is recomputed on chip (no saved tensor).  Any output pointer may be NULL
 * (that output is skipped).
 */
int gspn_scan_bwd(const void* x, const void* w3, const void* lambda, const void* u, const void* dy,
                  void* dx, void* dlambda, void* du, void* dw3, void* dh0,
                  int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream);

/*
 * Merge of per-direction outputs (Eq. 9):
 *     y[b,c] = sum_q m[q,c] * y_dirs[q,b,c]     (m NULL = ones), fp32 sum, one RNE.
 */
int gspn_merge(const void* y_dirs, const float* m, void* y,
               int B, int C, int H, int W, unsigned dir_mask, int dtype, void* stream);

/*
 * Row-stochastic normalisation of the raw tap logits, Eq. (3), fused in one pass as the paper's
 * normalisation kernel is ("sigmoid activation, local reduction, clamping, and division"):
 *     s_k = sigmoid(wt[k]),   S = sum of s_k over the taps k whose neighbour lies inside the grid (N(j) of Eq. 3),
 *     w3[k] = s_k / max(S, GSPN_NORM_EPS) for k in N(j),   0 for the out-of-grid taps
 * (tap k <-> neighbour k-1 on the cross axis: j for T->B / B->T, i for L->R / R->L).  wt, w3: DEVICE pointers,
 * [D,B,G,3,H,W] dense, storage type `dtype`, 16-byte aligned, w3 fully overwritten, must not alias wt; fp32
 * arithmetic, one RNE per output.  The paper states no clamp bound: GSPN_NORM_EPS is DESIGN.md reading R17.
 * gspn_normalize_bwd writes dwt = (d w3 / d wt)^T dw3 evaluated at wt (same layouts).  Asynchronous on `stream`;
 * returns a GSPN_* status (GSPN_EINVAL / GSPN_EALIGN / GSPN_ECUDA as for the scans).
 */
#define GSPN_NORM_EPS 1e-6f
int gspn_normalize_fwd(const void* wt, void* w3, int B, int G, int H, int W, unsigned dir_mask, int dtype,
                       void* stream);
int gspn_normalize_bwd(const void* wt, const void* dw3, void* dwt, int B, int G, int H, int W,
                       unsigned dir_mask, int dtype, void* stream);

/* Extended arguments: initial state and kernel selection. */
typedef struct gspn_args {
    size_t struct_size;            /* = sizeof(gspn_args_t) */
    const void *x, *w3, *lambda, *u;
    const void *h0;                /* [D,B,C,Lmax] or NULL (zeros) */
    const void *dy;                /* backward only */
    void *y;                       /* forward only */
    void *dx, *dlambda, *du, *dw3, *dh0;   /* backward only, each may be NULL */
    int B, C, H, W, G;
    unsigned dir_mask;
    int dtype;
    int impl;                      /* GSPN_IMPL_* */
    void *stream;
    /* r2 (reading 6; Eq. 7 writes the propagation operands without a direction index).
     * ELEMENT stride between the direction slabs of the INPUTS w3 / lambda / u:
     *     GSPN_DIR_STRIDE_DENSE, or the dense value itself (3*B*G*H*W for w3, B*C*H*W for lambda and u):
     *         the [D, ...] layout above, one slab per direction -- what every plain call uses;
     *     0:  ONE slab ([B,G,3,H,W] / [B,C,H,W]) read by every direction of dir_mask.  The operand's algorithmic
     *         bytes drop from D slabs to one.
     *     any other value: GSPN_EINVAL.
     * A struct whose fields were zeroed therefore asks for SHARED slabs: set the three fields to GSPN_DIR_STRIDE_DENSE
     * for the dense layout, or pass struct_size = GSPN_ARGS_SIZE_R1 (the struct up to `stream`), which means dense.
     * Outputs are never shared: dlambda, du, dw3 (and h0 / dh0) keep one slab per direction; the gradient of a shared
     * slab is the sum of its D per-direction slabs, in whatever order and precision the caller wants.
     * Shared slabs are served by the naive kernels only in this version (GSPN_IMPL_AUTO or GSPN_IMPL_NAIVE; any other
     * impl reports GSPN_EUNSUPPORTED), so the shapes are those the naive kernels hold. */
    size_t dir_stride_w3, dir_stride_lambda, dir_stride_u;
    /* r2 (PAPER.md:125,129 name `k_chunk` in the launch grid and never define it; reading 10).
     * Chunked scan: the scan axis of every direction is cut, in IMAGE coordinates, into bands of ceil(L / k_chunk) lines
     * (L = H for the vertical directions, W for the horizontal ones; the last band may be shorter), and every band is an
     * independent scan on its sub-grid with a zero initial state.  Both directions of an axis share the bands.  h0 / dh0
     * belong to the band that holds the direction's scan step 0.  0 or 1 = the global scan; negative: GSPN_EINVAL.
     * k_chunk > 1 is served by the naive kernels only in this version (as shared slabs above). */
    int k_chunk;
    /* r2 (second half; the paper's fused kernel consumes the logits).
     * GSPN_FLAG_W3_LOGITS: `w3` holds the raw tap LOGITS [D,B,G,3,H,W] (or one shared slab) and Eq. 3 (gspn_normalize_fwd
     * below: sigmoid, sum over the in-grid taps, clamp at GSPN_NORM_EPS, divide, out-of-grid taps 0) is applied where the
     * scan loads its taps, in fp32: the normalised taps are never written to memory and never rounded to the storage
     * type.  The backward then writes to `dw3` the gradient of the LOGITS (Eq. 3's adjoint, gspn_normalize_bwd, applied on
     * chip to the fp32 group sum; one rounding).  Other bits: GSPN_EINVAL.  Served by the naive kernels only in this
     * version (as shared slabs above). */
    unsigned flags;
    /* r2 (first step): caller-provided DEVICE scratch, 16-byte aligned, at least
     * gspn_workspace_bytes(...) bytes, or NULL.  Needed only where no kernel holds the shape on chip: planes beyond shared
     * memory (about 238 x 238 forward, 120 x 120 backward) with lines of at most 1024 positions are then served by the
     * naive kernels with their plane-sized fp32 arrays (y or h / dx / dw3 accumulators) in this scratch, one slice per
     * CTA.  The library never allocates it, never keeps it, and leaves its contents undefined; calls that share a
     * workspace must not overlap on the GPU.  Without it such a shape reports GSPN_EWORKSPACE (the plain calls above
     * pass none).  The fused kernels ignore it. */
    void *workspace;
    size_t workspace_bytes;
} gspn_args_t;

#define GSPN_FLAG_W3_LOGITS 1u

#define GSPN_DIR_STRIDE_DENSE ((size_t)-1)
#define GSPN_ARGS_SIZE_R1 (offsetof(gspn_args_t, dir_stride_w3))

int gspn_scan_fwd_ex(const gspn_args_t* a);
int gspn_scan_bwd_ex(const gspn_args_t* a);

/* Host-pointer entry points (same layouts, HOST memory; pinned memory makes the copies
 * asynchronous).  They synchronise `stream` before returning. */
int gspn_scan_fwd_host(const void* x, const void* w3, const void* lambda, const void* u, void* y,
                       int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream);
int gspn_scan_bwd_host(const void* x, const void* w3, const void* lambda, const void* u, const void* dy,
                       void* dx, void* dlambda, void* du, void* dw3, void* dh0,
                       int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream);

/*
 * One forward + backward step through HOST buffers (r2): the operands are uploaded ONCE (gspn_scan_fwd_host followed by
 * gspn_scan_bwd_host uploads x, w3, lambda, u twice) and the batch is cut into up to four chunks -- every (b, group) unit
 * is independent, PAPER.md:125 -- that move through three internal streams, so that the upload of chunk i + 1, the kernels
 * of chunk i and the download of chunk i - 1 overlap.  y and each gradient pointer may be NULL (skipped; with all
 * gradients NULL only the forward runs).  Same layouts and status codes as the calls above; synchronous on return
 * (`stream` is used for the allocations only).  Pinned host memory is what makes the copies overlap.
 */
int gspn_scan_fwd_bwd_host(const void* x, const void* w3, const void* lambda, const void* u, const void* dy, void* y,
                           void* dx, void* dlambda, void* du, void* dw3, void* dh0,
                           int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream);
/* Diagnostic: the batch-chunk walk of gspn_scan_fwd_bwd_host with memcpy, host to host (tests check its arithmetic
 * without a GPU).  A tensor of D slabs x B images x image_bytes; images [b0, b0 + bc) <-> a chunk laid out [D, bc]. */
int gspn_debug_chunk_copy(void* chunk, void* host, size_t image_bytes, int D, int B, int b0, int bc, int to_chunk);

/* Bytes of caller-provided scratch (gspn_args_t.workspace) with which every shape of at most 1024 lines is served: 0
 * where the fall-back kernel keeps its planes in shared memory (all five benchmark configs forward, cfg 2 / 3 / 5
 * backward), else the fp32 planes it moves to global memory (forward B*C*H*W*4; backward the larger of 2*B*C*H*W*4 and
 * 4*D*B*G*H*W*4).  An upper bound: a fused kernel that holds the shape does not touch the workspace. */
size_t gspn_workspace_bytes(int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, int is_bwd);

/* Number of kernel launches the last successful call on this thread enqueued. */
int gspn_last_launch_count(void);
/* Name of the kernel variant the last successful call on this thread selected. */
const char* gspn_last_variant(void);

const char* gspn_last_error(void);
int gspn_version(void);            /* 10000*major + 100*minor + patch */

#ifdef __cplusplus
}
#endif
#endif /* GSPN_H_ */
