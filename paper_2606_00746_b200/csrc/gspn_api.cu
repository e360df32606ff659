// gspn_api.cu -- the C ABI of libgspn (include/gspn.h): argument validation, kernel selection,
// host-pointer staging.  No arithmetic of the method lives here.
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include "../../include/gspn.h"
#include "gspn_kernels.h"

namespace gspn {

static thread_local char g_err[512] = "";
static thread_local int g_launches = 0;
static thread_local const char* g_variant = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int check_shape(int B, int C, int H, int W, int G, unsigned mask, int dtype) {
    if (B < 1 || C < 1 || H < 1 || W < 1 || G < 1) {
        set_error("invalid shape B=%d C=%d H=%d W=%d G=%d (all must be >= 1)", B, C, H, W, G);
        return GSPN_EINVAL;
    }
    if (C % G != 0) { set_error("C=%d is not a multiple of G=%d", C, G); return GSPN_EINVAL; }
    if (mask < 1 || mask > 15) { set_error("dir_mask=%u outside [1,15]", mask); return GSPN_EINVAL; }
    if (dtype != GSPN_F32 && dtype != GSPN_BF16) { set_error("unknown dtype %d", dtype); return GSPN_EINVAL; }
    // index arithmetic inside the kernels is 32-bit within a plane and size_t across planes
    if ((long long)H * W > (1ll << 28)) { set_error("H*W too large"); return GSPN_EUNSUPPORTED; }
    return GSPN_OK;
}

#define REQUIRE_PTR(p)                                                               \
    do {                                                                             \
        if (!(p)) { set_error("required pointer '%s' is NULL", #p); return GSPN_EINVAL; } \
        if (!aligned16(p)) { set_error("pointer '%s' is not 16-byte aligned", #p); return GSPN_EALIGN; } \
    } while (0)
#define OPTIONAL_PTR(p)                                                              \
    do {                                                                             \
        if ((p) && !aligned16(p)) { set_error("pointer '%s' is not 16-byte aligned", #p); return GSPN_EALIGN; } \
    } while (0)

// gspn_args_t.dir_stride_*: which inputs have one slab shared by every direction (validated by check_ex)
static unsigned shared_bits(const gspn_args_t* a) {
    if (a->struct_size == GSPN_ARGS_SIZE_R1) return 0;
    return (a->dir_stride_w3 == 0 ? kSharedW3 : 0u) | (a->dir_stride_lambda == 0 ? kSharedLam : 0u) |
           (a->dir_stride_u == 0 ? kSharedU : 0u);
}
static int chunks(const gspn_args_t* a) { return a->struct_size == GSPN_ARGS_SIZE_R1 ? 0 : a->k_chunk; }
static unsigned arg_flags(const gspn_args_t* a) { return a->struct_size == GSPN_ARGS_SIZE_R1 ? 0u : a->flags; }
static float* arg_ws(const gspn_args_t* a) { return a->struct_size == GSPN_ARGS_SIZE_R1 ? nullptr : (float*)a->workspace; }
static size_t arg_ws_bytes(const gspn_args_t* a) { return a->struct_size == GSPN_ARGS_SIZE_R1 || !a->workspace ? 0 : a->workspace_bytes; }

template <typename ST>
static int fwd_typed(const gspn_args_t* a) {
    FwdArgs<ST> f;
    f.x = (const ST*)a->x; f.w3 = (const ST*)a->w3; f.lam = (const ST*)a->lambda;
    f.u = (const ST*)a->u; f.h0 = (const ST*)a->h0; f.y = (ST*)a->y;
    f.sh = Shape{a->B, a->C, a->H, a->W, a->G, a->dir_mask, shared_bits(a), chunks(a), arg_flags(a)};
    f.ws = arg_ws(a); f.ws_bytes = arg_ws_bytes(a);
    cudaStream_t st = (cudaStream_t)a->stream;
    LaunchInfo li{0, ""};
    int rc;
    if (f.sh.shared || f.sh.k_chunk > 1 || f.sh.flags) {      // shared slabs, chunked scan, logits: the naive kernel only (include/gspn.h)
        if (a->impl != GSPN_IMPL_AUTO && a->impl != GSPN_IMPL_NAIVE) {
            set_error("shared direction slabs (dir_stride_* = 0), k_chunk > 1 and GSPN_FLAG_W3_LOGITS are served by the naive kernels only (impl %d asked)", a->impl);
            return GSPN_EUNSUPPORTED;
        }
        rc = naive_fwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_NAIVE) {
        rc = naive_fwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_FLAT) {
        rc = flat_fwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_CHAIN) {
        rc = chain_fwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_PAIR) {
        set_error("GSPN_IMPL_PAIR: the ring-staged pair kernel was removed in round 2 (nothing selected it)");
        rc = GSPN_EUNSUPPORTED;
    } else if (a->impl == GSPN_IMPL_PLANE) {
        rc = plane_fwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_LINE) {
        rc = line_fwd_launch<ST>(f, st, &li);
    } else {
        rc = a->impl == GSPN_IMPL_AUTO ? line_fwd_launch<ST>(f, st, &li) : GSPN_EUNSUPPORTED;
        if (rc == GSPN_EUNSUPPORTED) rc = fused_fwd_launch<ST>(f, st, &li);
        // rows that are not 16-byte aligned: lines of at most 64 positions whose planes fit on chip whole (twice
        // per SM) go to the whole-plane kernel (378-px config: 0.29 ms against 0.50 ms for the chain kernel; 45x45,
        // B=64, C=128: 0.30 against 0.41 ms), the rest to the chain kernel
        if (rc == GSPN_EUNSUPPORTED && a->impl == GSPN_IMPL_AUTO) rc = plane_fwd_launch<ST>(f, st, &li);
        if (rc == GSPN_EUNSUPPORTED && a->impl == GSPN_IMPL_AUTO) rc = chain_fwd_launch<ST>(f, st, &li);
        if (rc == GSPN_EUNSUPPORTED && a->impl == GSPN_IMPL_AUTO) rc = flat_fwd_launch<ST>(f, st, &li);
        if (rc == GSPN_EUNSUPPORTED && a->impl == GSPN_IMPL_AUTO) rc = naive_fwd_launch<ST>(f, st, &li);
    }
    if (rc == GSPN_OK) { g_launches = li.launches; g_variant = li.variant; }
    return rc;
}

template <typename ST>
static int bwd_typed(const gspn_args_t* a) {
    BwdArgs<ST> f;
    f.x = (const ST*)a->x; f.w3 = (const ST*)a->w3; f.lam = (const ST*)a->lambda;
    f.u = (const ST*)a->u; f.h0 = (const ST*)a->h0; f.dy = (const ST*)a->dy;
    f.dx = (ST*)a->dx; f.dlam = (ST*)a->dlambda; f.du = (ST*)a->du; f.dw3 = (ST*)a->dw3;
    f.dh0 = (ST*)a->dh0;
    f.sh = Shape{a->B, a->C, a->H, a->W, a->G, a->dir_mask, shared_bits(a), chunks(a), arg_flags(a)};
    f.ws = arg_ws(a); f.ws_bytes = arg_ws_bytes(a);
    cudaStream_t st = (cudaStream_t)a->stream;
    LaunchInfo li{0, ""};
    int rc;
    if (f.sh.shared || f.sh.k_chunk > 1 || f.sh.flags) {
        if (a->impl != GSPN_IMPL_AUTO && a->impl != GSPN_IMPL_NAIVE) {
            set_error("shared direction slabs (dir_stride_* = 0), k_chunk > 1 and GSPN_FLAG_W3_LOGITS are served by the naive kernels only (impl %d asked)", a->impl);
            return GSPN_EUNSUPPORTED;
        }
        rc = naive_bwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_NAIVE) {
        rc = naive_bwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_FUSED) {
        rc = fused_bwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_CHAIN) {
        rc = chain_bwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_PLANE) {
        rc = plane_bwd_launch<ST>(f, st, &li);
    } else if (a->impl == GSPN_IMPL_LINE) {
        rc = line_bwd_launch<ST>(f, st, &li);
    } else {
        // lines of at most one warp (378-px config: 27x27): the whole-plane kernel where the unit's planes fit on chip
        // (cfg3 0.89 ms), else the group kernel (2.45 ms; the per-block hand-shakes of the chain kernel cost more
        // there: 2.97 ms); longer lines: the chain kernel
        // (the line backward, gspn_line_bwd.cu, is selected with GSPN_IMPL_LINE only until it has passed the GPU
        // parity suite: see DESIGN.md section 7)
        const bool small = f.sh.Lmax() <= 32;
        rc = small ? plane_bwd_launch<ST>(f, st, &li) : chain_bwd_launch<ST>(f, st, &li);
        if (rc == GSPN_EUNSUPPORTED && small) rc = fused_bwd_launch<ST>(f, st, &li);
        if (rc == GSPN_EUNSUPPORTED) rc = small ? chain_bwd_launch<ST>(f, st, &li) : fused_bwd_launch<ST>(f, st, &li);
        if (rc == GSPN_EUNSUPPORTED) rc = naive_bwd_launch<ST>(f, st, &li);
    }
    if (rc == GSPN_OK) { g_launches = li.launches; g_variant = li.variant; }
    return rc;
}

static int check_ex(const gspn_args_t* a) {
    if (!a) { set_error("args is NULL"); return GSPN_EINVAL; }
    if (a->struct_size != sizeof(gspn_args_t) && a->struct_size != GSPN_ARGS_SIZE_R1) {
        set_error("gspn_args_t.struct_size=%zu, expected %zu (or %zu, the round-1 layout without dir_stride_*)", a->struct_size,
                  sizeof(gspn_args_t), (size_t)GSPN_ARGS_SIZE_R1);
        return GSPN_EINVAL;
    }
    if (a->impl < GSPN_IMPL_AUTO || a->impl > GSPN_IMPL_LINE) {
        set_error("unknown impl %d", a->impl);
        return GSPN_EINVAL;
    }
    int rc = check_shape(a->B, a->C, a->H, a->W, a->G, a->dir_mask, a->dtype);
    if (rc) return rc;
    if (a->struct_size == sizeof(gspn_args_t)) {
        const size_t hw = (size_t)a->H * a->W;
        const size_t dense[3] = {(size_t)3 * a->B * a->G * hw, (size_t)a->B * a->C * hw, (size_t)a->B * a->C * hw};
        const size_t got[3] = {a->dir_stride_w3, a->dir_stride_lambda, a->dir_stride_u};
        const char* name[3] = {"dir_stride_w3", "dir_stride_lambda", "dir_stride_u"};
        for (int t = 0; t < 3; ++t)
            if (got[t] != 0 && got[t] != GSPN_DIR_STRIDE_DENSE && got[t] != dense[t]) {
                set_error("%s=%zu: only 0 (one slab shared by every direction) and the dense stride %zu (GSPN_DIR_STRIDE_DENSE) "
                          "are supported", name[t], got[t], dense[t]);
                return GSPN_EINVAL;
            }
        if (a->k_chunk < 0) { set_error("k_chunk=%d is negative (0 or 1 = the global scan)", a->k_chunk); return GSPN_EINVAL; }
        if (a->flags & ~GSPN_FLAG_W3_LOGITS) { set_error("flags=0x%x: unknown bit(s)", a->flags); return GSPN_EINVAL; }
        if (a->workspace && !aligned16(a->workspace)) { set_error("pointer 'workspace' is not 16-byte aligned"); return GSPN_EALIGN; }
    }
    return GSPN_OK;
}

static size_t esize(int dtype) { return dtype == GSPN_F32 ? 4 : 2; }

}  // namespace gspn

using namespace gspn;

extern "C" {

int gspn_scan_fwd_ex(const gspn_args_t* a) {
    int rc = check_ex(a);
    if (rc) return rc;
    REQUIRE_PTR(a->x); REQUIRE_PTR(a->w3); REQUIRE_PTR(a->lambda); REQUIRE_PTR(a->u); REQUIRE_PTR(a->y);
    OPTIONAL_PTR(a->h0);
    return a->dtype == GSPN_F32 ? fwd_typed<float>(a) : fwd_typed<__nv_bfloat16>(a);
}

int gspn_scan_bwd_ex(const gspn_args_t* a) {
    int rc = check_ex(a);
    if (rc) return rc;
    REQUIRE_PTR(a->x); REQUIRE_PTR(a->w3); REQUIRE_PTR(a->lambda); REQUIRE_PTR(a->u); REQUIRE_PTR(a->dy);
    OPTIONAL_PTR(a->h0); OPTIONAL_PTR(a->dx); OPTIONAL_PTR(a->dlambda); OPTIONAL_PTR(a->du);
    OPTIONAL_PTR(a->dw3); OPTIONAL_PTR(a->dh0);
    if (!a->dx && !a->dlambda && !a->du && !a->dw3 && !a->dh0) { g_launches = 0; g_variant = "none"; return GSPN_OK; }
    return a->dtype == GSPN_F32 ? bwd_typed<float>(a) : bwd_typed<__nv_bfloat16>(a);
}

int gspn_scan_fwd(const void* x, const void* w3, const void* lambda, const void* u, void* y,
                  int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream) {
    gspn_args_t a;
    memset(&a, 0, sizeof(a));
    a.struct_size = sizeof(a);
    a.x = x; a.w3 = w3; a.lambda = lambda; a.u = u; a.y = y;
    a.B = B; a.C = C; a.H = H; a.W = W; a.G = G; a.dir_mask = dir_mask; a.dtype = dtype;
    a.impl = GSPN_IMPL_AUTO; a.stream = stream;
    a.dir_stride_w3 = a.dir_stride_lambda = a.dir_stride_u = GSPN_DIR_STRIDE_DENSE;
    return gspn_scan_fwd_ex(&a);
}

int gspn_scan_bwd(const void* x, const void* w3, const void* lambda, const void* u, const void* dy,
                  void* dx, void* dlambda, void* du, void* dw3, void* dh0,
                  int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream) {
    gspn_args_t a;
    memset(&a, 0, sizeof(a));
    a.struct_size = sizeof(a);
    a.x = x; a.w3 = w3; a.lambda = lambda; a.u = u; a.dy = dy;
    a.dx = dx; a.dlambda = dlambda; a.du = du; a.dw3 = dw3; a.dh0 = dh0;
    a.B = B; a.C = C; a.H = H; a.W = W; a.G = G; a.dir_mask = dir_mask; a.dtype = dtype;
    a.impl = GSPN_IMPL_AUTO; a.stream = stream;
    a.dir_stride_w3 = a.dir_stride_lambda = a.dir_stride_u = GSPN_DIR_STRIDE_DENSE;
    return gspn_scan_bwd_ex(&a);
}

int gspn_merge(const void* y_dirs, const float* m, void* y,
               int B, int C, int H, int W, unsigned dir_mask, int dtype, void* stream) {
    int rc = check_shape(B, C, H, W, 1, dir_mask, dtype);
    if (rc) return rc;
    REQUIRE_PTR(y_dirs); REQUIRE_PTR(y);
    if (m && (reinterpret_cast<uintptr_t>(m) & 3u)) { set_error("pointer 'm' is not 4-byte aligned"); return GSPN_EALIGN; }
    const int D = Shape{B, C, H, W, 1, dir_mask}.D();
    LaunchInfo li{0, ""};
    rc = dtype == GSPN_F32
             ? merge_launch<float>((const float*)y_dirs, m, (float*)y, D, B, C, H, W, (cudaStream_t)stream, &li)
             : merge_launch<__nv_bfloat16>((const __nv_bfloat16*)y_dirs, m, (__nv_bfloat16*)y, D, B, C, H, W,
                                           (cudaStream_t)stream, &li);
    if (rc == GSPN_OK) { g_launches = li.launches; g_variant = li.variant; }
    return rc;
}

int gspn_normalize_fwd(const void* wt, void* w3, int B, int G, int H, int W, unsigned dir_mask, int dtype,
                       void* stream) {
    int rc = check_shape(B, G, H, W, G, dir_mask, dtype);
    if (rc) return rc;
    REQUIRE_PTR(wt); REQUIRE_PTR(w3);
    LaunchInfo li{0, ""};
    rc = dtype == GSPN_F32
             ? norm_launch<float>((const float*)wt, nullptr, (float*)w3, B, G, H, W, dir_mask, (cudaStream_t)stream, &li)
             : norm_launch<__nv_bfloat16>((const __nv_bfloat16*)wt, nullptr, (__nv_bfloat16*)w3, B, G, H, W, dir_mask,
                                          (cudaStream_t)stream, &li);
    if (rc == GSPN_OK) { g_launches = li.launches; g_variant = li.variant; }
    return rc;
}

int gspn_normalize_bwd(const void* wt, const void* dw3, void* dwt, int B, int G, int H, int W,
                       unsigned dir_mask, int dtype, void* stream) {
    int rc = check_shape(B, G, H, W, G, dir_mask, dtype);
    if (rc) return rc;
    REQUIRE_PTR(wt); REQUIRE_PTR(dw3); REQUIRE_PTR(dwt);
    LaunchInfo li{0, ""};
    rc = dtype == GSPN_F32
             ? norm_launch<float>((const float*)wt, (const float*)dw3, (float*)dwt, B, G, H, W, dir_mask,
                                  (cudaStream_t)stream, &li)
             : norm_launch<__nv_bfloat16>((const __nv_bfloat16*)wt, (const __nv_bfloat16*)dw3, (__nv_bfloat16*)dwt, B, G,
                                          H, W, dir_mask, (cudaStream_t)stream, &li);
    if (rc == GSPN_OK) { g_launches = li.launches; g_variant = li.variant; }
    return rc;
}

// ---- host-pointer entry points ------------------------------------------------------------
#define CUDA_TRY(expr)                                                                   \
    do {                                                                                 \
        cudaError_t e_ = (expr);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            set_error("%s: %s", #expr, cudaGetErrorString(e_));                          \
            rc = GSPN_ECUDA;                                                             \
            goto done;                                                                   \
        }                                                                                \
    } while (0)

int gspn_scan_fwd_host(const void* x, const void* w3, const void* lambda, const void* u, void* y,
                       int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream) {
    int rc = check_shape(B, C, H, W, G, dir_mask, dtype);
    if (rc) return rc;
    if (!x || !w3 || !lambda || !u || !y) { set_error("NULL host pointer"); return GSPN_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t s = esize(dtype), D = Shape{B, C, H, W, G, dir_mask}.D();
    const size_t n = (size_t)B * C * H * W * s, nw = (size_t)3 * B * G * H * W * s;
    void *dx_ = nullptr, *dw = nullptr, *dl = nullptr, *du_ = nullptr, *dy_ = nullptr;
    CUDA_TRY(cudaMallocAsync(&dx_, n, st));
    CUDA_TRY(cudaMallocAsync(&dw, D * nw, st));
    CUDA_TRY(cudaMallocAsync(&dl, D * n, st));
    CUDA_TRY(cudaMallocAsync(&du_, D * n, st));
    CUDA_TRY(cudaMallocAsync(&dy_, n, st));
    CUDA_TRY(cudaMemcpyAsync(dx_, x, n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(dw, w3, D * nw, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(dl, lambda, D * n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(du_, u, D * n, cudaMemcpyHostToDevice, st));
    rc = gspn_scan_fwd(dx_, dw, dl, du_, dy_, B, C, H, W, G, dir_mask, dtype, stream);
    if (rc) goto done;
    CUDA_TRY(cudaMemcpyAsync(y, dy_, n, cudaMemcpyDeviceToHost, st));
done:
    if (dx_) cudaFreeAsync(dx_, st);
    if (dw) cudaFreeAsync(dw, st);
    if (dl) cudaFreeAsync(dl, st);
    if (du_) cudaFreeAsync(du_, st);
    if (dy_) cudaFreeAsync(dy_, st);
    cudaError_t e = cudaStreamSynchronize(st);
    if (rc == GSPN_OK && e != cudaSuccess) { set_error("cudaStreamSynchronize: %s", cudaGetErrorString(e)); rc = GSPN_ECUDA; }
    return rc;
}

int gspn_scan_bwd_host(const void* x, const void* w3, const void* lambda, const void* u, const void* dy,
                       void* dx, void* dlambda, void* du, void* dw3, void* dh0,
                       int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream) {
    int rc = check_shape(B, C, H, W, G, dir_mask, dtype);
    if (rc) return rc;
    if (!x || !w3 || !lambda || !u || !dy) { set_error("NULL host pointer"); return GSPN_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t s = esize(dtype), D = Shape{B, C, H, W, G, dir_mask}.D();
    const size_t n = (size_t)B * C * H * W * s, nw = (size_t)3 * B * G * H * W * s;
    const size_t nh = D * (size_t)B * C * (H > W ? H : W) * s;
    const void* hin[5] = {x, w3, lambda, u, dy};
    const size_t bin[5] = {n, D * nw, D * n, D * n, n};
    void* hout[5] = {dx, dlambda, du, dw3, dh0};
    const size_t bout[5] = {n, D * n, D * n, D * nw, nh};
    void* din[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    void* dout[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    for (int t = 0; t < 5; ++t) {
        CUDA_TRY(cudaMallocAsync(&din[t], bin[t], st));
        CUDA_TRY(cudaMemcpyAsync(din[t], hin[t], bin[t], cudaMemcpyHostToDevice, st));
        if (hout[t]) CUDA_TRY(cudaMallocAsync(&dout[t], bout[t], st));
    }
    rc = gspn_scan_bwd(din[0], din[1], din[2], din[3], din[4], dout[0], dout[1], dout[2], dout[3], dout[4],
                       B, C, H, W, G, dir_mask, dtype, stream);
    if (rc) goto done;
    for (int t = 0; t < 5; ++t)
        if (hout[t]) CUDA_TRY(cudaMemcpyAsync(hout[t], dout[t], bout[t], cudaMemcpyDeviceToHost, st));
done:
    for (int t = 0; t < 5; ++t) {
        if (din[t]) cudaFreeAsync(din[t], st);
        if (dout[t]) cudaFreeAsync(dout[t], st);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    if (rc == GSPN_OK && e != cudaSuccess) { set_error("cudaStreamSynchronize: %s", cudaGetErrorString(e)); rc = GSPN_ECUDA; }
    return rc;
}

// ---- one forward + backward step through host buffers, operands uploaded once, pipelined over batch chunks ----------
// Every tensor is [B, ...] or [D, B, ...] and every (b, group) unit is independent, so the batch is cut
// into chunks; a chunk lives on the device as the same layout with B = its own size.  chunk_copy walks the D slabs of
// one tensor for the images [b0, b0 + bc): `to_chunk` host -> chunk, else chunk -> host.
}  // extern "C"

template <typename Copy>
static int chunk_copy(unsigned char* chunk, unsigned char* host, size_t image_bytes, size_t D, size_t B, size_t b0, size_t bc,
                      bool to_chunk, Copy copy) {
    for (size_t q = 0; q < D; ++q) {
        unsigned char* h = host + (q * B + b0) * image_bytes;
        unsigned char* c = chunk + q * bc * image_bytes;
        const int rc = to_chunk ? copy(c, h, bc * image_bytes) : copy(h, c, bc * image_bytes);
        if (rc) return rc;
    }
    return 0;
}

extern "C" {

// the same walk with memcpy, host to host: what tests/test_abi.py checks the chunk arithmetic with (no GPU needed)
int gspn_debug_chunk_copy(void* chunk, void* host, size_t image_bytes, int D, int B, int b0, int bc, int to_chunk) {
    if (!chunk || !host || D < 1 || B < 1 || b0 < 0 || bc < 1 || b0 + bc > B) { set_error("gspn_debug_chunk_copy: bad arguments"); return GSPN_EINVAL; }
    return chunk_copy((unsigned char*)chunk, (unsigned char*)host, image_bytes, (size_t)D, (size_t)B, (size_t)b0, (size_t)bc,
                      to_chunk != 0, [](void* d, const void* s_, size_t n) { memcpy(d, s_, n); return 0; });
}

int gspn_scan_fwd_bwd_host(const void* x, const void* w3, const void* lambda, const void* u, const void* dy, void* y,
                           void* dx, void* dlambda, void* du, void* dw3, void* dh0,
                           int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, void* stream) {
    int rc = check_shape(B, C, H, W, G, dir_mask, dtype);
    if (rc) return rc;
    if (!x || !w3 || !lambda || !u || !dy) { set_error("NULL host pointer"); return GSPN_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t s = esize(dtype), D = Shape{B, C, H, W, G, dir_mask}.D(), L = (size_t)(H > W ? H : W);
    const size_t ic = (size_t)C * H * W * s, iw = (size_t)3 * G * H * W * s, ih = (size_t)C * L * s;   // bytes per image
    const int nchunk = B < 4 ? B : 4;
    const int bcmax = (B + nchunk - 1) / nchunk;
    // tensors: 0 x, 1 w3, 2 lambda, 3 u, 4 dy (inputs); 5 y, 6 dx, 7 dlambda, 8 du, 9 dw3, 10 dh0 (outputs)
    void* host[11] = {(void*)x, (void*)w3, (void*)lambda, (void*)u, (void*)dy, y, dx, dlambda, du, dw3, dh0};
    const size_t img[11] = {ic, iw, ic, ic, ic, ic, ic, ic, ic, iw, ih};
    const size_t slabs[11] = {1, D, D, D, 1, 1, 1, D, D, D, D};
    void* dev[2][11] = {};
    cudaStream_t sin = nullptr, sk = nullptr, sout = nullptr;
    cudaEvent_t in_done[2] = {}, k_done[2] = {}, out_done[2] = {};
    auto h2d = [&](void* d, const void* h, size_t n) { return cudaMemcpyAsync(d, h, n, cudaMemcpyHostToDevice, sin) == cudaSuccess ? 0 : 1; };
    auto d2h = [&](void* h, const void* d, size_t n) { return cudaMemcpyAsync(h, d, n, cudaMemcpyDeviceToHost, sout) == cudaSuccess ? 0 : 1; };
    for (int sl = 0; sl < 2 && sl < nchunk; ++sl)
        for (int t = 0; t < 11; ++t)
            if (host[t]) CUDA_TRY(cudaMallocAsync(&dev[sl][t], slabs[t] * bcmax * img[t], st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaStreamCreateWithFlags(&sin, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&sk, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&sout, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
        CUDA_TRY(cudaEventCreateWithFlags(&in_done[i], cudaEventDisableTiming));
        CUDA_TRY(cudaEventCreateWithFlags(&k_done[i], cudaEventDisableTiming));
        CUDA_TRY(cudaEventCreateWithFlags(&out_done[i], cudaEventDisableTiming));
    }
    for (int ci = 0, b0 = 0; b0 < B; ++ci, b0 += bcmax) {
        const int bc = B - b0 < bcmax ? B - b0 : bcmax, sl = ci & 1;
        // uploads of this chunk: its input buffers are free once the kernels of the chunk before last are done
        if (ci >= 2) CUDA_TRY(cudaStreamWaitEvent(sin, k_done[sl], 0));
        for (int t = 0; t < 5; ++t)
            if (chunk_copy((unsigned char*)dev[sl][t], (unsigned char*)host[t], img[t], slabs[t], (size_t)B, (size_t)b0, (size_t)bc, true, h2d)) {
                set_error("gspn_scan_fwd_bwd_host: cudaMemcpyAsync (H2D) failed"); rc = GSPN_ECUDA; goto done;
            }
        CUDA_TRY(cudaEventRecord(in_done[sl], sin));
        // kernels: after the uploads, and after the downloads of the chunk before last have left the output buffers
        CUDA_TRY(cudaStreamWaitEvent(sk, in_done[sl], 0));
        if (ci >= 2) CUDA_TRY(cudaStreamWaitEvent(sk, out_done[sl], 0));
        if (y) {
            rc = gspn_scan_fwd(dev[sl][0], dev[sl][1], dev[sl][2], dev[sl][3], dev[sl][5], bc, C, H, W, G, dir_mask, dtype, (void*)sk);
            if (rc) goto done;
        }
        if (dx || dlambda || du || dw3 || dh0) {
            rc = gspn_scan_bwd(dev[sl][0], dev[sl][1], dev[sl][2], dev[sl][3], dev[sl][4], dev[sl][6], dev[sl][7], dev[sl][8],
                               dev[sl][9], dev[sl][10], bc, C, H, W, G, dir_mask, dtype, (void*)sk);
            if (rc) goto done;
        }
        CUDA_TRY(cudaEventRecord(k_done[sl], sk));
        // downloads
        CUDA_TRY(cudaStreamWaitEvent(sout, k_done[sl], 0));
        for (int t = 5; t < 11; ++t)
            if (host[t] && chunk_copy((unsigned char*)dev[sl][t], (unsigned char*)host[t], img[t], slabs[t], (size_t)B, (size_t)b0, (size_t)bc, false, d2h)) {
                set_error("gspn_scan_fwd_bwd_host: cudaMemcpyAsync (D2H) failed"); rc = GSPN_ECUDA; goto done;
            }
        CUDA_TRY(cudaEventRecord(out_done[sl], sout));
    }
done:
    {
        cudaError_t e1 = sin ? cudaStreamSynchronize(sin) : cudaSuccess;
        cudaError_t e2 = sk ? cudaStreamSynchronize(sk) : cudaSuccess;
        cudaError_t e3 = sout ? cudaStreamSynchronize(sout) : cudaSuccess;
        for (int sl = 0; sl < 2; ++sl)
            for (int t = 0; t < 11; ++t)
                if (dev[sl][t]) cudaFreeAsync(dev[sl][t], st);
        cudaError_t e4 = cudaStreamSynchronize(st);
        for (int i = 0; i < 2; ++i) {
            if (in_done[i]) cudaEventDestroy(in_done[i]);
            if (k_done[i]) cudaEventDestroy(k_done[i]);
            if (out_done[i]) cudaEventDestroy(out_done[i]);
        }
        if (sin) cudaStreamDestroy(sin);
        if (sk) cudaStreamDestroy(sk);
        if (sout) cudaStreamDestroy(sout);
        const cudaError_t e = e1 != cudaSuccess ? e1 : e2 != cudaSuccess ? e2 : e3 != cudaSuccess ? e3 : e4;
        if (rc == GSPN_OK && e != cudaSuccess) { set_error("gspn_scan_fwd_bwd_host: %s", cudaGetErrorString(e)); rc = GSPN_ECUDA; }
    }
    return rc;
}

size_t gspn_workspace_bytes(int B, int C, int H, int W, int G, unsigned dir_mask, int dtype, int is_bwd) {
    if (check_shape(B, C, H, W, G, dir_mask, dtype) != GSPN_OK) return 0;
    return naive_workspace_bytes(Shape{B, C, H, W, G, dir_mask}, is_bwd != 0);
}

int gspn_last_launch_count(void) { return g_launches; }
const char* gspn_last_variant(void) { return g_variant; }
const char* gspn_last_error(void) { return g_err; }
int gspn_version(void) { return 100; }   /* 0.1.0 */

}  // extern "C"
