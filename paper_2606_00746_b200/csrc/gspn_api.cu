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

template <typename ST>
static int fwd_typed(const gspn_args_t* a) {
    FwdArgs<ST> f;
    f.x = (const ST*)a->x; f.w3 = (const ST*)a->w3; f.lam = (const ST*)a->lambda;
    f.u = (const ST*)a->u; f.h0 = (const ST*)a->h0; f.y = (ST*)a->y;
    f.sh = Shape{a->B, a->C, a->H, a->W, a->G, a->dir_mask};
    cudaStream_t st = (cudaStream_t)a->stream;
    LaunchInfo li{0, ""};
    int rc;
    if (a->impl == GSPN_IMPL_NAIVE) {
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
    f.sh = Shape{a->B, a->C, a->H, a->W, a->G, a->dir_mask};
    cudaStream_t st = (cudaStream_t)a->stream;
    LaunchInfo li{0, ""};
    int rc;
    if (a->impl == GSPN_IMPL_NAIVE) {
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
    if (a->struct_size != sizeof(gspn_args_t)) {
        set_error("gspn_args_t.struct_size=%zu, expected %zu", a->struct_size, sizeof(gspn_args_t));
        return GSPN_EINVAL;
    }
    if (a->impl < GSPN_IMPL_AUTO || a->impl > GSPN_IMPL_LINE) {
        set_error("unknown impl %d", a->impl);
        return GSPN_EINVAL;
    }
    return check_shape(a->B, a->C, a->H, a->W, a->G, a->dir_mask, a->dtype);
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

size_t gspn_workspace_bytes(int, int, int, int, int, unsigned, int, int) { return 0; }

int gspn_last_launch_count(void) { return g_launches; }
const char* gspn_last_variant(void) { return g_variant; }
const char* gspn_last_error(void) { return g_err; }
int gspn_version(void) { return 100; }   /* 0.1.0 */

}  // extern "C"
