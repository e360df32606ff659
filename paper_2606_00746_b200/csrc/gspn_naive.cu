// gspn_naive.cu -- the naive GPU path of libgspn: one CTA per (b,c) plane (forward, backward
// main) or per (direction, b, group) (weight gradients), one thread per cross position p,
// operands read straight from global memory (a thread fetches the operands of kChunk consecutive
// steps together, so the global latency is paid once per chunk), one __syncthreads per scan step.  It exists as the
// simple-by-construction GPU implementation of Eq. (1),(2),(5) that the
// fused kernels are A/B-checked against and that serves shapes the fused kernels do not take.
// Operation order matches a left-to-right evaluation of the recurrence with fused multiply-adds.
#include "gspn_kernels.h"
#include "gspn_naive.cuh"
#include "../../include/gspn.h"

namespace gspn {

static int round_up32(int v) { return (v + 31) / 32 * 32; }

template <typename K>
static int prep_smem(K kernel, size_t bytes, const char* what) {
    if (bytes > (size_t)kMaxSmemOptin) {
        set_error("%s: needs %zu B of shared memory per CTA (> %d)", what, bytes, kMaxSmemOptin);
        return GSPN_EUNSUPPORTED;
    }
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemOptin);
    if (e != cudaSuccess) {
        set_error("%s: cudaFuncSetAttribute: %s", what, cudaGetErrorString(e));
        return GSPN_ECUDA;
    }
    return GSPN_OK;
}

static int check_launch(const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("%s: launch failed: %s", what, cudaGetErrorString(e));
        return GSPN_ECUDA;
    }
    return GSPN_OK;
}

// Planes too large for shared memory: the plane-sized fp32 arrays move to the caller's workspace, one
// slice per CTA; shared memory then holds the lines only.  Bytes needed, 0 when shared memory is enough:
static size_t aux_bytes(const Shape& sh) { return 3 * (size_t)(sh.Lmax() + 2) * sizeof(float); }
static size_t fwd_smem(const Shape& sh) { return (sh.plane() + 2 * (size_t)(sh.Lmax() + 2)) * sizeof(float); }
static size_t fwd_ws(const Shape& sh) { return (size_t)sh.B * sh.C * sh.plane() * sizeof(float); }
static size_t main_smem(const Shape& sh) { return 2 * sh.plane() * sizeof(float) + aux_bytes(sh); }
static size_t main_ws(const Shape& sh) { return (size_t)sh.B * sh.C * 2 * sh.plane() * sizeof(float); }
static size_t dw_smem(const Shape& sh) { return 4 * sh.plane() * sizeof(float) + aux_bytes(sh); }
static size_t dw_ws(const Shape& sh) { return (size_t)sh.D() * sh.B * sh.G * 4 * sh.plane() * sizeof(float); }

size_t naive_workspace_bytes(const Shape& sh, bool bwd) {
    if (sh.Lmax() > 1024) return 0;                       // not held at all
    if (!bwd) return fwd_smem(sh) > (size_t)kMaxSmemOptin ? fwd_ws(sh) : 0;
    const size_t a = main_smem(sh) > (size_t)kMaxSmemOptin ? main_ws(sh) : 0;
    const size_t b = dw_smem(sh) > (size_t)kMaxSmemOptin ? dw_ws(sh) : 0;
    return a > b ? a : b;                                 // the two launches run one after the other on the same stream
}

// shared memory if the planes fit, else the workspace (GSPN_EWORKSPACE when it is missing or too small)
static int pick_store(size_t smem_need, size_t ws_need, float* ws, size_t ws_bytes, const char* what, bool* use_ws) {
    *use_ws = smem_need > (size_t)kMaxSmemOptin;
    if (*use_ws && (!ws || ws_bytes < ws_need)) {
        set_error("%s: planes beyond shared memory need a workspace of %zu bytes (gspn_workspace_bytes; gspn_args_t.workspace holds %zu)",
                  what, ws_need, ws ? ws_bytes : (size_t)0);
        return GSPN_EWORKSPACE;
    }
    return GSPN_OK;
}

template <typename ST>
int naive_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    const Shape& sh = a.sh;
    if (sh.Lmax() > 1024) { set_error("naive fwd: max(H,W) = %d > 1024", sh.Lmax()); return GSPN_EUNSUPPORTED; }
    bool use_ws;
    int rc = pick_store(fwd_smem(sh), fwd_ws(sh), a.ws, a.ws_bytes, "naive fwd", &use_ws);
    if (rc) return rc;
    const size_t smem = use_ws ? 2 * (size_t)(sh.Lmax() + 2) * sizeof(float) : fwd_smem(sh);
    rc = prep_smem(naive_fwd_kernel<ST>, smem, "naive fwd");
    if (rc) return rc;
    GSPN_LAUNCH(naive_fwd_kernel<ST>, sh.B * sh.C, round_up32(sh.Lmax()), smem, st, a, use_ws ? a.ws : nullptr);
    li->launches = 1;
    li->variant = use_ws ? "naive_fwd_ws" : "naive_fwd";
    return check_launch("naive fwd");
}

template <typename ST>
int naive_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    const Shape& sh = a.sh;
    if (sh.Lmax() > 1024) { set_error("naive bwd: max(H,W) = %d > 1024", sh.Lmax()); return GSPN_EUNSUPPORTED; }
    li->launches = 0;
    li->variant = "naive_bwd";
    if (a.dx || a.dlam || a.du || a.dh0) {
        bool use_ws;
        int rc = pick_store(main_smem(sh), main_ws(sh), a.ws, a.ws_bytes, "naive bwd (dx,dlambda,du,dh0)", &use_ws);
        if (rc) return rc;
        const size_t smem = use_ws ? aux_bytes(sh) : main_smem(sh);
        rc = prep_smem(naive_bwd_main_kernel<ST>, smem, "naive bwd (dx,dlambda,du,dh0)");
        if (rc) return rc;
        GSPN_LAUNCH(naive_bwd_main_kernel<ST>, sh.B * sh.C, round_up32(sh.Lmax()), smem, st, a, use_ws ? a.ws : nullptr);
        ++li->launches;
        if (use_ws) li->variant = "naive_bwd_ws";
        rc = check_launch("naive bwd main");
        if (rc) return rc;
    }
    if (a.dw3) {
        bool use_ws;
        int rc = pick_store(dw_smem(sh), dw_ws(sh), a.ws, a.ws_bytes, "naive bwd (dw3)", &use_ws);
        if (rc) return rc;
        const size_t smem = use_ws ? aux_bytes(sh) : dw_smem(sh);
        rc = prep_smem(naive_bwd_dw_kernel<ST>, smem, "naive bwd (dw3)");
        if (rc) return rc;
        GSPN_LAUNCH(naive_bwd_dw_kernel<ST>, sh.D() * sh.B * sh.G, round_up32(sh.Lmax()), smem, st, a, use_ws ? a.ws : nullptr);
        ++li->launches;
        if (use_ws) li->variant = "naive_bwd_ws";
        rc = check_launch("naive bwd dw");
        if (rc) return rc;
    }
    return GSPN_OK;
}

template int naive_fwd_launch<float>(const FwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int naive_fwd_launch<__nv_bfloat16>(const FwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);
template int naive_bwd_launch<float>(const BwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int naive_bwd_launch<__nv_bfloat16>(const BwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);

}  // namespace gspn
