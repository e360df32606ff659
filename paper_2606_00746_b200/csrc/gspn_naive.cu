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

template <typename ST>
int naive_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    const Shape& sh = a.sh;
    if (sh.Lmax() > 1024) { set_error("naive fwd: max(H,W) = %d > 1024", sh.Lmax()); return GSPN_EUNSUPPORTED; }
    const size_t smem = (sh.plane() + 2 * (sh.Lmax() + 2)) * sizeof(float);
    int rc = prep_smem(naive_fwd_kernel<ST>, smem, "naive fwd");
    if (rc) return rc;
    naive_fwd_kernel<ST><<<sh.B * sh.C, round_up32(sh.Lmax()), smem, st>>>(a);
    li->launches = 1;
    li->variant = "naive_fwd";
    return check_launch("naive fwd");
}

template <typename ST>
int naive_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li) {
    const Shape& sh = a.sh;
    if (sh.Lmax() > 1024) { set_error("naive bwd: max(H,W) = %d > 1024", sh.Lmax()); return GSPN_EUNSUPPORTED; }
    const size_t aux = 3 * (sh.Lmax() + 2) * sizeof(float);
    li->launches = 0;
    li->variant = "naive_bwd";
    if (a.dx || a.dlam || a.du || a.dh0) {
        const size_t smem = 2 * sh.plane() * sizeof(float) + aux;
        int rc = prep_smem(naive_bwd_main_kernel<ST>, smem, "naive bwd (dx,dlambda,du,dh0)");
        if (rc) return rc;
        naive_bwd_main_kernel<ST><<<sh.B * sh.C, round_up32(sh.Lmax()), smem, st>>>(a);
        ++li->launches;
        rc = check_launch("naive bwd main");
        if (rc) return rc;
    }
    if (a.dw3) {
        const size_t smem = 4 * sh.plane() * sizeof(float) + aux;
        int rc = prep_smem(naive_bwd_dw_kernel<ST>, smem, "naive bwd (dw3)");
        if (rc) return rc;
        naive_bwd_dw_kernel<ST><<<sh.D() * sh.B * sh.G, round_up32(sh.Lmax()), smem, st>>>(a);
        ++li->launches;
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
