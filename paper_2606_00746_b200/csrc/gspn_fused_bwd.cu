// placeholder, replaced by the fused backward kernel
#include "gspn_kernels.h"
#include "../../include/gspn.h"
namespace gspn {
template <typename ST> int fused_bwd_launch(const BwdArgs<ST>&, cudaStream_t, LaunchInfo*) {
    set_error("fused bwd: not built"); return GSPN_EUNSUPPORTED;
}
template int fused_bwd_launch<float>(const BwdArgs<float>&, cudaStream_t, LaunchInfo*);
template int fused_bwd_launch<__nv_bfloat16>(const BwdArgs<__nv_bfloat16>&, cudaStream_t, LaunchInfo*);
}
