// flat_fwd_emu.cpp -- TEST ONLY.  csrc/gspn_flat_fwd.cu (kernel and launcher) built for the host with GSPN_EMU; see line_fwd_emu.cpp and emu_rt.h.
#define GSPN_EMU 1
#include <cuda_runtime.h>
namespace gspn { extern unsigned char smem_flat_fwd[]; }
#define GSPN_EMU_SMEM (::gspn::smem_flat_fwd)
#define smem smem_flat_fwd
#include "gspn_flat_fwd.cu"
#undef smem
namespace gspn { alignas(1024) unsigned char smem_flat_fwd[227 * 1024]; }

template <typename ST>
static int run(const void* x, const void* w3, const void* lam, const void* u, const void* h0, void* y, gspn::Shape sh) {
    gspn::FwdArgs<ST> a{(const ST*)x, (const ST*)w3, (const ST*)lam, (const ST*)u, (const ST*)h0, (ST*)y, sh};
    gspn::LaunchInfo li{0, ""};
    return gspn::flat_fwd_launch<ST>(a, nullptr, &li);
}
extern "C" int emu_flat_fwd(const void* x, const void* w3, const void* lam, const void* u, const void* h0, void* y, int B, int C, int H,
                      int W, int G, unsigned mask, int dtype, double wait_limit_s) {
    emu::wait_limit_s = wait_limit_s;
    const gspn::Shape sh{B, C, H, W, G, mask};
    return dtype == 0 ? run<float>(x, w3, lam, u, h0, y, sh) : run<__nv_bfloat16>(x, w3, lam, u, h0, y, sh);
}
