// plane_bwd_emu.cpp -- TEST ONLY.  csrc/gspn_plane_bwd.cu (kernel and launcher) built for the host with GSPN_EMU; see line_fwd_emu.cpp and emu_rt.h.
#define GSPN_EMU 1
#include <cuda_runtime.h>
namespace gspn { extern unsigned char smem_plane_bwd[]; }
#define GSPN_EMU_SMEM (::gspn::smem_plane_bwd)
#define smem smem_plane_bwd
#include "gspn_plane_bwd.cu"
#undef smem
namespace gspn { alignas(1024) unsigned char smem_plane_bwd[227 * 1024]; }

template <typename ST>
static int run(const void* x, const void* w3, const void* lam, const void* u, const void* h0, const void* dy, void* dx, void* dlam,
               void* du, void* dw3, void* dh0, gspn::Shape sh) {
    gspn::BwdArgs<ST> a{(const ST*)x, (const ST*)w3, (const ST*)lam, (const ST*)u, (const ST*)h0, (const ST*)dy,
                        (ST*)dx, (ST*)dlam, (ST*)du, (ST*)dw3, (ST*)dh0, sh};
    gspn::LaunchInfo li{0, ""};
    return gspn::plane_bwd_launch<ST>(a, nullptr, &li);
}
extern "C" int emu_plane_bwd(const void* x, const void* w3, const void* lam, const void* u, const void* h0, const void* dy, void* dx,
                      void* dlam, void* du, void* dw3, void* dh0, int B, int C, int H, int W, int G, unsigned mask, int dtype,
                      double wait_limit_s) {
    emu::wait_limit_s = wait_limit_s;
    const gspn::Shape sh{B, C, H, W, G, mask};
    return dtype == 0 ? run<float>(x, w3, lam, u, h0, dy, dx, dlam, du, dw3, dh0, sh)
                      : run<__nv_bfloat16>(x, w3, lam, u, h0, dy, dx, dlam, du, dw3, dh0, sh);
}
