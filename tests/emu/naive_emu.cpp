// naive_emu.cpp -- TEST ONLY.  Runs the DEVICE code of the naive kernels (paper_2606_00746_b200/csrc/gspn_naive.cuh, the
// file the library compiles with nvcc) on the host: compiled with g++ against tests/emu/shim (a few lines standing in for
// the CUDA headers) and tests/emu/emu_rt.h: one thread block at a time, its threads as host threads.  It exists
// so that a change to those kernels can be checked against the oracle on a machine without a GPU
// (tests/test_naive_emulated_cpu.py).  It is not a CPU path of the library: nothing under paper_2606_00746_b200/ knows
// about it, and it emulates nothing but the naive kernels' plain threadIdx / __syncthreads / shared-memory model.
#include <cuda_runtime.h>

#include "gspn_naive.cuh"

namespace gspn {
alignas(16) float smem[1 << 16];      // dynamic shared memory of the running block (256 KB; a real CTA has 227 KB)
}

template <typename F>
static void run_grid(unsigned blocks, unsigned threads, F kernel) {
    emu::launch(dim3(blocks), dim3(threads), reinterpret_cast<unsigned char*>(gspn::smem), sizeof(gspn::smem), kernel);
}

static int round_up32(int v) { return (v + 31) / 32 * 32; }

// ws: NULL (plane-sized arrays in shared memory) or the global scratch of the large-plane mode (naive_workspace_bytes)
template <typename ST>
static int fwd_t(const void* x, const void* w3, const void* lam, const void* u, const void* h0, void* y, gspn::Shape sh, float* ws) {
    gspn::FwdArgs<ST> a{(const ST*)x, (const ST*)w3, (const ST*)lam, (const ST*)u, (const ST*)h0, (ST*)y, sh};
    if ((sh.plane() + 2 * (sh.Lmax() + 2)) > sizeof(gspn::smem) / 4) return 2;
    run_grid(sh.B * sh.C, round_up32(sh.Lmax()), [=] { gspn::naive_fwd_kernel<ST>(a, ws); });      // grid / block of naive_fwd_launch
    return emu::failed.load() ? 5 : 0;
}

template <typename ST>
static int bwd_t(const void* x, const void* w3, const void* lam, const void* u, const void* h0, const void* dy, void* dx,
                 void* dlam, void* du, void* dw3, void* dh0, gspn::Shape sh, float* ws) {
    gspn::BwdArgs<ST> a{(const ST*)x, (const ST*)w3, (const ST*)lam, (const ST*)u, (const ST*)h0, (const ST*)dy,
                        (ST*)dx, (ST*)dlam, (ST*)du, (ST*)dw3, (ST*)dh0, sh};
    if ((4 * sh.plane() + 3 * (sh.Lmax() + 2)) > sizeof(gspn::smem) / 4) return 2;
    // the two launches of naive_bwd_launch, same grids and blocks
    if (a.dx || a.dlam || a.du || a.dh0)
        run_grid(sh.B * sh.C, round_up32(sh.Lmax()), [=] { gspn::naive_bwd_main_kernel<ST>(a, ws); });
    if (a.dw3)
        run_grid(sh.D() * sh.B * sh.G, round_up32(sh.Lmax()), [=] { gspn::naive_bwd_dw_kernel<ST>(a, ws); });
    return emu::failed.load() ? 5 : 0;
}

extern "C" {

// dtype: 0 fp32, 1 bf16 (include/gspn.h); shared: bits of gspn::kShared*; k_chunk, flags as in gspn_args_t
int emu_naive_fwd(const void* x, const void* w3, const void* lam, const void* u, const void* h0, void* y, int B, int C, int H,
                  int W, int G, unsigned mask, unsigned shared, int k_chunk, unsigned flags, int dtype, float* ws) {
    const gspn::Shape sh{B, C, H, W, G, mask, shared, k_chunk, flags};
    return dtype == 0 ? fwd_t<float>(x, w3, lam, u, h0, y, sh, ws) : fwd_t<__nv_bfloat16>(x, w3, lam, u, h0, y, sh, ws);
}

int emu_naive_bwd(const void* x, const void* w3, const void* lam, const void* u, const void* h0, const void* dy, void* dx,
                  void* dlam, void* du, void* dw3, void* dh0, int B, int C, int H, int W, int G, unsigned mask,
                  unsigned shared, int k_chunk, unsigned flags, int dtype, float* ws) {
    const gspn::Shape sh{B, C, H, W, G, mask, shared, k_chunk, flags};
    return dtype == 0 ? bwd_t<float>(x, w3, lam, u, h0, dy, dx, dlam, du, dw3, dh0, sh, ws)
                      : bwd_t<__nv_bfloat16>(x, w3, lam, u, h0, dy, dx, dlam, du, dw3, dh0, sh, ws);
}

}  // extern "C"
