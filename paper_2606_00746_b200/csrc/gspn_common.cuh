// gspn_common.cuh -- shared device helpers of libgspn (storage-type conversion, direction
// indexing, launch bookkeeping).  Notation follows PAPER.md Sec. 3 (lines 82-99): scan step s,
// cross position p, image pixel (i,j); see include/gspn.h for the operator and the layouts.
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gspn {

// ---- storage types: every tensor is stored as ST, all arithmetic is fp32 -------------------
__device__ __forceinline__ float ld_f(const float* p) { return __ldg(p); }
__device__ __forceinline__ float ld_f(const __nv_bfloat16* p) {
    return __uint_as_float(((uint32_t)__ldg(reinterpret_cast<const unsigned short*>(p))) << 16);
}
__device__ __forceinline__ void st_f(float* p, float v) { *p = v; }
__device__ __forceinline__ void st_f(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }

// ---- direction geometry (include/gspn.h): dir 0 T->B, 1 B->T, 2 L->R, 3 R->L -----------------
// offset inside one [H,W] plane of scan step s, cross position p
__device__ __forceinline__ int img_off(int dir, int s, int p, int H, int W) {
    switch (dir) {
    case 0:  return s * W + p;
    case 1:  return (H - 1 - s) * W + p;
    case 2:  return p * W + s;
    default: return p * W + (W - 1 - s);
    }
}

constexpr unsigned kSharedW3 = 1u, kSharedLam = 2u, kSharedU = 4u;
constexpr unsigned kFlagLogits = 1u;

struct Shape {
    int B, C, H, W, G;
    unsigned mask;
    // operands whose direction slabs are ONE slab read by every direction (gspn_args_t.dir_stride_* == 0, DESIGN.md
    // reading 6): bits kSharedW3 / kSharedLam / kSharedU.  0 = the dense [D, ...] layout.  Outputs are never shared.
    unsigned shared;
    // chunked scan (gspn_args_t.k_chunk, reading 10): bands of ceil(L / k_chunk) lines of the scan axis in image
    // coordinates, each an independent scan with a zero initial state.  0 or 1 = one band (the global scan).
    int k_chunk;
    // kFlagLogits: `w3` holds the raw tap LOGITS and Eq. 3 is applied where the taps are loaded (gspn_args_t.flags,
    // SURVEY 8(f) f1, second half); the backward then writes the gradient of the logits to dw3
    unsigned flags;
    __host__ __device__ bool logits() const { return (flags & 1u) != 0; }
    __host__ __device__ int band(int Ls) const { const int k = k_chunk > 1 ? k_chunk : 1; return (Ls + k - 1) / k; }
    __host__ __device__ int cg() const { return C / G; }
    __host__ __device__ int Lmax() const { return H > W ? H : W; }
    __host__ __device__ size_t plane() const { return (size_t)H * W; }
    __host__ __device__ int D() const {
        return (int)((mask & 1) + (mask >> 1 & 1) + (mask >> 2 & 1) + (mask >> 3 & 1));
    }
};

// operand pointers of one call (device memory, layouts of include/gspn.h)
template <typename ST>
struct FwdArgs {
    const ST *x, *w3, *lam, *u, *h0;
    ST* y;
    Shape sh;
    float* ws;            // caller workspace (gspn_args_t.workspace) or NULL, and its size
    size_t ws_bytes;
};

template <typename ST>
struct BwdArgs {
    const ST *x, *w3, *lam, *u, *h0, *dy;
    ST *dx, *dlam, *du, *dw3, *dh0;
    Shape sh;
    float* ws;
    size_t ws_bytes;
};

// launch results reported back to the C ABI
struct LaunchInfo {
    int launches;
    const char* variant;
};

constexpr int kMaxSmemOptin = 227 * 1024;   // B200: 227 KB usable shared memory per CTA

// A kernel launch: the CUDA launch statement -- or, under tests/emu only (GSPN_EMU), the host emulation that runs the
// blocks one after another with host threads (the launchers are then checked together with their kernels: shared-memory
// layout, tensor maps, grid).
#ifdef GSPN_EMU
#define GSPN_LAUNCH(kern, grid, block, smem_bytes, stream, ...) \
    (void)emu::launch(dim3(grid), dim3(block), GSPN_EMU_SMEM, (size_t)(smem_bytes), [&] { kern(__VA_ARGS__); })
#else
#define GSPN_LAUNCH(kern, grid, block, smem_bytes, stream, ...) kern<<<grid, block, smem_bytes, stream>>>(__VA_ARGS__)
#endif

}  // namespace gspn
