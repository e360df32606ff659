// gspn_line.cuh -- shared pieces of the "line" kernels (gspn_line_fwd.cu, gspn_line_bwd.cu): rows that are
// 16-byte aligned, one warp per (channel, direction) scan line, P adjacent positions per lane, operand stages of
// kLineSteps scan steps brought by TMA tensor maps and consumed with vector loads.
//
// Geometry (include/gspn.h): scan step s, cross position p.  T->B / B->T: a stage is kLineSteps image rows, a lane
// owns the P adjacent columns P*lane .. P*lane+P-1 and reads them with one P*ES-byte load per operand and step.
// L->R / R->L (the transposed tile): a stage is kLineSteps image columns = NCH 16-byte column
// chunks; a lane owns the P adjacent rows P*lane .. P*lane+P-1.  The tensor map splits the row index into
// (row / P, row % P) and orders the box as [chunk][row % P][row / P][16 B], so that the lanes of a warp read
// consecutive 16-byte pieces (no bank conflict) and each piece holds 16/ES scan steps of one operand.
#pragma once

#include "gspn_fused.cuh"

namespace gspn {

constexpr int kLineSteps = 8;          // scan steps per ring stage
constexpr int kLineStages = 3;         // ring stages per direction

// pitch (in floats) of a scratch / accumulator row: a multiple of 4 whose quarter is odd, so that lanes one pitch apart
// reading 16 bytes each fall into different banks
static inline int line_pitch(int W) {
    int p = (W + 3) / 4 * 4;
    if ((p / 4) % 2 == 0) p += 4;
    return p;
}

// P storage elements from shared memory, widened to fp32
template <typename ST, int P> __device__ __forceinline__ void line_ld(const ST* p, float (&f)[P]) {
    if constexpr (sizeof(ST) == 4) {
        ldf<P>(reinterpret_cast<const float*>(p), f);
    } else if constexpr (P == 1) {
        f[0] = __uint_as_float(((uint32_t)*reinterpret_cast<const unsigned short*>(p)) << 16);
    } else {
        uint32_t r[P / 2];
        lds_vec<2 * P>(p, r);
        Store<__nv_bfloat16>::template unpack<2 * P>(r, f);
    }
}

// 16 bytes = K storage elements, widened
template <typename ST> __device__ __forceinline__ void line_ld16(const void* p, float (&f)[16 / sizeof(ST)]) {
    uint32_t r[4];
    lds_vec<16>(p, r);
    Store<ST>::template unpack<16>(r, f);
}

// element e (compile-time) of a raw 16-byte piece, widened
template <typename ST> __device__ __forceinline__ float line_elem(const uint32_t (&w)[4], int e) {
    if constexpr (sizeof(ST) == 4) return __uint_as_float(w[e]);
    else return (e & 1) ? __uint_as_float(w[e >> 1] & 0xffff0000u) : __uint_as_float(w[e >> 1] << 16);
}

#ifndef GSPN_EMU      // (tests/emu/emu_ptx.h stands in for the PTX wrappers, see gspn_fused.cuh)
// spinning wait (mbarrier.test_wait never suspends the thread)
__device__ __forceinline__ void mbar_wait_spin(uint64_t* b, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "GSPN_SPIN:\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra GSPN_SPIN_DONE;\n"
        "bra GSPN_SPIN;\n"
        "GSPN_SPIN_DONE:\n"
        "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}

// ---- tensor memory (TMEM) as the fp32 accumulator store ----------------------------------------------------------
// 128 lanes x 512 columns x 32 bit per SM; warp w of a CTA reaches lanes 32*(w % 4) .. +31, one lane per thread
// (shape 32x32b: thread t reads / writes N consecutive columns of its own lane).  Addresses: lane << 16 | column.
// No "memory" clobber: these do not touch shared or global memory, and the operand loads must stay free to move.
template <int N> __device__ __forceinline__ void tm_ld(uint32_t ta, float (&f)[N]) {
    static_assert(N == 1 || N == 2 || N == 4 || N == 8 || N == 16 || N == 32, "tm_ld: N");
    if constexpr (N == 1)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(f[0]) : "r"(ta));
    if constexpr (N == 2)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=f"(f[0]), "=f"(f[1]) : "r"(ta));
    if constexpr (N == 4)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=f"(f[0]), "=f"(f[1]), "=f"(f[2]), "=f"(f[3]) : "r"(ta));
    if constexpr (N == 8)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];" : "=f"(f[0]), "=f"(f[1]), "=f"(f[2]), "=f"(f[3]), "=f"(f[4]), "=f"(f[5]), "=f"(f[6]), "=f"(f[7]) : "r"(ta));
    if constexpr (N == 16)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];" : "=f"(f[0]), "=f"(f[1]), "=f"(f[2]), "=f"(f[3]), "=f"(f[4]), "=f"(f[5]), "=f"(f[6]), "=f"(f[7]), "=f"(f[8]), "=f"(f[9]), "=f"(f[10]), "=f"(f[11]), "=f"(f[12]), "=f"(f[13]), "=f"(f[14]), "=f"(f[15]) : "r"(ta));
    if constexpr (N == 32)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];" : "=f"(f[0]), "=f"(f[1]), "=f"(f[2]), "=f"(f[3]), "=f"(f[4]), "=f"(f[5]), "=f"(f[6]), "=f"(f[7]), "=f"(f[8]), "=f"(f[9]), "=f"(f[10]), "=f"(f[11]), "=f"(f[12]), "=f"(f[13]), "=f"(f[14]), "=f"(f[15]), "=f"(f[16]), "=f"(f[17]), "=f"(f[18]), "=f"(f[19]), "=f"(f[20]), "=f"(f[21]), "=f"(f[22]), "=f"(f[23]), "=f"(f[24]), "=f"(f[25]), "=f"(f[26]), "=f"(f[27]), "=f"(f[28]), "=f"(f[29]), "=f"(f[30]), "=f"(f[31]) : "r"(ta));
}
template <int N> __device__ __forceinline__ void tm_st(uint32_t ta, const float (&f)[N]) {
    static_assert(N == 1 || N == 2 || N == 4 || N == 8 || N == 16 || N == 32, "tm_st: N");
    if constexpr (N == 1)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(ta), "f"(f[0]));
    if constexpr (N == 2)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(ta), "f"(f[0]), "f"(f[1]));
    if constexpr (N == 4)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(ta), "f"(f[0]), "f"(f[1]), "f"(f[2]), "f"(f[3]));
    if constexpr (N == 8)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(ta), "f"(f[0]), "f"(f[1]), "f"(f[2]), "f"(f[3]), "f"(f[4]), "f"(f[5]), "f"(f[6]), "f"(f[7]));
    if constexpr (N == 16)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(ta), "f"(f[0]), "f"(f[1]), "f"(f[2]), "f"(f[3]), "f"(f[4]), "f"(f[5]), "f"(f[6]), "f"(f[7]), "f"(f[8]), "f"(f[9]), "f"(f[10]), "f"(f[11]), "f"(f[12]), "f"(f[13]), "f"(f[14]), "f"(f[15]));
    if constexpr (N == 32)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(ta), "f"(f[0]), "f"(f[1]), "f"(f[2]), "f"(f[3]), "f"(f[4]), "f"(f[5]), "f"(f[6]), "f"(f[7]), "f"(f[8]), "f"(f[9]), "f"(f[10]), "f"(f[11]), "f"(f[12]), "f"(f[13]), "f"(f[14]), "f"(f[15]), "f"(f[16]), "f"(f[17]), "f"(f[18]), "f"(f[19]), "f"(f[20]), "f"(f[21]), "f"(f[22]), "f"(f[23]), "f"(f[24]), "f"(f[25]), "f"(f[26]), "f"(f[27]), "f"(f[28]), "f"(f[29]), "f"(f[30]), "f"(f[31]));
}
// wait for the loads of this thread; the loaded registers are operands so that no use of them can move above the wait
template <int N> __device__ __forceinline__ void tm_wait_ld(float (&f)[N]) {
    if constexpr (N == 1) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(f[0]));
    if constexpr (N == 2) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(f[0]), "+f"(f[1]));
    if constexpr (N == 4) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(f[0]), "+f"(f[1]), "+f"(f[2]), "+f"(f[3]));
    if constexpr (N == 8) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(f[0]), "+f"(f[1]), "+f"(f[2]), "+f"(f[3]), "+f"(f[4]), "+f"(f[5]), "+f"(f[6]), "+f"(f[7]));
    if constexpr (N == 16) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(f[0]), "+f"(f[1]), "+f"(f[2]), "+f"(f[3]), "+f"(f[4]), "+f"(f[5]), "+f"(f[6]), "+f"(f[7]), "+f"(f[8]), "+f"(f[9]), "+f"(f[10]), "+f"(f[11]), "+f"(f[12]), "+f"(f[13]), "+f"(f[14]), "+f"(f[15]));
    if constexpr (N == 32) asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(f[0]), "+f"(f[1]), "+f"(f[2]), "+f"(f[3]), "+f"(f[4]), "+f"(f[5]), "+f"(f[6]), "+f"(f[7]), "+f"(f[8]), "+f"(f[9]), "+f"(f[10]), "+f"(f[11]), "+f"(f[12]), "+f"(f[13]), "+f"(f[14]), "+f"(f[15]), "+f"(f[16]), "+f"(f[17]), "+f"(f[18]), "+f"(f[19]), "+f"(f[20]), "+f"(f[21]), "+f"(f[22]), "+f"(f[23]), "+f"(f[24]), "+f"(f[25]), "+f"(f[26]), "+f"(f[27]), "+f"(f[28]), "+f"(f[29]), "+f"(f[30]), "+f"(f[31]));
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;"); }
__device__ __forceinline__ void tm_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// one warp allocates `cols` columns (a power of two >= 32) for the CTA and publishes the base address in shared memory
__device__ __forceinline__ void tm_alloc(uint32_t* slot, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tm_dealloc(uint32_t base, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(cols) : "memory");
}
#endif  // GSPN_EMU
// the two warps of a channel meet: tensor-memory writes of one are visible to the other afterwards
__device__ __forceinline__ void tm_pair_sync(int id) {
    tm_wait_st();
    tm_fence_before();
    named_bar_sync(id, 64);
    tm_fence_after();
}

// ---- TMA stores shared -> global (tiled), bulk-group completion --------------------------------------------------
#ifndef GSPN_EMU
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* m, const void* src, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
                 ::"l"(m), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap* m, const void* src, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"(m), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* m, int c0, int c1, int c2, int c3, int c4,
                                            uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}
// fma.rn.f32.bf16 (SASS FHFMA.BF16): c + a * b with a, b the low or the high bf16 half of a 32-bit word, no widening
__device__ __forceinline__ float fma_bf16_half(uint32_t a, uint32_t b, bool high, float c) {
    float d;
    if (high)
        asm("{ .reg .b16 al, ah, bl, bh;\n mov.b32 {al, ah}, %1;\n mov.b32 {bl, bh}, %2;\n fma.rn.f32.bf16 %0, ah, bh, %3; }"
            : "=f"(d) : "r"(a), "r"(b), "f"(c));
    else
        asm("{ .reg .b16 al, ah, bl, bh;\n mov.b32 {al, ah}, %1;\n mov.b32 {bl, bh}, %2;\n fma.rn.f32.bf16 %0, al, bl, %3; }"
            : "=f"(d) : "r"(a), "r"(b), "f"(c));
    return d;
}
#endif  // GSPN_EMU

// raw storage words of P elements (lambda and x are multiplied without widening: one FHFMA.BF16 per position)
template <typename ST, int P> struct LineRaw { uint32_t w[(P * sizeof(ST) + 3) / 4]; };
template <typename ST, int P> __device__ __forceinline__ void line_ld_raw(const ST* p, LineRaw<ST, P>& r) {
    if constexpr (P * sizeof(ST) == 2) r.w[0] = *reinterpret_cast<const unsigned short*>(p);
    else lds_vec<P * sizeof(ST)>(p, r.w);
}
// c + a[k] * b[k] on raw storage words
template <typename ST> __device__ __forceinline__ float line_fma_raw(const uint32_t* a, const uint32_t* b, int k, float c) {
    if constexpr (sizeof(ST) == 4) {
        return fmaf(__uint_as_float(a[k]), __uint_as_float(b[k]), c);
    } else {
        return fma_bf16_half(a[k >> 1], b[k >> 1], (k & 1) != 0, c);      // k is a compile-time constant after unrolling
    }
}

// the plane of one channel turns from the column-owner layout into the row-owner layout (one warp, in place)
template <int P>
__device__ __forceinline__ void line_transpose(uint32_t tb, float* tile, int pitch, int H, int W, int lane) {
    const int WP = W / P;
    for (int t = 0; t * 32 < H; ++t) {
#pragma unroll
        for (int r8 = 0; r8 < 4; ++r8) {
            float f[8 * P];                                   // rows 32t + 8*r8 + r, columns P*lane + k
            tm_ld<8 * P>(tb + (32 * t + 8 * r8) * P, f);
            tm_wait_ld<8 * P>(f);
            if (lane < WP) {
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    float g[P];
#pragma unroll
                    for (int k = 0; k < P; ++k) g[k] = f[r * P + k];
                    stf<P>(tile + (8 * r8 + r) * pitch + P * lane, g);
                }
            }
        }
        __syncwarp();
        const float* row = tile + lane * pitch;               // image row 32t + lane
        int j0 = 0;
        for (; j0 + 32 <= W; j0 += 32) {
            float f[32];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float4 v = *reinterpret_cast<const float4*>(row + j0 + 4 * q);
                f[4 * q] = v.x; f[4 * q + 1] = v.y; f[4 * q + 2] = v.z; f[4 * q + 3] = v.w;
            }
            tm_st<32>(tb + t * 32 * P + j0, f);
        }
        for (; j0 + 4 <= W; j0 += 4) {
            float f[4];
            ldf<4>(row + j0, f);
            tm_st<4>(tb + t * 32 * P + j0, f);
        }
        tm_wait_st();
        __syncwarp();
    }
}


}  // namespace gspn
