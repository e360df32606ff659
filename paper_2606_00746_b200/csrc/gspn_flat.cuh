// gspn_flat.cuh -- pieces shared by the "flat" fused kernels (gspn_flat_fwd.cu, gspn_flat_bwd.cu):
// the kernels that take ANY H, W and storage type, including rows and planes that are not
// 16-byte aligned (W = 27, 73 in bf16: BASELINE.json configs 3 and 5).
//
// How operands reach the SM.  A CTA owns `nch` channels of one (b, group)
// unit; per direction it needs np = 3 + 3*nch operand planes (3 tap planes of w3, then lambda, u, x
// (forward) of its channels).  No tensor map can describe planes whose row pitch is not a multiple
// of 16 bytes, and TMA refuses box coordinates that are not 16-byte aligned (measured: illegal
// instruction), so the flat kernels move raw 16-byte-aligned SUPERSETS and index them with the
// byte phase of each plane:
//   vertical   (T->B, B->T): a ring of row blocks.  One stage = Kv image rows of every plane, one
//              1-D bulk copy (cp.async.bulk, mbarrier complete_tx) per plane covering
//              [floor16(first byte), ceil16(last byte)).
//   horizontal (L->R, R->L): a ring of "chunk columns".  One stage = for every (plane, row) the q-th
//              16-byte chunk of that row (counted from the chunk holding the row's first element),
//              gathered with 16-byte cp.async by a producer warp; a row keeps NSh+1 chunk slots
//              contiguous in shared memory (slot NSh duplicates slot 0), so the 2-chunk window a
//              row needs for one block of 16/ES columns is always contiguous and a lane reads its
//              elements with immediate offsets -- the transposed-tile path for unaligned rows.
// The few bytes of a tensor that lie beyond its last whole 16-byte chunk are copied with ordinary
// loads by the producer (never read past the end of an operand).
#pragma once

#include "gspn_fused.cuh"

namespace gspn {

#ifndef GSPN_EMU      // (tests/emu/emu_ptx.h stands in for the PTX wrappers, see gspn_fused.cuh)
// 16-byte cp.async (LDGSTS) global -> shared
__device__ __forceinline__ void cp_async_16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
// makes `bar` observe the completion of all cp.async issued so far by this thread (count pre-armed)
__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// one storage element from shared memory, widened to fp32
template <typename ST> __device__ __forceinline__ float lds_f(uint32_t addr);
template <> __device__ __forceinline__ float lds_f<float>(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
template <> __device__ __forceinline__ float lds_f<__nv_bfloat16>(uint32_t addr) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
    return __uint_as_float(((uint32_t)v) << 16);
}
__device__ __forceinline__ float lds_f32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_f32(uint32_t addr, float v) {
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
#endif  // GSPN_EMU

__device__ __forceinline__ int warp_sum(int v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// global plane bookkeeping of one operand plane of a stage
struct PlaneRef {
    const uint8_t* base;      // tensor base (16-byte aligned)
    unsigned long long e0;    // first element of the plane inside the tensor
    unsigned long long tbytes; // bytes of the whole tensor
};

}  // namespace gspn
