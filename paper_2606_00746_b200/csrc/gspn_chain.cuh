// gspn_chain.cuh -- pieces shared by the "chain" kernels of libgspn (gspn_chain_bwd.cu,
// gspn_chain_fwd.cu): one WARP runs one scan chain (direction d, channel c) with the hidden state of
// Eq. (1) in registers, neighbours by warp shuffle, and no block barrier on the serial
// path.  Operands reach shared memory asynchronously through a ring of stages filled by one producer
// warp (row blocks for T->B / B->T, chunk columns for L->R / R->L: the transposed tile), exactly as
// they lie in HBM: 16-byte-aligned supersets for rows that are not 16-byte aligned (gspn_flat.cuh
// explains why TMA tensor maps cannot realign them).
//
// Storage-type access.  bf16 operands are read as 16-bit scalars and used WITHOUT a widening
// instruction wherever both factors are storage values: sm_100a's mixed-precision FMA
// (PTX fma.rn.f32.bf16, SASS FHFMA.BF16) computes fp32 = bf16*bf16 + fp32 in one instruction, so
// lambda*x (forward) and dy*u (backward) cost one issue slot each.
#pragma once

#include "gspn_flat.cuh"

namespace gspn {

constexpr int kBlk = 4;            // scan steps per block = checkpoint interval = ring stage (lines / chunk columns)
constexpr int kChSlots = 8;        // mbarrier pairs (ring slots) available

#ifndef GSPN_EMU      // (tests/emu/emu_ptx.h stands in for Elem, cp_async_cb, l2_prefetch_bulk, chain_bar, lds32, sts32)
template <typename ST> struct Elem;
template <> struct Elem<__nv_bfloat16> {
    using raw_t = unsigned short;
    static __device__ __forceinline__ raw_t lds(uint32_t a) {
        raw_t v;
        asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
        return v;
    }
    static __device__ __forceinline__ void sts(uint32_t a, raw_t v) {
        asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"(v));
    }
    static __device__ __forceinline__ float f(raw_t r) { return __uint_as_float(((uint32_t)r) << 16); }
    // fp32 = a*b + c with a, b storage values: one FHFMA.BF16
    static __device__ __forceinline__ float fma2(raw_t a, raw_t b, float c) {
        float d;
        asm("fma.rn.f32.bf16 %0, %1, %2, %3;" : "=f"(d) : "h"(a), "h"(b), "f"(c));
        return d;
    }
    static __device__ __forceinline__ raw_t pack(float v) { return __bfloat16_as_ushort(__float2bfloat16_rn(v)); }
    static __device__ __forceinline__ void stg(__nv_bfloat16* p, raw_t v) { *reinterpret_cast<raw_t*>(p) = v; }
};
template <> struct Elem<float> {
    using raw_t = float;
    static __device__ __forceinline__ raw_t lds(uint32_t a) {
        raw_t v;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
        return v;
    }
    static __device__ __forceinline__ void sts(uint32_t a, raw_t v) {
        asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v));
    }
    static __device__ __forceinline__ float f(raw_t r) { return r; }
    static __device__ __forceinline__ float fma2(raw_t a, raw_t b, float c) { return fmaf(a, b, c); }
    static __device__ __forceinline__ raw_t pack(float v) { return v; }
    static __device__ __forceinline__ void stg(float* p, raw_t v) { *p = v; }
};

// cp.async of CB = 8 or 16 bytes (source and destination CB-aligned)
template <int CB> __device__ __forceinline__ void cp_async_cb(uint32_t dst, const void* src);
template <> __device__ __forceinline__ void cp_async_cb<8>(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
template <> __device__ __forceinline__ void cp_async_cb<16>(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}

// L2 prefetch of [p, p+bytes): p 16-byte aligned, bytes a multiple of 16 (cp.async.bulk.prefetch.L2).  The
// producers announce the operand planes of a direction before they stream them in small stages, so the
// stage copies find their lines in L2 instead of paying the DRAM latency once per stage.
__device__ __forceinline__ void l2_prefetch_bulk(const void* p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
#endif  // GSPN_EMU
// prefetch the 16-byte-aligned superset of plane e (HWB bytes long) that lies inside its tensor
__device__ __forceinline__ void l2_prefetch_plane(const uint8_t* base, unsigned long long b0, unsigned long long tbytes,
                                                  unsigned long long HWB) {
    const unsigned long long a0 = b0 & ~15ull;
    unsigned long long a1 = (b0 + HWB + 15) & ~15ull;
    const unsigned long long lim = tbytes & ~15ull;
    if (a1 > lim) a1 = lim;
    if (a1 > a0) l2_prefetch_bulk(base + a0, (uint32_t)(a1 - a0));
}

// named barrier among the chain warps of a CTA (the producer warp does not take part)
__device__ __forceinline__ void chain_bar(int nthreads) { named_bar_sync(1, nthreads); }

struct ChPlane {                  // one operand plane of one direction (table in shared memory)
    const uint8_t* base;          // tensor base (16-byte aligned)
    unsigned long long b0;        // first byte of the plane inside the tensor
    unsigned long long tbytes;    // bytes of the whole tensor
};

__device__ __forceinline__ float maskf(float v, uint32_t m) { return __uint_as_float(__float_as_uint(v) & m); }
#ifndef GSPN_EMU
__device__ __forceinline__ float lds32(uint32_t a) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v)); }
#endif

// ---------------------------------------------------------------------------------------------------
// Ring hand-shake of a consumer warp.  Block bi (image lines [4bi, 4bi+4)) needs row block bi
// (vertical) or chunk columns bi and bi+1 (horizontal).  Every consumer warp of the CTA acquires and
// releases every stage, whether its role has work in it or not, so the mbarrier phases stay aligned.
template <bool VH>
struct RingSync {
    uint64_t *full, *empty;
    int NSV, NSH, NQ, lane, hq;
    uint32_t pf;
    __device__ __forceinline__ void wait_full(int slot) {
        mbar_wait(&full[slot], (pf >> slot) & 1u);
        pf ^= 1u << slot;
    }
    __device__ __forceinline__ void begin_pass(bool desc) { hq = desc ? NQ - 1 : 0; }
    __device__ __forceinline__ void acquire(int bi, bool desc) {
        if constexpr (!VH) {
            wait_full(bi % NSV);
        } else if (!desc) {
            const int need = min(bi + 1, NQ - 1);
            for (; hq <= need; ++hq) wait_full(hq % NSH);
        } else {
            for (; hq >= bi; --hq) wait_full(hq % NSH);
        }
    }
    __device__ __forceinline__ void release(int bi, bool desc, bool last) {
        __syncwarp();
        if (lane == 0) {
            if constexpr (!VH) {
                mbar_arrive(&empty[bi % NSV]);
            } else if (!desc) {
                mbar_arrive(&empty[bi % NSH]);
                if (last) for (int qq = bi + 1; qq < NQ; ++qq) mbar_arrive(&empty[qq % NSH]);
            } else {
                if (bi + 1 < NQ) mbar_arrive(&empty[(bi + 1) % NSH]);
                if (last) mbar_arrive(&empty[bi % NSH]);
            }
        }
    }
};

}  // namespace gspn
