// gspn_fused.cuh -- building blocks of the fused (single-launch) libgspn kernels for sm_100a:
// mbarrier / TMA (cp.async.bulk[.tensor]) wrappers, storage-type vector unpacking, and the host
// side tensor-map encoder (driver entry point fetched through the runtime, no -lcuda).
//
// Why TMA: the scan is HBM-bound and B200 needs >= 64 KB of loads in flight per SM
// to reach its copy bandwidth (measured); bulk copies keep that many
// bytes outstanding without holding registers or LSU issue slots.
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "gspn_common.cuh"

// GSPN_EMU is defined by tests/emu only: the PTX wrappers below are then replaced by host stand-ins of the same names
// (tests/emu/emu_ptx.h), so that the kernels written on top of them can be run, and their protocols checked, without a GPU.
#ifdef GSPN_EMU
#include "emu_ptx.h"
#endif

namespace gspn {

#ifndef GSPN_EMU
// ---- shared-memory addresses / mbarriers -----------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* b, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_init_fence() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "GSPN_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra GSPN_DONE;\n"
        "bra GSPN_WAIT;\n"
        "GSPN_DONE:\n"
        "}\n" ::"r"(smem_u32(b)),
        "r"(parity), "r"(0x989680)      // suspend-time hint: a waiting warp sleeps instead of spinning on issue slots
        : "memory");
}

// ---- TMA: tiled tensor copies global -> shared, completion on an mbarrier ---------------------
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* m, int c0, int c1, int c2,
                                            uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* m, int c0, int c1, int c2,
                                            int c3, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
// 1-D bulk copy (no tensor map): src and dst 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* m) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(m) : "memory");
}
// 1-D bulk store shared -> global (bulk-group completion): dst and src 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_store_1d(void* dst, const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// all but the newest N groups of this thread have finished READING shared memory
template <int N> __device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N> __device__ __forceinline__ void bulk_wait_all() {
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}
// named barrier `id` (1..15) among `nthreads` threads (whole warps) of the CTA
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// generic-proxy writes to shared memory are ordered before later async-proxy (bulk / TMA) accesses
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
#endif  // GSPN_EMU

// ---- storage vectors ---------------------------------------------------------------------------
// NB bytes (4, 8 or 16) of storage type ST read from shared memory and widened to fp32.
template <typename ST> struct Store { };
template <> struct Store<float> {
    static constexpr int ES = 4;
    template <int NB> __device__ static __forceinline__ void unpack(const uint32_t (&r)[NB / 4], float (&f)[NB / 4]) {
#pragma unroll
        for (int t = 0; t < NB / 4; ++t) f[t] = __uint_as_float(r[t]);
    }
    template <int NB> __device__ static __forceinline__ void pack(const float (&f)[NB / 4], uint32_t (&r)[NB / 4]) {
#pragma unroll
        for (int t = 0; t < NB / 4; ++t) r[t] = __float_as_uint(f[t]);
    }
};
template <> struct Store<__nv_bfloat16> {
    static constexpr int ES = 2;
    template <int NB> __device__ static __forceinline__ void unpack(const uint32_t (&r)[NB / 4], float (&f)[NB / 2]) {
#pragma unroll
        for (int t = 0; t < NB / 4; ++t) {
            f[2 * t] = __uint_as_float(r[t] << 16);              // bf16 -> fp32 is a 16-bit shift (exact)
            f[2 * t + 1] = __uint_as_float(r[t] & 0xffff0000u);
        }
    }
    template <int NB> __device__ static __forceinline__ void pack(const float (&f)[NB / 2], uint32_t (&r)[NB / 4]) {
#pragma unroll
        for (int t = 0; t < NB / 4; ++t) {
            __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * t], f[2 * t + 1]);   // one RNE per element
            r[t] = *reinterpret_cast<uint32_t*>(&h);
        }
    }
};

template <int NB> __device__ __forceinline__ void lds_vec(const void* p, uint32_t (&r)[NB / 4]) {
    if constexpr (NB == 16) {
        const uint4 v = *reinterpret_cast<const uint4*>(p);
        r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w;
    } else if constexpr (NB == 8) {
        const uint2 v = *reinterpret_cast<const uint2*>(p);
        r[0] = v.x; r[1] = v.y;
    } else {
        r[0] = *reinterpret_cast<const uint32_t*>(p);
    }
}
template <int NB> __device__ __forceinline__ void st_vec(void* p, const uint32_t (&r)[NB / 4]) {
    if constexpr (NB == 16) *reinterpret_cast<uint4*>(p) = make_uint4(r[0], r[1], r[2], r[3]);
    else if constexpr (NB == 8) *reinterpret_cast<uint2*>(p) = make_uint2(r[0], r[1]);
    else *reinterpret_cast<uint32_t*>(p) = r[0];
}
// N floats (N = 1, 2, 4 or 8) from / to 4N-byte aligned shared memory
template <int N> __device__ __forceinline__ void ldf(const float* p, float (&f)[N]) {
    if constexpr (N == 8) {
        const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
        f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w; f[4] = b.x; f[5] = b.y; f[6] = b.z; f[7] = b.w;
    } else if constexpr (N == 4) {
        const float4 a = *reinterpret_cast<const float4*>(p);
        f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w;
    } else if constexpr (N == 2) {
        const float2 a = *reinterpret_cast<const float2*>(p);
        f[0] = a.x; f[1] = a.y;
    } else {
        f[0] = *p;
    }
}
template <int N> __device__ __forceinline__ void stf(float* p, const float (&f)[N]) {
    if constexpr (N == 8) {
        *reinterpret_cast<float4*>(p) = make_float4(f[0], f[1], f[2], f[3]);
        *reinterpret_cast<float4*>(p + 4) = make_float4(f[4], f[5], f[6], f[7]);
    } else if constexpr (N == 4) {
        *reinterpret_cast<float4*>(p) = make_float4(f[0], f[1], f[2], f[3]);
    } else if constexpr (N == 2) {
        *reinterpret_cast<float2*>(p) = make_float2(f[0], f[1]);
    } else {
        *p = f[0];
    }
}

// ---- host: tensor maps --------------------------------------------------------------------------
// Encodes a tiled, unswizzled tensor map over `rank` dimensions (dims[0] is the contiguous one,
// strides_bytes[i] is the stride of dims[i+1]).  Returns false and sets the library error on failure.
#ifndef GSPN_EMU
bool encode_tensor_map(CUtensorMap* out, int es, void* base, int rank, const uint64_t* dims,
                       const uint64_t* strides_bytes, const uint32_t* box, int swizzle32 = 0);
#endif

static inline int round_up_int(int v, int m) { return (v + m - 1) / m * m; }

}  // namespace gspn
