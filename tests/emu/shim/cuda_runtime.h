// Shim of <cuda_runtime.h> for tests/emu (TEST ONLY): enough of the CUDA C++ vocabulary to compile the DEVICE code of this
// repository's kernels, and the few host calls of their launchers, with g++; the run time behind it is tests/emu/emu_rt.h.
#pragma once
#include <math.h>
#include <cstddef>
#include <cstdint>
#include <cstring>

#include "emu_rt.h"

#define __device__
#define __host__
#define __global__
#define __forceinline__ inline
#define __noinline__
#define __shared__
#define __restrict__
#define __grid_constant__
#define __launch_bounds__(...)
#define __align__(n)

struct uint2 { unsigned x, y; };
struct uint4 { unsigned x, y, z, w; };
struct float2 { float x, y; };
struct float4 { float x, y, z, w; };
inline uint2 make_uint2(unsigned x, unsigned y) { return uint2{x, y}; }
inline uint4 make_uint4(unsigned x, unsigned y, unsigned z, unsigned w) { return uint4{x, y, z, w}; }
inline float2 make_float2(float x, float y) { return float2{x, y}; }
inline float4 make_float4(float x, float y, float z, float w) { return float4{x, y, z, w}; }

#define threadIdx (emu::tid)
#define blockIdx (emu::bid)
#define blockDim (emu::bdim)
#define gridDim (emu::gdim)

inline void __syncthreads() { emu::sync_block(); }
inline void __syncwarp(unsigned mask = 0xffffffffu) {
    if (mask != 0xffffffffu) emu::fail("__syncwarp: partial mask 0x%x is not emulated", mask);
    emu::sync_warp();
}
template <typename T> inline T __ldg(const T* p) { return *p; }
inline float __uint_as_float(uint32_t v) { float f; std::memcpy(&f, &v, 4); return f; }
inline uint32_t __float_as_uint(float f) { uint32_t v; std::memcpy(&v, &f, 4); return v; }
template <typename T> inline T min(T a, T b) { return b < a ? b : a; }      // CUDA declares these at global scope
template <typename T> inline T max(T a, T b) { return a < b ? b : a; }

// PRMT: byte i of the result is byte (selector nibble i & 7) of {y:x}; nibble bit 3 replicates that byte's sign bit
inline unsigned __byte_perm(unsigned x, unsigned y, unsigned s) {
    const unsigned long long v = ((unsigned long long)y << 32) | x;
    unsigned r = 0;
    for (int i = 0; i < 4; ++i) {
        const unsigned sel = (s >> (4 * i)) & 0xfu;
        unsigned b = (unsigned)(v >> (8 * (sel & 7u))) & 0xffu;
        if (sel & 8u) b = (b & 0x80u) ? 0xffu : 0u;
        r |= b << (8 * i);
    }
    return r;
}

// warp shuffles, full mask only (every lane of the warp must execute them, as the hardware requires for the mask)
template <typename T> inline T emu_shfl(unsigned mask, T v, int src) {
    static_assert(sizeof(T) == 4, "shuffle of 32-bit values");
    if (mask != 0xffffffffu) emu::fail("shuffle: partial mask 0x%x is not emulated", mask);
    uint32_t raw; std::memcpy(&raw, &v, 4);
    raw = emu::shfl_raw(raw, src);
    T r; std::memcpy(&r, &raw, 4);
    return r;
}
template <typename T> inline T __shfl_sync(unsigned mask, T v, int src) { return emu_shfl(mask, v, src & 31); }
template <typename T> inline T __shfl_up_sync(unsigned mask, T v, unsigned d) {
    const int l = emu::lane();
    return emu_shfl(mask, v, l - (int)d >= 0 ? l - (int)d : l);
}
template <typename T> inline T __shfl_down_sync(unsigned mask, T v, unsigned d) {
    const int l = emu::lane();
    return emu_shfl(mask, v, l + (int)d < 32 ? l + (int)d : l);
}
template <typename T> inline T __shfl_xor_sync(unsigned mask, T v, int x) { return emu_shfl(mask, v, emu::lane() ^ x); }

// the few run-time calls the launchers make
typedef void* cudaStream_t;
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorLaunchFailure = 719 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
template <typename K> inline cudaError_t cudaFuncSetAttribute(K, cudaFuncAttribute, int) { return cudaSuccess; }
inline cudaError_t cudaGetLastError() { return emu::failed.load() ? cudaErrorLaunchFailure : cudaSuccess; }
inline const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : emu::err_msg; }
