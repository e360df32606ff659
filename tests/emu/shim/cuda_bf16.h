// Shim of <cuda_bf16.h> for tests/emu (TEST ONLY): storage type and round-to-nearest-even conversion.
#pragma once
#include <cstdint>
#include <cstring>
struct __nv_bfloat16 { unsigned short x; };
struct __nv_bfloat162 { __nv_bfloat16 x, y; };
inline __nv_bfloat16 __float2bfloat16_rn(float f) {
    uint32_t v; std::memcpy(&v, &f, 4);
    __nv_bfloat16 r;
    if ((v & 0x7fffffffu) > 0x7f800000u) { r.x = 0x7fff; return r; }      // NaN
    v += 0x7fffu + ((v >> 16) & 1u);                                      // round to nearest, ties to even
    r.x = (unsigned short)(v >> 16);
    return r;
}
inline unsigned short __bfloat16_as_ushort(__nv_bfloat16 v) { return v.x; }
inline __nv_bfloat162 __floats2bfloat162_rn(float a, float b) { return __nv_bfloat162{__float2bfloat16_rn(a), __float2bfloat16_rn(b)}; }
