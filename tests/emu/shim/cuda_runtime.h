// Shim of <cuda_runtime.h> for tests/emu: just enough of the CUDA C++ device vocabulary to compile the device code of
// csrc/gspn_naive.cuh with g++ and run one thread block as host threads (see tests/emu/naive_emu.cpp).  TEST ONLY.
#pragma once
#include <barrier>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstring>

#define __device__
#define __host__
#define __global__
#define __forceinline__ inline
#define __shared__
#define __restrict__
#define __launch_bounds__(...)

struct uint3 { unsigned x, y, z; };
struct dim3 { unsigned x = 1, y = 1, z = 1; };
typedef void* cudaStream_t;

namespace emu {
extern thread_local uint3 tid;          // threadIdx of the calling host thread
extern uint3 bid;                       // blockIdx of the block being run (one block at a time)
extern dim3 bdim, gdim;
extern std::barrier<>* block_barrier;   // __syncthreads of the running block
}  // namespace emu
#define threadIdx (emu::tid)
#define blockIdx (emu::bid)
#define blockDim (emu::bdim)
#define gridDim (emu::gdim)

inline void __syncthreads() { emu::block_barrier->arrive_and_wait(); }
template <typename T> inline T __ldg(const T* p) { return *p; }
inline float __uint_as_float(uint32_t v) { float f; std::memcpy(&f, &v, 4); return f; }
inline uint32_t __float_as_uint(float f) { uint32_t v; std::memcpy(&v, &f, 4); return v; }
using std::fmaf;
