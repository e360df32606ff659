// emu_selftest.cpp -- TEST ONLY.  Small scenarios that pin the emulation's own semantics (tests/test_emu_selftest_cpu.py):
// what an mbarrier wait by parity sees, transaction counts, over-arrival, TMA boxes (clipping, zero fill, SWIZZLE_32B),
// the tensor-memory lane-quarter rule, deadlock reporting.  Each scenario is a "kernel" of one block.
#define GSPN_EMU 1
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdio>
#include "emu_ptx.h"

namespace gspn {
static thread_local char g_err[2048] = "";
void set_error(const char* fmt, ...) { va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof(g_err), fmt, ap); va_end(ap); }
}
alignas(1024) static unsigned char smem[64 * 1024];
static int out[64];

template <typename F> static int run(unsigned threads, F f) {
    emu::wait_limit_s = 2.0;
    for (int& v : out) v = -1;
    return emu::launch(dim3(1), dim3(threads), smem, sizeof(smem), f) ? 0 : 1;
}
extern "C" const char* emu_err() { return emu::err_msg; }
extern "C" const int* emu_out() { return out; }

// 1: parity waits.  A fresh barrier is in phase 0: wait(1) returns at once, wait(0) blocks until count arrivals.
extern "C" int st_mbar_parity() {
    return run(64, [] {
        uint64_t* b = reinterpret_cast<uint64_t*>(smem);
        if (threadIdx.x == 0) gspn::mbar_init(b, 2);
        __syncthreads();
        gspn::mbar_wait(b, 1);                                   // the phase "before the first" counts as complete
        if (threadIdx.x == 0) out[0] = 1;
        __syncthreads();                                         // (nobody may still be in that wait when phase 0 completes)
        if (threadIdx.x == 32 || threadIdx.x == 33) gspn::mbar_arrive(b);
        gspn::mbar_wait(b, 0);                                   // completes with the second arrival
        if (threadIdx.x == 0) out[1] = 1;
        gspn::mbar_wait(b, 0);                                   // still true: phase 1 is open, parity 0 stays complete
        __syncthreads();
        if (threadIdx.x == 0) { gspn::mbar_arrive(b); gspn::mbar_arrive(b); }
        gspn::mbar_wait(b, 1);
        if (threadIdx.x == 0) out[2] = 1;
    });
}
// 2: a phase with transaction bytes completes only when arrivals AND bytes are in
extern "C" int st_mbar_tx() {
    return run(32, [] {
        uint64_t* b = reinterpret_cast<uint64_t*>(smem);
        static float src[64];
        if (threadIdx.x == 0) gspn::mbar_init(b, 1);
        __syncthreads();                                         // as in the kernels: nobody touches a barrier before its init
        if (threadIdx.x == 0) {
            for (int i = 0; i < 64; ++i) src[i] = (float)i;
            gspn::mbar_arrive_expect_tx(b, 256);
            gspn::bulk_load_1d(smem + 1024, src, 128, b);
            out[0] = 0;                                          // half the bytes: not complete (checked by the waiter below)
            gspn::bulk_load_1d(smem + 1024 + 128, src + 32, 128, b);
        }
        gspn::mbar_wait(b, 0);
        if (threadIdx.x == 1) out[1] = (int)reinterpret_cast<float*>(smem + 1024)[63];
    });
}
// 3: one arrival too many in a phase is an error, not silence
extern "C" int st_mbar_overarrive() {
    return run(32, [] {
        uint64_t* b = reinterpret_cast<uint64_t*>(smem);
        if (threadIdx.x == 0) { gspn::mbar_init(b, 1); gspn::mbar_arrive_expect_tx(b, 16); gspn::mbar_arrive(b); }
    });
}
// 4: a wait nobody completes is reported with the barrier's state
extern "C" int st_deadlock() {
    return run(64, [] {
        uint64_t* b = reinterpret_cast<uint64_t*>(smem);
        if (threadIdx.x == 0) gspn::mbar_init(b, 2);
        __syncthreads();
        if (threadIdx.x == 0) gspn::mbar_arrive(b);
        gspn::mbar_wait(b, 0);
    });
}
// 5: TMA box over the edge of a [planes=2][H=5][W=8] fp32 tensor: rows 3..6 of plane 1 -> rows 5, 6 arrive as zeros;
//    the store of the same box writes rows 3, 4 only
extern "C" int st_tma_clip(float* tensor) {
    return run(32, [=] {
        uint64_t* b = reinterpret_cast<uint64_t*>(smem);
        static CUtensorMap m;
        if (threadIdx.x == 0) {
            const uint64_t dims[3] = {8, 5, 2}, strides[2] = {32, 160};
            const uint32_t box[3] = {8, 4, 1};
            out[0] = gspn::encode_tensor_map(&m, 4, tensor, 3, dims, strides, box) ? 1 : 0;
            gspn::mbar_init(b, 1);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            gspn::mbar_arrive_expect_tx(b, 8 * 4 * 4);
            gspn::tma_load_3d(smem + 1024, &m, 0, 3, 1, b);
        }
        gspn::mbar_wait(b, 0);
        float* s = reinterpret_cast<float*>(smem + 1024);
        if (threadIdx.x == 0) {
            out[1] = (int)s[0]; out[2] = (int)s[8 + 7]; out[3] = (int)s[16]; out[4] = (int)s[31];
            for (int i = 0; i < 32; ++i) s[i] = 1000.f + i;
            gspn::tma_store_3d(&m, s, 0, 3, 1);
            gspn::bulk_commit();
            gspn::bulk_wait_all<0>();
        }
    });
}
// 6: SWIZZLE_32B: a box of 16 bf16 (32 bytes) x 16 rows lands with the 16-byte halves of rows 4..7, 12..15 exchanged
extern "C" int st_tma_swizzle(unsigned short* tensor) {
    return run(32, [=] {
        uint64_t* b = reinterpret_cast<uint64_t*>(smem);
        static CUtensorMap m;
        if (threadIdx.x == 0) {
            const uint64_t dims[3] = {16, 16, 1}, strides[2] = {32, 512};
            const uint32_t box[3] = {16, 16, 1};
            out[0] = gspn::encode_tensor_map(&m, 2, tensor, 3, dims, strides, box, 1) ? 1 : 0;
            gspn::mbar_init(b, 1);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            gspn::mbar_arrive_expect_tx(b, 512);
            gspn::tma_load_3d(smem + 1024, &m, 0, 0, 0, b);
        }
        gspn::mbar_wait(b, 0);
        const unsigned short* s = reinterpret_cast<const unsigned short*>(smem + 1024);
        if (threadIdx.x < 16) out[1 + threadIdx.x] = s[threadIdx.x * 16];        // first element of the physical row
    });
}
// 7: tensor memory: own lane quarter works, a foreign one is an error; columns beyond the allocation are an error
extern "C" int st_tmem(int mode) {
    return run(64, [=] {
        uint32_t* slot = reinterpret_cast<uint32_t*>(smem);
        if (threadIdx.x < 32) gspn::tm_alloc(slot, 32);
        __syncthreads();
        const uint32_t base = *slot, w = threadIdx.x >> 5;
        float f[4] = {1.f * threadIdx.x, 2.f, 3.f, 4.f}, g[4];
        const uint32_t quarter = mode == 1 ? (w ^ 1u) : w, col = mode == 2 ? 30u : 8u;
        gspn::tm_st<4>(base + ((32u * quarter) << 16) + col, f);
        gspn::tm_ld<4>(base + ((32u * quarter) << 16) + col, g);
        if (threadIdx.x == 37) out[0] = (int)g[0];
        __syncthreads();
        if (threadIdx.x < 32) gspn::tm_dealloc(base, 32);
    });
}
