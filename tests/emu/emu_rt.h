// emu_rt.h -- TEST ONLY.  The run time of the host emulation under tests/emu: one CUDA thread block at a time, its threads
// as host threads, with the synchronisation objects the kernels use (block / warp / named barriers, warp shuffles,
// mbarriers with transaction counts) and two on-chip memories (dynamic shared memory is a plain array defined beside
// the kernel; tensor memory lives here).  Every blocking wait has a time limit and polls a failure flag, so a protocol
// error (a barrier nobody completes, an mbarrier over-arrival, an access outside an allocation) ends the launch with a
// message instead of hanging or faulting the test process.  Nothing under paper_2606_00746_b200/ includes this.
#pragma once

#include <atomic>
#include <chrono>
#include <condition_variable>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <functional>
#include <memory>
#include <mutex>
#include <thread>
#include <unordered_map>
#include <vector>

struct uint3 { unsigned x, y, z; };
struct dim3 {
    unsigned x = 1, y = 1, z = 1;
    dim3() = default;
    dim3(unsigned a, unsigned b = 1, unsigned c = 1) : x(a), y(b), z(c) {}
};

namespace emu {

struct Error {};                                   // thrown inside a kernel thread once the launch has failed
inline std::atomic<bool> failed{false};
inline std::mutex err_m;
inline char err_msg[2048] = "";
inline double wait_limit_s = 30.0;                 // a wait longer than this is reported as a deadlock

[[noreturn]] inline void fail(const char* fmt, ...) {
    {
        std::lock_guard<std::mutex> l(err_m);
        if (!failed.load()) {
            va_list ap;
            va_start(ap, fmt);
            vsnprintf(err_msg, sizeof(err_msg), fmt, ap);
            va_end(ap);
            failed.store(true);
        }
    }
    throw Error{};
}
inline void check_failed() { if (failed.load(std::memory_order_relaxed)) throw Error{}; }
using Clock = std::chrono::steady_clock;
inline Clock::time_point deadline() { return Clock::now() + std::chrono::milliseconds((long long)(wait_limit_s * 1e3)); }

// a counting barrier whose participants may leave (a thread that returns from the kernel counts as arrived for good)
struct Bar {
    std::mutex m;
    std::condition_variable cv;
    int expected = 0, waiting = 0;
    uint64_t gen = 0;
    void reset(int n) { expected = n; waiting = 0; gen = 0; }
    void wait(const char* what, int id = -1) {
        std::unique_lock<std::mutex> l(m);
        const uint64_t g = gen;
        if (++waiting >= expected) { waiting = 0; ++gen; cv.notify_all(); return; }
        const auto dl = deadline();
        while (gen == g) {
            cv.wait_for(l, std::chrono::milliseconds(20));
            if (gen != g) break;
            if (failed.load()) throw Error{};
            if (Clock::now() > dl) {
                const int w = waiting, e = expected;
                l.unlock();
                fail("deadlock at %s %d: %d of %d threads arrived", what, id, w, e);
            }
        }
    }
    void drop() {
        std::lock_guard<std::mutex> l(m);
        --expected;
        if (expected > 0 && waiting >= expected) { waiting = 0; ++gen; cv.notify_all(); }
    }
};

struct Warp {
    Bar bar;
    uint32_t xch[32];
};

// mbarrier (PTX mbarrier.*): pending arrivals and a signed transaction count; a phase completes when both are zero
struct MBar { int expected = 0, pending = 0; long long tx = 0; unsigned phase = 0; };

struct Block {
    // lazy mode: TMA loads that have been issued but not yet performed, per mbarrier (performed when a thread waits on it)
    std::unordered_map<const void*, std::vector<std::function<long long()>>> lazy_loads;
    Bar bar;                                        // __syncthreads
    std::vector<std::unique_ptr<Warp>> warps;
    Bar named[16];                                  // bar.sync id, n
    std::mutex mb_m;
    std::unordered_map<const void*, MBar> mbars;
    uint32_t tm_cols = 0;                           // tensor-memory columns allocated by this CTA (0 = none)
};
inline Block* blk = nullptr;
inline thread_local uint3 tid;
inline thread_local Warp* my_warp = nullptr;
inline uint3 bid;
inline dim3 bdim, gdim;
inline const unsigned char* smem_lo = nullptr;      // bounds of the running kernel's shared memory (set by the launch)
inline const unsigned char* smem_hi = nullptr;
inline uint32_t tmem[128][512];                     // tensor memory of the SM: 128 lanes x 512 columns x 32 bit

// Optional timing noise: with jitter_us > 0 a thread sleeps for a random 0..jitter_us microseconds at one in four of its
// synchronisation operations, so that repeated runs walk through different interleavings of producers and consumers.
inline int jitter_us = 0;
inline unsigned jitter_seed = 1;
inline void jitter() {
    if (jitter_us <= 0) return;
    static thread_local uint32_t s = 0;
    if (s == 0) s = (jitter_seed * 2654435761u) ^ ((tid.x + 1u) * 40503u) ^ ((bid.x + 1u) * 69069u) | 1u;
    s ^= s << 13; s ^= s >> 17; s ^= s << 5;
    if ((s & 3u) == 0) std::this_thread::sleep_for(std::chrono::microseconds((s >> 8) % (unsigned)jitter_us));
}

// Lazy mode: asynchronous copies happen as LATE as the program allows instead of at once.  A TMA load lands only when a
// thread waits on its mbarrier (a consumer that reads without waiting finds the poison the stage was filled with); a TMA
// store reads shared memory only when its thread executes cp.async.bulk.wait_group[.read] for its group (a stage that is
// overwritten before that wait sends the new bytes, and the comparison with the oracle fails).  Eager mode (the default)
// is the other extreme: a refill destroys a stage that is still being read at once.
inline bool lazy = false;
inline thread_local std::vector<std::vector<std::function<void()>>> store_groups;      // closed groups, oldest first
inline thread_local std::vector<std::function<void()>> store_open;                      // stores since the last commit
inline void stores_commit() { if (lazy) { store_groups.push_back(std::move(store_open)); store_open.clear(); } }
inline void stores_wait(int keep_newest) {
    while ((int)store_groups.size() > keep_newest) {
        for (auto& f : store_groups.front()) f();
        store_groups.erase(store_groups.begin());
    }
}

inline int lane() { return (int)(tid.x & 31u); }
inline int warp() { return (int)(tid.x >> 5); }

inline void sync_block() { jitter(); blk->bar.wait("__syncthreads"); }
inline void sync_warp() { my_warp->bar.wait("__syncwarp of warp", warp()); }
inline uint32_t shfl_raw(uint32_t v, int src) {
    Warp& w = *my_warp;
    w.xch[lane()] = v;
    w.bar.wait("shuffle (publish) of warp", warp());
    const uint32_t r = w.xch[src & 31];
    w.bar.wait("shuffle (read) of warp", warp());
    return r;
}
inline void named_sync(int id, int nthreads) {
    if (id < 1 || id > 15) fail("bar.sync: id %d outside 1..15", id);
    if (nthreads % 32 || nthreads < 32) fail("bar.sync %d: thread count %d is not a multiple of the warp size", id, nthreads);
    Bar& b = blk->named[id];
    int other = 0;
    {
        std::lock_guard<std::mutex> l(b.m);
        if (b.waiting == 0) b.expected = nthreads;
        else if (b.expected != nthreads) other = b.expected;
    }
    if (other) fail("bar.sync %d: called with %d threads while a round with %d threads is open", id, nthreads, other);
    jitter();
    b.wait("bar.sync", id);
}

// ---- mbarrier --------------------------------------------------------------------------------------------------------
inline long smem_off(const void* p) { return (long)((const unsigned char*)p - smem_lo); }
inline void check_smem(const void* p, size_t bytes, const char* what) {
    const unsigned char* q = (const unsigned char*)p;
    if (q < smem_lo || q + bytes > smem_hi) fail("%s: [%ld, %ld) lies outside the CTA's %ld bytes of shared memory", what, smem_off(p), smem_off(p) + (long)bytes, (long)(smem_hi - smem_lo));
}
inline MBar& mb_get(const void* b, const char* what) {
    auto it = blk->mbars.find(b);
    if (it == blk->mbars.end()) fail("%s: mbarrier at shared offset %ld was never initialised", what, smem_off(b));
    return it->second;
}
inline void mb_complete_if_done(MBar& m) {
    if (m.pending == 0 && m.tx == 0) { m.phase ^= 1u; m.pending = m.expected; }
}
inline void mb_init(const void* b, uint32_t count) {
    check_smem(b, 8, "mbarrier.init");
    if ((uintptr_t)b & 7u) fail("mbarrier.init: shared offset %ld is not 8-byte aligned", smem_off(b));
    std::lock_guard<std::mutex> l(blk->mb_m);
    MBar m; m.expected = (int)count; m.pending = (int)count;
    blk->mbars[b] = m;
}
inline void mb_arrive(const void* b, long long expect_tx) {
    jitter();
    std::unique_lock<std::mutex> l(blk->mb_m);
    MBar& m = mb_get(b, "mbarrier.arrive");
    m.tx += expect_tx;
    if (m.pending <= 0) { l.unlock(); fail("mbarrier at shared offset %ld: more arrivals than its count %d in one phase", smem_off(b), m.expected); }
    --m.pending;
    mb_complete_if_done(m);
}
inline void mb_complete_tx(const void* b, long long bytes) {
    jitter();
    std::lock_guard<std::mutex> l(blk->mb_m);
    MBar& m = mb_get(b, "complete_tx");
    m.tx -= bytes;
    mb_complete_if_done(m);
}
inline void mb_wait(const void* b, uint32_t parity) {
    jitter();
    const auto dl = deadline();
    for (unsigned spin = 0;; ++spin) {
        if (lazy) {      // the copies that complete on this barrier land now, when somebody is waiting for them
            std::vector<std::function<long long()>> todo;
            {
                std::lock_guard<std::mutex> l(blk->mb_m);
                auto it = blk->lazy_loads.find(b);
                if (it != blk->lazy_loads.end()) todo.swap(it->second);
            }
            for (auto& f : todo) {
                const long long bytes = f();
                std::lock_guard<std::mutex> l(blk->mb_m);
                MBar& m = mb_get(b, "complete_tx");
                m.tx -= bytes;
                mb_complete_if_done(m);
            }
        }
        {
            std::unique_lock<std::mutex> l(blk->mb_m);
            MBar& m = mb_get(b, "mbarrier.try_wait");
            if ((m.phase & 1u) != (parity & 1u)) return;
            if ((spin & 255u) == 255u && Clock::now() > dl) {
                const MBar c = m;
                l.unlock();
                fail("deadlock: thread %u (warp %d) waits on the mbarrier at shared offset %ld for parity %u; phase %u, %d of %d arrivals "
                     "pending, %lld transaction bytes outstanding", tid.x, warp(), smem_off(b), parity, c.phase, c.pending, c.expected, c.tx);
            }
        }
        check_failed();
        if (spin < 64) std::this_thread::yield(); else std::this_thread::sleep_for(std::chrono::microseconds(50));
    }
}

// ---- launch ------------------------------------------------------------------------------------------------------------
// runs `body` once per thread of every block, block after block; returns false (message in err_msg) when a block failed
template <typename F>
bool launch(dim3 grid, dim3 block, unsigned char* smem, size_t smem_bytes, F body) {
    failed.store(false);
    err_msg[0] = 0;
    gdim = grid; bdim = block;
    const unsigned nthr = block.x, nwarp = (nthr + 31) / 32;
    if (nthr % 32) { snprintf(err_msg, sizeof(err_msg), "block of %u threads is not whole warps", nthr); failed.store(true); return false; }
    for (unsigned b = 0; b < grid.x && !failed.load(); ++b) {
        Block state;
        state.bar.reset((int)nthr);
        for (unsigned w = 0; w < nwarp; ++w) { state.warps.emplace_back(new Warp); state.warps.back()->bar.reset(32); }
        blk = &state;
        bid = uint3{b, 0, 0};
        smem_lo = smem; smem_hi = smem + smem_bytes;
        memset(smem, 0xc1, smem_bytes);              // what a CTA finds in shared memory is not zero
        for (auto& row : tmem) for (auto& v : row) v = 0x7fc00123u;      // nor in tensor memory: NaN
        std::vector<std::thread> pool;
        for (unsigned t = 0; t < nthr; ++t)
            pool.emplace_back([&, t] {
                tid = uint3{t, 0, 0};
                my_warp = state.warps[t >> 5].get();
                store_groups.clear(); store_open.clear();
                try {
                    body();
                    if (!store_open.empty() || !store_groups.empty())
                        fail("thread %u returns with bulk stores it never waited for (cp.async.bulk.wait_group)", t);
                } catch (const Error&) {}
                my_warp->bar.drop();
                state.bar.drop();
            });
        for (auto& th : pool) th.join();
        if (!failed.load() && state.tm_cols) {
            snprintf(err_msg, sizeof(err_msg), "block %u exited without tcgen05.dealloc of its %u tensor-memory columns", b, state.tm_cols);
            failed.store(true);
        }
        blk = nullptr;
    }
    return !failed.load();
}

}  // namespace emu
