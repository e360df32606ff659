// emu_ptx.h -- TEST ONLY.  Host stand-ins, under the same names, for the PTX wrappers of csrc/gspn_fused.cuh and
// csrc/gspn_line.cuh (mbarrier, TMA tensor / bulk copies, tensor memory, named barriers, the bf16 FMA).  Those headers
// include this file instead of their inline assembly when GSPN_EMU is defined, which only tests/emu does.  Each stand-in
// also checks what the hardware would fault on or silently get wrong: alignment of TMA destinations, boxes against the
// tensor-map rules, tensor-memory accesses against the allocation and the warp's lane quarter, shared-memory bounds.
// Copies complete at once (the fastest TMA there could be): a consumer that reads before waiting still sees its data, but
// a producer that overwrites a stage too early destroys it at once, which is the direction that bites.
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

namespace gspn {

inline uint32_t smem_u32(const void* p) { return (uint32_t)emu::smem_off(p); }
inline void mbar_init(uint64_t* b, uint32_t count) { emu::mb_init(b, count); }
inline void mbar_init_fence() {}
inline void mbar_arrive(uint64_t* b) { emu::mb_arrive(b, 0); }
inline void mbar_arrive_expect_tx(uint64_t* b, uint32_t bytes) { emu::mb_arrive(b, bytes); }
inline void mbar_wait(uint64_t* b, uint32_t parity) { emu::mb_wait(b, parity); }
inline void mbar_wait_spin(uint64_t* b, uint32_t parity) { emu::mb_wait(b, parity); }
inline void named_bar_sync(int id, int nthreads) { emu::named_sync(id, nthreads); }
inline void fence_proxy_async() {}
inline void bulk_commit() { emu::stores_commit(); }
template <int N> inline void bulk_wait_read() { emu::stores_wait(N); }
template <int N> inline void bulk_wait_all() { emu::stores_wait(N); }

// ---- tensor maps ---------------------------------------------------------------------------------------------------------
struct EmuMap {
    uint64_t magic;
    unsigned char* base;
    uint32_t es, rank, swizzle32;
    uint64_t strides[5];               // in bytes, strides[0] = es
    uint32_t dims[5], box[5];
};
static_assert(sizeof(EmuMap) <= sizeof(CUtensorMap), "EmuMap must fit the opaque tensor map");
constexpr uint64_t kEmuMapMagic = 0x454d554d41503031ull;

void set_error(const char* fmt, ...);

// same contract as the library's encoder (csrc/gspn_tmap.cu) plus the driver's argument rules
inline bool encode_tensor_map(CUtensorMap* out, int es, void* base, int rank, const uint64_t* dims, const uint64_t* strides_bytes,
                              const uint32_t* box, int swizzle32 = 0) {
    auto bad = [&](const char* why) { set_error("encode_tensor_map (emulated driver rules): %s", why); return false; };
    if (rank < 3 || rank > 5) return bad("rank outside 3..5");
    if ((uintptr_t)base & 15u) return bad("global address not 16-byte aligned");
    if (es != 2 && es != 4) return bad("element size");
    EmuMap m{};
    m.magic = kEmuMapMagic; m.base = (unsigned char*)base; m.es = (uint32_t)es; m.rank = (uint32_t)rank; m.swizzle32 = swizzle32 ? 1u : 0u;
    for (int i = 0; i < rank; ++i) {
        if (dims[i] == 0 || dims[i] >= (1ull << 32)) return bad("dimension of size 0 or of 2^32 and more");
        if (box[i] == 0 || box[i] > 256) return bad("box dimension outside 1..256");
        m.dims[i] = (uint32_t)dims[i]; m.box[i] = box[i];
        m.strides[i] = i == 0 ? (uint64_t)es : strides_bytes[i - 1];
        if (i > 0 && (m.strides[i] & 15u)) return bad("stride not a multiple of 16 bytes");
    }
    if (((uint64_t)box[0] * es) & 15u) return bad("inner box extent not a multiple of 16 bytes");
    if (swizzle32 && (uint64_t)box[0] * es > 32) return bad("SWIZZLE_32B with an inner box extent above 32 bytes");
    std::memset(out, 0, sizeof(*out));
    std::memcpy(out, &m, sizeof(m));
    return true;
}

inline const EmuMap& emu_map(const CUtensorMap* m) {
    const EmuMap* e = reinterpret_cast<const EmuMap*>(m);
    if (e->magic != kEmuMapMagic) emu::fail("TMA: the tensor map was not encoded");
    return *e;
}

// the box at `coord` <-> shared memory at `smem`; LOAD: out-of-range elements arrive as zeros; STORE: they are not written
template <bool LOAD>
inline uint64_t emu_tma(const CUtensorMap* map, unsigned char* smem, const int* coord, int rank_given) {
    const EmuMap& m = emu_map(map);
    if ((int)m.rank != rank_given) emu::fail("TMA: %d coordinates for a tensor map of rank %u", rank_given, m.rank);
    uint64_t elems = 1;
    for (uint32_t i = 0; i < m.rank; ++i) elems *= m.box[i];
    const uint64_t bytes = elems * m.es;
    if ((uintptr_t)smem & 127u) emu::fail("TMA %s: shared address (offset %ld) is not 128-byte aligned", LOAD ? "load" : "store", emu::smem_off(smem));
    emu::check_smem(smem, bytes, LOAD ? "TMA load" : "TMA store");
    uint32_t idx[5] = {0, 0, 0, 0, 0};
    for (uint64_t e = 0; e < elems; ++e) {
        bool inside = true;
        uint64_t goff = 0;
        for (uint32_t i = 0; i < m.rank; ++i) {
            const long long c = (long long)coord[i] + idx[i];
            if (c < 0 || c >= (long long)m.dims[i]) { inside = false; break; }
            goff += (uint64_t)c * m.strides[i];
        }
        uintptr_t sa = (uintptr_t)smem + e * m.es;
        if (m.swizzle32) sa ^= ((sa >> 7) & 1u) << 4;        // SWIZZLE_32B: the 16-byte half of a 32-byte row flips with address bit 7
        unsigned char* sp = reinterpret_cast<unsigned char*>(sa);
        if (LOAD) {
            if (inside) std::memcpy(sp, m.base + goff, m.es); else std::memset(sp, 0, m.es);
        } else if (inside) {
            std::memcpy(m.base + goff, sp, m.es);
        }
        for (uint32_t i = 0; i < m.rank; ++i) { if (++idx[i] < m.box[i]) break; idx[i] = 0; }
    }
    return bytes;
}
// a load: at once (eager) or when a thread waits on `bar` (lazy, emu_rt.h)
template <typename F> inline void emu_issue_load(uint64_t* bar, F copy) {
    if (!emu::lazy) { emu::mb_complete_tx(bar, copy()); return; }
    std::lock_guard<std::mutex> l(emu::blk->mb_m);
    (void)emu::mb_get(bar, "TMA load");
    emu::blk->lazy_loads[bar].emplace_back(copy);
}
template <int R> inline void emu_load(void* dst, const CUtensorMap* m, const int (&c)[R], uint64_t* bar) {
    const CUtensorMap mc = *m;
    int cc[5] = {0, 0, 0, 0, 0};
    for (int i = 0; i < R; ++i) cc[i] = c[i];
    struct Job { CUtensorMap m; unsigned char* dst; int c[5]; };
    const Job j{mc, (unsigned char*)dst, {cc[0], cc[1], cc[2], cc[3], cc[4]}};
    emu_issue_load(bar, [j]() -> long long { return (long long)emu_tma<true>(&j.m, j.dst, j.c, R); });
}
template <int R> inline void emu_store(const CUtensorMap* m, const void* src, const int (&c)[R]) {
    if (!emu::lazy) { emu_tma<false>(m, (unsigned char*)src, c, R); return; }
    struct Job { CUtensorMap m; unsigned char* src; int c[5]; };
    Job j{*m, (unsigned char*)src, {0, 0, 0, 0, 0}};
    for (int i = 0; i < R; ++i) j.c[i] = c[i];
    emu::store_open.emplace_back([j] { emu_tma<false>(&j.m, j.src, j.c, R); });
}
inline void tma_load_3d(void* dst, const CUtensorMap* m, int c0, int c1, int c2, uint64_t* bar) { emu_load<3>(dst, m, {c0, c1, c2}, bar); }
inline void tma_load_4d(void* dst, const CUtensorMap* m, int c0, int c1, int c2, int c3, uint64_t* bar) { emu_load<4>(dst, m, {c0, c1, c2, c3}, bar); }
inline void tma_load_5d(void* dst, const CUtensorMap* m, int c0, int c1, int c2, int c3, int c4, uint64_t* bar) { emu_load<5>(dst, m, {c0, c1, c2, c3, c4}, bar); }
inline void tma_store_3d(const CUtensorMap* m, const void* src, int c0, int c1, int c2) { emu_store<3>(m, src, {c0, c1, c2}); }
inline void tma_store_4d(const CUtensorMap* m, const void* src, int c0, int c1, int c2, int c3) { emu_store<4>(m, src, {c0, c1, c2, c3}); }
inline void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    if (((uintptr_t)dst & 15u) || ((uintptr_t)src & 15u) || (bytes & 15u))
        emu::fail("cp.async.bulk: destination (shared offset %ld), source or size %u not 16-byte aligned", emu::smem_off(dst), bytes);
    emu::check_smem(dst, bytes, "cp.async.bulk");
    emu_issue_load(bar, [=]() -> long long { std::memcpy(dst, src, bytes); return (long long)bytes; });
}
inline void bulk_store_1d(void* dst, const void* src, uint32_t bytes) {
    if (((uintptr_t)dst & 15u) || ((uintptr_t)src & 15u) || (bytes & 15u))
        emu::fail("cp.async.bulk (store): source (shared offset %ld), destination or size %u not 16-byte aligned", emu::smem_off(src), bytes);
    emu::check_smem(src, bytes, "cp.async.bulk (store)");
    if (!emu::lazy) { std::memcpy(dst, src, bytes); return; }
    emu::store_open.emplace_back([=] { std::memcpy(dst, src, bytes); });
}
inline void tma_prefetch_desc(const CUtensorMap* m) { (void)emu_map(m); }

// ---- tensor memory: shape 32x32b, thread t of a warp reaches lane 32 * (warp % 4) + t only ------------------------------------
inline void tm_alloc(uint32_t* slot, uint32_t cols) {
    if (cols < 32 || cols > 512 || (cols & (cols - 1))) emu::fail("tcgen05.alloc: %u columns is not a power of two in 32..512", cols);
    emu::sync_warp();                                       // .sync.aligned: the whole warp executes it
    if (emu::lane() == 0) {
        if (emu::blk->tm_cols) emu::fail("tcgen05.alloc: the CTA already holds %u columns", emu::blk->tm_cols);
        emu::check_smem(slot, 4, "tcgen05.alloc result slot");
        emu::blk->tm_cols = cols;
        *slot = 0;                                          // base: lane 0, column 0
    }
    emu::sync_warp();
}
inline void tm_dealloc(uint32_t base, uint32_t cols) {
    emu::sync_warp();
    if (emu::lane() == 0) {
        if (base != 0 || cols != emu::blk->tm_cols) emu::fail("tcgen05.dealloc: base %u / %u columns, allocated %u", base, cols, emu::blk->tm_cols);
        emu::blk->tm_cols = 0;
    }
    emu::sync_warp();
}
inline uint32_t* emu_tm_row(uint32_t ta, int n, const char* what) {
    const uint32_t lane_base = ta >> 16, col = ta & 0xffffu;
    if (lane_base != 32u * ((uint32_t)emu::warp() & 3u))
        emu::fail("%s: warp %d addresses lanes %u.. but reaches only its own quarter %u..", what, emu::warp(), lane_base, 32u * ((uint32_t)emu::warp() & 3u));
    if (col + (uint32_t)n > emu::blk->tm_cols)
        emu::fail("%s: columns [%u, %u) beyond the %u allocated (warp %d, lane %d)", what, col, col + n, emu::blk->tm_cols, emu::warp(), emu::lane());
    return &emu::tmem[lane_base + (uint32_t)emu::lane()][col];
}
template <int N> inline void tm_ld(uint32_t ta, float (&f)[N]) {
    const uint32_t* r = emu_tm_row(ta, N, "tcgen05.ld");
    for (int i = 0; i < N; ++i) f[i] = __uint_as_float(r[i]);
}
template <int N> inline void tm_st(uint32_t ta, const float (&f)[N]) {
    uint32_t* r = emu_tm_row(ta, N, "tcgen05.st");
    for (int i = 0; i < N; ++i) r[i] = __float_as_uint(f[i]);
}
template <int N> inline void tm_wait_ld(float (&)[N]) {}
inline void tm_wait_st() {}
inline void tm_fence_before() {}
inline void tm_fence_after() {}

// ---- csrc/gspn_flat.cuh / gspn_chain.cuh: shared memory addressed by 32-bit shared-window addresses, cp.async ----------------
// smem_u32() above hands out offsets from the start of the CTA's shared memory; these turn them back into pointers.
template <typename T> inline T* emu_sptr(uint32_t a, const char* what) {
    unsigned char* p = const_cast<unsigned char*>(emu::smem_lo) + a;
    emu::check_smem(p, sizeof(T), what);
    if ((uintptr_t)p % sizeof(T)) emu::fail("%s: shared address %u is not %zu-byte aligned", what, a, sizeof(T));
    return reinterpret_cast<T*>(p);
}
inline float lds_f32(uint32_t a) { return *emu_sptr<float>(a, "ld.shared.f32"); }
inline void sts_f32(uint32_t a, float v) { *emu_sptr<float>(a, "st.shared.f32") = v; }
inline float lds32(uint32_t a) { return lds_f32(a); }
inline void sts32(uint32_t a, float v) { sts_f32(a, v); }
template <typename ST> inline float lds_f(uint32_t a);
template <> inline float lds_f<float>(uint32_t a) { return lds_f32(a); }
template <> inline float lds_f<__nv_bfloat16>(uint32_t a) { return __uint_as_float(((uint32_t)*emu_sptr<unsigned short>(a, "ld.shared.u16")) << 16); }
// cp.async: the copy happens at once; cp.async.mbarrier.arrive.noinc is then a plain arrival (the count was pre-armed)
inline void emu_cp_async(void* dst, const void* src, int bytes) {
    if (((uintptr_t)dst | (uintptr_t)src) % bytes) emu::fail("cp.async: %d-byte copy with an unaligned address (shared offset %ld)", bytes, emu::smem_off(dst));
    emu::check_smem(dst, bytes, "cp.async");
    std::memcpy(dst, src, bytes);
}
inline void cp_async_16(void* dst, const void* src) { emu_cp_async(dst, src, 16); }
inline void cp_async_arrive_noinc(uint64_t* bar) { emu::mb_arrive(bar, 0); }
template <int CB> inline void cp_async_cb(uint32_t dst, const void* src) {
    static_assert(CB == 8 || CB == 16, "cp_async_cb");
    emu_cp_async(const_cast<unsigned char*>(emu::smem_lo) + dst, src, CB);
}
inline void l2_prefetch_bulk(const void* p, uint32_t bytes) {
    if (((uintptr_t)p & 15u) || (bytes & 15u) || bytes == 0) emu::fail("cp.async.bulk.prefetch.L2: address or size %u not a multiple of 16", bytes);
}
template <typename ST> struct Elem;
template <> struct Elem<__nv_bfloat16> {
    using raw_t = unsigned short;
    static raw_t lds(uint32_t a) { return *emu_sptr<raw_t>(a, "ld.shared.u16"); }
    static void sts(uint32_t a, raw_t v) { *emu_sptr<raw_t>(a, "st.shared.u16") = v; }
    static float f(raw_t r) { return __uint_as_float(((uint32_t)r) << 16); }
    static float fma2(raw_t a, raw_t b, float c) { return fmaf(f(a), f(b), c); }
    static raw_t pack(float v) { return __bfloat16_as_ushort(__float2bfloat16_rn(v)); }
    static void stg(__nv_bfloat16* p, raw_t v) { *reinterpret_cast<raw_t*>(p) = v; }
};
template <> struct Elem<float> {
    using raw_t = float;
    static raw_t lds(uint32_t a) { return lds_f32(a); }
    static void sts(uint32_t a, raw_t v) { sts_f32(a, v); }
    static float f(raw_t r) { return r; }
    static float fma2(raw_t a, raw_t b, float c) { return fmaf(a, b, c); }
    static raw_t pack(float v) { return v; }
    static void stg(float* p, raw_t v) { *p = v; }
};

// fma.rn.f32.bf16: c + a * b with a, b the low or high bf16 half of a 32-bit word, one rounding
inline float fma_bf16_half(uint32_t a, uint32_t b, bool high, float c) {
    const float fa = __uint_as_float(high ? (a & 0xffff0000u) : (a << 16)), fb = __uint_as_float(high ? (b & 0xffff0000u) : (b << 16));
    return fmaf(fa, fb, c);
}

}  // namespace gspn
