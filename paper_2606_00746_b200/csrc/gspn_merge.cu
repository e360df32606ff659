// gspn_merge.cu -- merge of per-direction outputs (Eq. 9):
//   y[b,c,:,:] = sum_q m[q,c] * y_dirs[q,b,c,:,:]   (m NULL = ones), fp32 sum, one RNE.
// Pure streaming op: D reads + 1 write per element, 16-byte vector accesses on the aligned
// body of each (b,c) plane group, scalar accesses on ragged tails.
#include "gspn_kernels.h"
#include "../../include/gspn.h"

namespace gspn {

template <typename ST> struct Vec16;
template <> struct Vec16<float> { static constexpr int N = 4; };
template <> struct Vec16<__nv_bfloat16> { static constexpr int N = 8; };

__device__ __forceinline__ void unpack16(const uint4& v, float (&f)[4], const float*) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y);
    f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
}
__device__ __forceinline__ void unpack16(const uint4& v, float (&f)[8], const __nv_bfloat16*) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        f[2 * t] = __uint_as_float(w[t] << 16);
        f[2 * t + 1] = __uint_as_float(w[t] & 0xffff0000u);
    }
}
__device__ __forceinline__ uint4 pack16(const float (&f)[4], const float*) {
    return make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]),
                      __float_as_uint(f[3]));
}
__device__ __forceinline__ uint4 pack16(const float (&f)[8], const __nv_bfloat16*) {
    uint32_t w[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * t], f[2 * t + 1]);
        w[t] = *reinterpret_cast<uint32_t*>(&h);
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}

// One thread per 16-byte vector of the flat [B*C*H*W] output; the channel of a vector's first
// element selects m (a vector never straddles planes when plane % N == 0; otherwise the scalar
// kernel is used).
template <typename ST>
__global__ void merge_vec_kernel(const ST* __restrict__ yd, const float* __restrict__ m,
                                 ST* __restrict__ y, int D, int C, size_t plane, size_t n) {
    constexpr int N = Vec16<ST>::N;
    const size_t nv = n / N;
    for (size_t v = blockIdx.x * (size_t)blockDim.x + threadIdx.x; v < nv;
         v += (size_t)gridDim.x * blockDim.x) {
        const size_t e = v * N;
        const int c = (int)((e / plane) % C);
        float acc[N];
#pragma unroll
        for (int t = 0; t < N; ++t) acc[t] = 0.f;
        for (int q = 0; q < D; ++q) {
            const uint4 raw = __ldg(reinterpret_cast<const uint4*>(yd + q * n + e));
            float f[N];
            unpack16(raw, f, (const ST*)nullptr);
            const float mq = m ? __ldg(m + q * C + c) : 1.f;
#pragma unroll
            for (int t = 0; t < N; ++t) acc[t] = fmaf(mq, f[t], acc[t]);
        }
        *reinterpret_cast<uint4*>(y + e) = pack16(acc, (const ST*)nullptr);
    }
}

template <typename ST>
__global__ void merge_scalar_kernel(const ST* __restrict__ yd, const float* __restrict__ m,
                                    ST* __restrict__ y, int D, int C, size_t plane, size_t n) {
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n;
         e += (size_t)gridDim.x * blockDim.x) {
        const int c = (int)((e / plane) % C);
        float acc = 0.f;
        for (int q = 0; q < D; ++q)
            acc = fmaf(m ? __ldg(m + q * C + c) : 1.f, ld_f(yd + q * n + e), acc);
        st_f(y + e, acc);
    }
}

template <typename ST>
int merge_launch(const ST* y_dirs, const float* m, ST* y, int D, int B, int C, int H, int W,
                 cudaStream_t st, LaunchInfo* li) {
    const size_t plane = (size_t)H * W, n = (size_t)B * C * plane;
    constexpr int N = Vec16<ST>::N;
    const int threads = 256;
    // slab q starts at q*n elements: 16-byte aligned iff n % N == 0
    const bool vec = (plane % N == 0);
    const size_t work = vec ? n / N : n;
    size_t blocks = (work + threads - 1) / threads;
    const size_t cap = 148 * 16;                      // a few waves of the 148 SMs, grid-stride beyond
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    if (vec) merge_vec_kernel<ST><<<(unsigned)blocks, threads, 0, st>>>(y_dirs, m, y, D, C, plane, n);
    else     merge_scalar_kernel<ST><<<(unsigned)blocks, threads, 0, st>>>(y_dirs, m, y, D, C, plane, n);
    li->launches = 1;
    li->variant = vec ? "merge_vec16" : "merge_scalar";
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("merge: launch failed: %s", cudaGetErrorString(e));
        return GSPN_ECUDA;
    }
    return GSPN_OK;
}

template int merge_launch<float>(const float*, const float*, float*, int, int, int, int, int,
                                 cudaStream_t, LaunchInfo*);
template int merge_launch<__nv_bfloat16>(const __nv_bfloat16*, const float*, __nv_bfloat16*, int, int,
                                         int, int, int, cudaStream_t, LaunchInfo*);

}  // namespace gspn
