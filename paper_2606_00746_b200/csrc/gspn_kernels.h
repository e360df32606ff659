// gspn_kernels.h -- host-side launchers of the libgspn kernels (internal to csrc/).
// Each launcher validates only what its kernel needs (shape already checked by the C ABI),
// enqueues on `st`, fills LaunchInfo and returns a GSPN_* status.
#pragma once

#include "gspn_common.cuh"

namespace gspn {

// naive kernels (gspn_naive.cu): one CTA per plane, one thread per cross position, operands read
// straight from global memory.  Reference GPU path for A/B runs; slow by design.
template <typename ST> int naive_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);
template <typename ST> int naive_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);
// bytes of caller workspace the naive kernels need for this shape (planes beyond shared memory), 0 if none
size_t naive_workspace_bytes(const Shape& sh, bool bwd);

// fused kernels: forward tile kernel (gspn_fused_fwd.cu), backward group kernel (gspn_group_bwd.cu).
template <typename ST> int fused_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);
template <typename ST> int fused_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);

// flat kernels (gspn_flat_fwd.cu / gspn_flat_bwd.cu): fused single-launch kernels for ANY H, W and
// storage type (rows / planes need not be 16-byte aligned).
template <typename ST> int flat_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);

// chain kernels (gspn_chain_bwd.cu / gspn_chain_fwd.cu): one warp per scan chain, no block barrier on the
// serial path, operands staged asynchronously by a producer warp; any H, W <= 128 and storage type.
template <typename ST> int chain_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);
template <typename ST> int chain_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);

// pair kernel (gspn_pair_fwd.cu): one warp carries all channels of a CTA for one direction (shared taps, NC*P
// independent recurrences per lane), the two opposite directions of an axis run at the same time and share Y.
// whole-plane variant of the same for small planes (max(H,W) <= 64 and two CTAs' planes per SM): no rings
template <typename ST> int plane_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);

// whole-plane backward for small planes (gspn_plane_bwd.cu): lines of at most one warp, C/G in {1, 2, 4}
template <typename ST> int plane_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);

// line kernels (gspn_line_fwd.cu / gspn_line_bwd.cu): 16-byte-aligned rows, warp per (channel, direction) line with 1, 2 or
// 4 positions per lane, NC channels of a unit per CTA sharing the taps, one fp32 accumulator plane per channel.
template <typename ST> int line_fwd_launch(const FwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);
template <typename ST> int line_bwd_launch(const BwdArgs<ST>& a, cudaStream_t st, LaunchInfo* li);

// merge (gspn_merge.cu)
template <typename ST>
int merge_launch(const ST* y_dirs, const float* m, ST* y, int D, int B, int C, int H, int W,
                 cudaStream_t st, LaunchInfo* li);

// Eq. 3 normalisation of the tap logits and its adjoint (gspn_norm.cu); dw3 == nullptr selects the forward
template <typename ST>
int norm_launch(const ST* wt, const ST* dw3, ST* out, int B, int G, int H, int W, unsigned mask,
                cudaStream_t st, LaunchInfo* li);

void set_error(const char* fmt, ...);

}  // namespace gspn
