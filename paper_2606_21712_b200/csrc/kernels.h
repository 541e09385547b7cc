// kernels.h -- internal launcher interface between api.cu and the kernel translation units.
// Not part of the public ABI (include/bg_moe.h is).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/bg_moe.h"

namespace bg {

// Launch with programmatic stream serialization (PDL): the kernel may begin before the previous
// kernel on the stream has finished; each kernel calls pdl_wait_then_trigger() (ptx_sm100.cuh)
// before it touches anything its predecessor wrote.  Hides launch latency and prologues between
// the eight kernels of the fused chain.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// ---- router logits on tensor cores (router_gemm.cu): step a1
cudaError_t router_kernels_init();
// pieces: bf16 [3][d][round_up(E,16)] = exact hi/mid/lo split of W_r (zero padded)
cudaError_t launch_split_wr(const float* W_r, int d, int E, void* pieces, cudaStream_t st);
int router_ksplit(int T, int d, int num_sms);
// partial: fp32 [ksplit][T][E].  Also zeroes zero_buf[0..zero_n) (the histogram the top-k kernel fills).
// tm_w: box of all three pieces (4-D view) or one 3-D block; tm_w1: the 4-D view with a one-piece box
cudaError_t launch_router_gemm(const CUtensorMap& tm_h, const CUtensorMap& tm_w, const CUtensorMap& tm_w1, int T, int d, int E, int ksplit,
                               float* partial, int32_t* zero_buf, int zero_n, cudaStream_t st);

// ---- segments (zero-copy COMBINE): the combined tokens given as a list
// of per-coroutine buffers.  Token t lives in row (t - start[s]) of hidden[s] (and of out[s]), s = the segment
// with start[s] <= t < start[s+1].  All three arrays are DEVICE arrays.
struct SegTable {
  const void* const* hidden;   // [n] bf16 [n_tokens_s, d]
  void* const* out;            // [n] bf16 [n_tokens_s, d]
  const int32_t* start;        // [n+1] exclusive prefix sum of the segment lengths
  int n;
};

// ---- workspace layout (plan.cu): byte offsets of every slab of the context's single allocation
struct WsLayout {
  int64_t logits, idx, w, part, pieces, counts, offsets, bc, bb, rs, ip, wp, x, h, y, hd, od, seg_hidden, seg_out,
      seg_start, tile_counters, total;
};
WsLayout ws_layout(const bg_moe_config& c, int64_t max_tokens, int num_sms);

cudaError_t launch_router_gemm_segments(const SegTable& seg, const CUtensorMap& tm_w, const CUtensorMap& tm_w1, int T,
                                        int d, int E, int ksplit, float* partial, int32_t* zero_buf, int zero_n,
                                        cudaStream_t st);

// ---- routing (routing.cu): steps a1 (sum of partials + bias) - a5 of DESIGN.md §1
// Tokens handled by one block of the top-k / rank kernels: chosen so that a block owns at most
// 1024 flat (token,slot) entries, one per thread of the rank kernel.
inline int route_tokens_per_block(int k) { return 1024 / k; }
inline int route_num_blocks(int T, int k) {
  const int tb = route_tokens_per_block(k);
  return (T + tb - 1) / tb;
}

// src: fp32 [n_src][T][E] slabs added in ascending order (+ b_r) -> logits_out (may be NULL).
// block_counts [route_num_blocks][E] must be zero on entry (router kernel or a memset does that).
cudaError_t launch_topk_hist(const float* src, int n_src, const float* b_r, float* logits_out, int T, int E, int k,
                             int32_t* topk_idx, float* topk_w, int32_t* block_counts, cudaStream_t st);
// block_counts [nblk,E]: per-block counts -> block_base [nblk,E]: expert offset + exclusive prefix
// over blocks (the first row of block b inside expert e).  counts / offsets may be NULL.
cudaError_t launch_scan(const int32_t* block_counts, int nblk, int E, int32_t* block_base, int32_t* counts,
                        int32_t* offsets, cudaStream_t st);
// Recomputes block_counts from topk_idx (used by the split bg_moe_permute, which receives only
// topk_idx and offsets).
cudaError_t launch_block_hist(const int32_t* topk_idx, int T, int E, int k, int32_t* block_counts,
                              cudaStream_t st);
// topk_w / w_perm may be nullptr; otherwise w_perm[r] = topk_w[row_src[r]] (gate weights in expert order).
cudaError_t launch_rank(const int32_t* topk_idx, const int32_t* block_base, int T, int E, int k,
                        int32_t* row_src, int32_t* inv_perm, const float* topk_w, float* w_perm, cudaStream_t st);

// ---- gather / reduce (gather_reduce.cu): steps a6 and a9
// seg != nullptr: token rows are read from / written to the segments' own buffers (hidden / out unused).
cudaError_t launch_gather(const void* hidden, const int32_t* inv_perm, int T, int k, int d, void* x_perm,
                          int num_sms, cudaStream_t st, const SegTable* seg = nullptr);
// weights == nullptr: plain sum (fused path, Y already gate-weighted).
cudaError_t launch_unpermute(const void* y_perm, const int32_t* inv_perm, const float* weights, int T, int k,
                             int d, void* out, int num_sms, cudaStream_t st, const SegTable* seg = nullptr);

// ---- grouped GEMM (grouped_gemm.cu): steps a7 and a8
// Activation tensor maps: the same [rows, K] bf16 matrix with TMA boxes of {64 k, 8 (i + 1) rows},
// so that any token count that is a multiple of 8 (<= 128) is ONE TMA operation: the TMA unit's
// per-operation cost (~40 ns), not its bandwidth, is what limits a 64-wide k-block.
struct ActMaps {
  CUtensorMap m[16];   // box rows 8, 16, ..., 128
};
struct GemmLaunch {
  ActMaps tm_act;      // activations [rows, K] bf16
  CUtensorMap tm_b0;   // weights [E, K, N] bf16, box {64, 64, 1}: W_gate (gate/up GEMM) or W_down
  CUtensorMap tm_b1;   // W_up (gate/up GEMM only)
  // The same weights viewed as [E, N/64, K, 64] with box {64 n, 64 k, nblk, 1}: one TMA operation
  // brings nblk 64-column blocks in the [block][k][64 n] order the MN-major UMMA operand wants.
  // Valid only when N % 64 == 0 (w4d); otherwise the kernels issue one 3-D box per block.
  CUtensorMap tm_b0_4d, tm_b1_4d;
  bool w4d;
  int* tile_counter;   // pair kernel, dynamic tile feed: two ints (tickets, clusters finished), zero between launches; nullptr = static
  int sg_max;          // pair kernel: token tiles per super-group (0 = sized from K to ~48 MB of tokens)
  const int32_t* offsets;  // [E+1]
  int E, K, N;         // N = output columns (f for gate/up, d for down)
  void* out;           // bf16 [rows, N]
  const float* row_scale;   // down GEMM, fused path: topk_w flat [T*k] (else nullptr)
  const int32_t* row_src;   // down GEMM, fused path: row -> flat index
  const float* row_scale_perm;   // down GEMM, fused path: the same gate weights in expert order, w_perm[r] = topk_w[row_src[r]]
  int num_sms;
};
cudaError_t launch_gateup_swiglu(const GemmLaunch& g, cudaStream_t st);
cudaError_t launch_down(const GemmLaunch& g, cudaStream_t st);
cudaError_t gemm_kernels_init();   // sets the dynamic shared-memory attributes once
// CTA-pair kernels (grouped_gemm_pair.cu): weights on UMMA M (256 per pair), tokens on UMMA N.
cudaError_t launch_gateup_swiglu_pair(const GemmLaunch& g, cudaStream_t st);
cudaError_t launch_down_pair(const GemmLaunch& g, cudaStream_t st);
cudaError_t pair_kernels_init();

}  // namespace bg
