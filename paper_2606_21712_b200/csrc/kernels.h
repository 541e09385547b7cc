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
// the five kernels of the fused chain.
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

// ---- fused router (router_fused.cu): steps a1-a4 + tile-local ranks in one kernel
cudaError_t router_kernels_init();
// pieces: bf16 [3][d][round_up(E,16)] = exact hi/mid/lo split of W_r (zero padded)
cudaError_t launch_split_wr(const float* W_r, int d, int E, void* pieces, cudaStream_t st);
int router_nch(int d);   // K chunks = cluster size of the router: a function of d only

// Routing works on tiles of 128 consecutive tokens (routing_common.cuh).
inline int route_num_tiles(int T) { return (T + 127) / 128; }

struct RouterLaunch {
  int T, d, E, k;
  const float* b_r;         // [E] or nullptr
  float* logits_out;        // [T,E]
  int32_t* topk_idx;        // [T,k]
  float* topk_w;            // [T,k]
  int32_t* tile_rank;       // [T,k]
  int32_t* tile_counts;     // [route_num_tiles(T), E]
  int32_t* tile_base;       // [route_num_tiles(T), E]
  int32_t* counts;          // [E]
  int32_t* offsets;         // [E+1]
  int32_t* done_counter;    // one int, zero between launches (re-armed by the kernel)
  int32_t* gemm_counters;   // eight ints zeroed by the kernel's last tile (or nullptr)
  int num_sms;
  int force_form;           // 0 = choose from T (router_sequential); 1 = sequential form; 2 = cluster form (tests)
};

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
  int64_t logits, idx, w, pieces, counts, offsets, tc, tb, tr, rs, ip, wp, x, h, y, hd, od, seg_hidden, seg_out,
      seg_start, tile_counters, total;
};
WsLayout ws_layout(const bg_moe_config& c, int64_t max_tokens, int num_sms);

// tm_h: hidden [T,d] (box {64 k, 128 rows}), ignored when seg != nullptr (rows come through the segment table);
// tm_w: box of all three W_r pieces (4-D view) or one 3-D block; tm_w1: the 4-D view with a one-piece box.
cudaError_t launch_router_fused(const CUtensorMap* tm_h, const CUtensorMap& tm_w, const CUtensorMap& tm_w1,
                                const RouterLaunch& r, const SegTable* seg, cudaStream_t st);

// ---- stand-alone routing kernels of the split API (routing.cu)
// a2 + a3 + tile-local rank from given logits [T,E].
cudaError_t launch_topk_tile(const float* logits, int T, int E, int k, int32_t* topk_idx, float* topk_w,
                             int32_t* tile_rank, int32_t* tile_counts, cudaStream_t st);
// a3 + tile-local rank from given indices [T,k].
cudaError_t launch_tile_rank(const int32_t* topk_idx, int T, int E, int k, int32_t* tile_rank, int32_t* tile_counts,
                             cudaStream_t st);
// a4: tile_counts [n_tiles,E] -> tile_base [n_tiles,E] (expert offset + exclusive prefix over tiles), counts [E],
// offsets [E+1] (either may be NULL).  n_tiles == 0 writes zeros.
cudaError_t launch_scan(const int32_t* tile_counts, int n_tiles, int E, int32_t* tile_base, int32_t* counts,
                        int32_t* offsets, cudaStream_t st);

// ---- gather / reduce (gather_reduce.cu): steps a6 and a9
// seg != nullptr: token rows are read from / written to the segments' own buffers (hidden / out unused).
// The gather also finishes the permutation (a5): row(t,s) = tile_base[t/128][idx[t,s]] + tile_rank[t,s].
struct PermLaunch {
  const int32_t* topk_idx;   // [T,k]
  const int32_t* tile_rank;  // [T,k]
  const int32_t* tile_base;  // [n_tiles,E]
  const float* topk_w;       // [T,k] or nullptr
  int32_t* row_src;          // [T*k]
  int32_t* inv_perm;         // [T*k]
  float* w_perm;             // [T*k] gate weights in expert order, or nullptr
};
// x_perm == nullptr: only the permutation is written.
cudaError_t launch_gather(const void* hidden, const PermLaunch& pl, int T, int E, int k, int d, void* x_perm,
                          int num_sms, cudaStream_t st, const SegTable* seg = nullptr);
// weights == nullptr: plain sum (fused path, Y already gate-weighted).
cudaError_t launch_unpermute(const void* y_perm, const int32_t* inv_perm, const float* weights, int T, int k,
                             int d, void* out, int num_sms, cudaStream_t st, const SegTable* seg = nullptr);

// ---- FP8 quantisation (fp8_quant.cu; readings F1-F3 of DESIGN.md §2)
// W [E, K, N] bf16 -> Wq [E, N, K] e4m3 bytes + sw [E, N] fp32 (one scale per expert and output channel)
cudaError_t launch_quantize_weights(const void* W, int E, int K, int N, void* Wq, float* sw, cudaStream_t st);
// a5'' + a6 with quantisation: as launch_gather, but the k expert-order rows of a token are written as e4m3 bytes
// xq_perm [T*k, d] with the token's fp32 scale in sx_perm [T*k]
// hmax (may be NULL): [T*k] zeroed here for the rows the token owns (the gate/up epilogue accumulates max |H| there)
cudaError_t launch_gather_fp8(const void* hidden, const PermLaunch& pl, int T, int E, int k, int d, void* xq_perm,
                              float* sx_perm, unsigned* hmax, int num_sms, cudaStream_t st, const SegTable* seg = nullptr);
// Reading F5: H [rows, f] bf16 + hmax [rows] (float bits of max |H[r,:]|) -> Hq [rows, f] e4m3, sh [rows] = max / 448,
// sc [rows] = sh * (w_perm ? w_perm[r] : 1): the per-row factor the down GEMM's epilogue applies
cudaError_t launch_quantize_h(const void* H, const unsigned* hmax, const float* w_perm, int64_t rows, int f, void* Hq,
                              float* sh, float* sc, int num_sms, cudaStream_t st);

// ---- grouped GEMM (grouped_gemm_pair.cu): steps a7 and a8
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
  const float* row_scale_perm;   // down GEMM, fused path: gate weights in expert order, w_perm[r] = topk_w[row_src[r]] (else nullptr)
  // FP8 gate/up (launch_gateup_swiglu_pair_fp8): dequantisation scales
  const float* sx = nullptr;     // [rows] per expert-order token row
  const float* sw0 = nullptr;    // [E, N] W_gate, per expert and output channel
  const float* sw1 = nullptr;    // [E, N] W_up
  unsigned* hmax = nullptr;      // gate/up GEMM: [rows] running max |H| as float bits (FP8 down GEMM downstream), or nullptr
  int num_sms;
};
// CTA-pair kernels (grouped_gemm_pair.cu): weights on UMMA M (256 per pair), tokens on UMMA N.
cudaError_t launch_gateup_swiglu_pair(const GemmLaunch& g, cudaStream_t st);
cudaError_t launch_gateup_swiglu_pair_fp8(const GemmLaunch& g, cudaStream_t st);
cudaError_t launch_down_pair_fp8(const GemmLaunch& g, cudaStream_t st);
cudaError_t launch_down_pair(const GemmLaunch& g, cudaStream_t st);
cudaError_t pair_kernels_init();

}  // namespace bg
