// routing.cu -- steps a1-a5 of the combined MoE layer:
//   a1 (tail)         L[t,e] = sum_s partial[s][t][e] (+ b_r[e]): the split-K partials of
//                     router_gemm.cu added in ascending s (fixed order => deterministic logits)
//   a2 top-k          k passes of a warp arg-max under (logit desc, expert index asc);
//                     gates = softmax over the k selected logits
//   a3 histogram      per-block shared-memory counts (integer atomics: order-independent)
//   a4 exclusive scan over experts (and over blocks, which gives every block its base row)
//   a5 stable rank    row = base[block][e] + #{earlier entries of the block with the same e}
// BASELINE.json north_star: "fp32 router top-k over all yielded tokens, a per-expert histogram and
// exclusive scan, a token permutation into expert-contiguous rows"; "ties broken by the lower
// expert index"; routing artefacts bit-exact given the same fp32 logits.
#include "kernels.h"
#include "ptx_sm100.cuh"
#include <cuda_bf16.h>
#include <math_constants.h>

namespace bg {
namespace {

constexpr int MAX_E = 256;

// ------------------------------------------------------------------ a2 + a3
// One warp per token.  (logit, expert) is packed into one 64-bit key whose unsigned order IS the
// order of reading S3: larger logit first, equal logits -> lower expert index first
// (-0.0 == +0.0: both map to the same key half).  Lane l holds the keys of experts l, l+32, ...
constexpr int RB = 1024;     // flat (token,slot) entries owned by one block of the rank kernel

__device__ __forceinline__ uint32_t float_to_ordered(float f) {
  f = f + 0.0f;                                    // canonicalise -0.0 to +0.0 (they tie)
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ordered_to_float(uint32_t o) {
  return __uint_as_float((o & 0x80000000u) ? (o ^ 0x80000000u) : ~o);
}

// src: fp32 [n_src][T][E]: n_src >= 1 slabs added in ascending order (n_src = 1: plain logits),
// plus b_r.  logits_out (never aliases src) receives the summed logits.  block_counts [nblk][E]
// must be zero on entry; it receives the histogram of each rank block (integer RED: the result
// does not depend on arrival order).
template <int NE>
__global__ void __launch_bounds__(256) topk_hist_kernel(const float* __restrict__ src, int n_src,
                                                        const float* __restrict__ b_r,
                                                        float* __restrict__ logits_out, int T, int E, int k,
                                                        int tokens_per_block, int32_t* __restrict__ topk_idx,
                                                        float* __restrict__ topk_w,
                                                        int32_t* __restrict__ block_counts) {
  pdl_wait_then_trigger();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * 8 + warp;
  if (t >= T) return;
  const int64_t slab = static_cast<int64_t>(T) * E;
  // Sum of the n_src slabs in ascending order (+ bias); loads are issued SB slabs at a time so
  // their latencies overlap while the additions stay in slab order (deterministic logits).
  constexpr int SB = (NE <= 4) ? 4 : 2;
  float v[NE];
  {
    const float* p = src + static_cast<int64_t>(t) * E + lane;
    #pragma unroll
    for (int j = 0; j < NE; ++j) v[j] = (lane + 32 * j < E) ? __ldg(p + 32 * j) : 0.0f;
    for (int s = 1; s < n_src; s += SB) {
      float a[SB][NE];
      #pragma unroll
      for (int u = 0; u < SB; ++u)
        #pragma unroll
        for (int j = 0; j < NE; ++j)
          a[u][j] = (s + u < n_src && lane + 32 * j < E) ? __ldg(p + (s + u) * slab + 32 * j) : 0.0f;
      #pragma unroll
      for (int u = 0; u < SB; ++u)
        #pragma unroll
        for (int j = 0; j < NE; ++j)
          if (s + u < n_src) v[j] += a[u][j];
    }
  }
  unsigned long long key[NE];
  #pragma unroll
  for (int j = 0; j < NE; ++j) {
    const int e = lane + 32 * j;
    key[j] = 0ull;                                  // 0 = "no candidate": below every real key
    if (e < E) {
      if (b_r) v[j] += __ldg(b_r + e);
      if (logits_out) logits_out[static_cast<int64_t>(t) * E + e] = v[j];
      key[j] = (static_cast<unsigned long long>(float_to_ordered(v[j])) << 32) | (0xFFFFFFFFu - static_cast<uint32_t>(e));
    }
  }
  int my_e = 0;
  float my_v = 0.0f, v_max = 0.0f;
  for (int s = 0; s < k; ++s) {
    unsigned long long best = key[0];
    #pragma unroll
    for (int j = 1; j < NE; ++j) best = max(best, key[j]);
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    #pragma unroll
    for (int j = 0; j < NE; ++j)
      if (key[j] == best) key[j] = 0ull;            // taken
    const float val = ordered_to_float(static_cast<uint32_t>(best >> 32));
    if (s == 0) v_max = val;
    if (lane == s) { my_e = static_cast<int>(0xFFFFFFFFu - static_cast<uint32_t>(best)); my_v = val; }
  }
  // gates: softmax over the k selected logits; slot 0 holds the maximum (reading S2)
  const float ex = (lane < k) ? expf(my_v - v_max) : 0.0f;
  float denom = 0.0f;
  for (int s = 0; s < k; ++s) denom += __shfl_sync(0xffffffffu, ex, s);     // slot order
  if (lane < k) {
    topk_idx[static_cast<int64_t>(t) * k + lane] = my_e;
    topk_w[static_cast<int64_t>(t) * k + lane] = ex / denom;
    atomicAdd(block_counts + static_cast<int64_t>(t / tokens_per_block) * E + my_e, 1);
  }
}

// Recount per-block histograms from topk_idx (split API: bg_moe_permute gets only idx + offsets).
__global__ void __launch_bounds__(RB) block_hist_kernel(const int32_t* __restrict__ topk_idx, int T, int E, int k,
                                                         int tokens_per_block,
                                                         int32_t* __restrict__ block_counts) {
  pdl_wait_then_trigger();
  __shared__ int hist[MAX_E];
  for (int e = threadIdx.x; e < E; e += RB) hist[e] = 0;
  __syncthreads();
  const int64_t i0 = static_cast<int64_t>(blockIdx.x) * tokens_per_block * k;
  const int64_t n = min(static_cast<int64_t>(tokens_per_block) * k, static_cast<int64_t>(T) * k - i0);
  if (threadIdx.x < n) {
    const int e = __ldg(topk_idx + i0 + threadIdx.x);
    if (e >= 0 && e < E) atomicAdd(&hist[e], 1);
  }
  __syncthreads();
  for (int e = threadIdx.x; e < E; e += RB) block_counts[static_cast<int64_t>(blockIdx.x) * E + e] = hist[e];
}

// ------------------------------------------------------------------ a4 scans (one block of 1024)
// counts[e] = sum_b block_counts[b][e]; offsets = exclusive scan over e; then
// block_base[b][e] = offsets[e] + sum_{b'<b} block_counts[b'][e]   (first row of block b in expert e)
// Thread (g, e): expert e = tid % 256, block group g = tid / 256 owns blocks [g*per, (g+1)*per).
__global__ void __launch_bounds__(1024) scan_kernel(const int32_t* __restrict__ block_counts, int nblk, int E,
                                                    int32_t* __restrict__ block_base,
                                                    int32_t* __restrict__ counts, int32_t* __restrict__ offsets) {
  pdl_wait_then_trigger();
  __shared__ int gtot[4][MAX_E];
  __shared__ int excl_e[MAX_E];
  __shared__ int warp_tot[8];
  const int e = threadIdx.x & 255, g = threadIdx.x >> 8;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int per = (nblk + 3) / 4;
  const int b0 = min(nblk, g * per), b1 = min(nblk, b0 + per);
  int part = 0;
  if (e < E) {
    #pragma unroll 8
    for (int b = b0; b < b1; ++b) part += __ldg(block_counts + static_cast<int64_t>(b) * E + e);
  }
  gtot[g][e] = part;
  __syncthreads();
  if (g == 0) {
    const int total = gtot[0][e] + gtot[1][e] + gtot[2][e] + gtot[3][e];
    int v = total;
    #pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v += u;
    }
    if (lane == 31) warp_tot[warp] = v;
    asm volatile("bar.sync 1, 256;" ::: "memory");      // only the 256 threads of group 0
    int add = 0;
    for (int w = 0; w < warp; ++w) add += warp_tot[w];
    const int incl = v + add, excl = incl - total;
    excl_e[e] = excl;
    if (e < E) {
      if (counts) counts[e] = total;
      if (offsets) {
        offsets[e] = excl;
        if (e == E - 1) offsets[E] = incl;
      }
    }
  }
  __syncthreads();
  if (e < E) {
    int run = excl_e[e];
    for (int gg = 0; gg < g; ++gg) run += gtot[gg][e];
    #pragma unroll 8
    for (int b = b0; b < b1; ++b) {
      const int64_t at = static_cast<int64_t>(b) * E + e;
      block_base[at] = run;
      run += __ldg(block_counts + at);
    }
  }
}

// ------------------------------------------------------------------ a5 stable rank
// One thread per flat entry of the block.  Entries of a block are in flat-index order, so the
// rank of entry j inside its expert is (#lower warps' entries with the same expert) + (#lower
// lanes of this warp with the same expert): independent of any arrival order.
__global__ void __launch_bounds__(RB) rank_kernel(const int32_t* __restrict__ topk_idx,
                                                   const int32_t* __restrict__ block_base, int T, int E, int k,
                                                   int tokens_per_block, int32_t* __restrict__ row_src,
                                                   int32_t* __restrict__ inv_perm, const float* __restrict__ topk_w,
                                                   float* __restrict__ w_perm) {
  pdl_wait_then_trigger();
  __shared__ int wcnt[RB / 32][MAX_E];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < (RB / 32) * MAX_E; i += RB) (&wcnt[0][0])[i] = 0;
  __syncthreads();
  const int64_t i0 = static_cast<int64_t>(blockIdx.x) * tokens_per_block * k;
  const int64_t n = min(static_cast<int64_t>(tokens_per_block) * k, static_cast<int64_t>(T) * k - i0);
  const bool active = threadIdx.x < n;
  int e = -1;
  if (active) e = __ldg(topk_idx + i0 + threadIdx.x);
  const bool ok = active && e >= 0 && e < E;
  // lanes with the same expert (inactive lanes form their own group with key -1)
  const unsigned same = __match_any_sync(0xffffffffu, ok ? e : -1);
  const int rank_in_warp = __popc(same & ((1u << lane) - 1u));
  if (ok && rank_in_warp == 0) wcnt[warp][e] = __popc(same);
  __syncthreads();
  if (ok) {
    int r = __ldg(block_base + static_cast<int64_t>(blockIdx.x) * E + e) + rank_in_warp;
    for (int w = 0; w < warp; ++w) r += wcnt[w][e];
    const int64_t i = i0 + threadIdx.x;
    row_src[r] = static_cast<int32_t>(i);
    inv_perm[i] = r;
    if (w_perm != nullptr) w_perm[r] = __ldg(topk_w + i);
  }
}

}  // namespace

cudaError_t launch_topk_hist(const float* src, int n_src, const float* b_r, float* logits_out, int T, int E, int k,
                             int32_t* topk_idx, float* topk_w, int32_t* block_counts, cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  const int tb = route_tokens_per_block(k);
  const int ne = (E + 31) / 32;
#define BG_TOPK(NE_) launch_pdl(topk_hist_kernel<NE_>, (T + 7) / 8, 256, 0, st, src, n_src, b_r, logits_out, T, E, k, tb, \
                                                                       topk_idx, topk_w, block_counts)
  switch (ne) {
    case 1: BG_TOPK(1); break;
    case 2: BG_TOPK(2); break;
    case 3: case 4: BG_TOPK(4); break;
    default: BG_TOPK(8); break;
  }
#undef BG_TOPK
  return cudaGetLastError();
}

cudaError_t launch_block_hist(const int32_t* topk_idx, int T, int E, int k, int32_t* block_counts,
                              cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  launch_pdl(block_hist_kernel, route_num_blocks(T, k), RB, 0, st, topk_idx, T, E, k, route_tokens_per_block(k),
                                                            block_counts);
  return cudaGetLastError();
}

cudaError_t launch_scan(const int32_t* block_counts, int nblk, int E, int32_t* block_base, int32_t* counts,
                        int32_t* offsets, cudaStream_t st) {
  launch_pdl(scan_kernel, 1, 1024, 0, st, block_counts, nblk, E, block_base, counts, offsets);
  return cudaGetLastError();
}

cudaError_t launch_rank(const int32_t* topk_idx, const int32_t* block_base, int T, int E, int k,
                        int32_t* row_src, int32_t* inv_perm, const float* topk_w, float* w_perm,
                        cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  launch_pdl(rank_kernel, route_num_blocks(T, k), RB, 0, st, topk_idx, block_base, T, E, k, route_tokens_per_block(k),
                                                      row_src, inv_perm, topk_w, w_perm);
  return cudaGetLastError();
}

}  // namespace bg
