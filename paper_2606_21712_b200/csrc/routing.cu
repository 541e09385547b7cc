// routing.cu -- steps a1-a5 of the combined MoE layer:
//   a1 router logits  L[t,e] = sum_j float(hidden[t,j]) * W_r[j,e] (+ b_r[e])      fp32 FMA
//   a2 top-k          k passes of a warp arg-max under (logit desc, expert index asc);
//                     gates = softmax over the k selected logits
//   a3 histogram      per-block shared-memory counts (integer atomics: order-independent)
//   a4 exclusive scan over experts (and over blocks, which gives every block its base row)
//   a5 stable rank    row = base[block][e] + #{earlier entries of the block with the same e}
// BASELINE.json north_star: "fp32 router top-k over all yielded tokens, a per-expert histogram and
// exclusive scan, a token permutation into expert-contiguous rows"; "ties broken by the lower
// expert index"; routing artefacts bit-exact given the same fp32 logits.
#include "kernels.h"
#include <cuda_bf16.h>
#include <math_constants.h>

namespace bg {
namespace {

constexpr int MAX_E = 256;
constexpr int MAX_K = 8;

// ------------------------------------------------------------------ a1 router logits
// Block: 32 tokens x all E experts, 256 threads.  Warp w owns tokens 4w..4w+3; lane l owns experts
// l, l+32, ... (NE = ceil(E/32) of them).  k is consumed in chunks of 32 staged in shared memory.
constexpr int RT_TOK = 32;
constexpr int RT_KC = 32;

template <int NE>
__global__ void __launch_bounds__(256) router_logits_kernel(const __nv_bfloat16* __restrict__ hidden,
                                                            const float* __restrict__ W_r,
                                                            const float* __restrict__ b_r, int T, int d, int E,
                                                            float* __restrict__ logits) {
  __shared__ float hs[RT_TOK][RT_KC + 1];
  __shared__ float ws[RT_KC][NE * 32];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t0 = blockIdx.x * RT_TOK;
  float acc[4][NE];
  #pragma unroll
  for (int i = 0; i < 4; ++i)
    #pragma unroll
    for (int j = 0; j < NE; ++j) acc[i][j] = 0.0f;

  for (int k0 = 0; k0 < d; k0 += RT_KC) {
    // hidden chunk: 32 tokens x 32 k; thread -> (token = tid/8, 4 consecutive k)
    {
      const int tt = threadIdx.x >> 3, kk = (threadIdx.x & 7) * 4;
      const int t = t0 + tt;
      float v[4] = {0.f, 0.f, 0.f, 0.f};
      if (t < T) {
        #pragma unroll
        for (int i = 0; i < 4; ++i)
          if (k0 + kk + i < d) v[i] = __bfloat162float(hidden[static_cast<int64_t>(t) * d + k0 + kk + i]);
      }
      #pragma unroll
      for (int i = 0; i < 4; ++i) hs[tt][kk + i] = v[i];
    }
    // W_r chunk: 32 k x E
    for (int idx = threadIdx.x; idx < RT_KC * NE * 32; idx += 256) {
      const int kk = idx / (NE * 32), e = idx - kk * (NE * 32);
      ws[kk][e] = (e < E && k0 + kk < d) ? __ldg(W_r + static_cast<int64_t>(k0 + kk) * E + e) : 0.0f;
    }
    __syncthreads();
    #pragma unroll 8
    for (int kk = 0; kk < RT_KC; ++kk) {
      float h[4], w[NE];
      #pragma unroll
      for (int i = 0; i < 4; ++i) h[i] = hs[warp * 4 + i][kk];
      #pragma unroll
      for (int j = 0; j < NE; ++j) w[j] = ws[kk][lane + 32 * j];
      #pragma unroll
      for (int i = 0; i < 4; ++i)
        #pragma unroll
        for (int j = 0; j < NE; ++j) acc[i][j] = fmaf(h[i], w[j], acc[i][j]);
    }
    __syncthreads();
  }
  #pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int t = t0 + warp * 4 + i;
    if (t >= T) continue;
    #pragma unroll
    for (int j = 0; j < NE; ++j) {
      const int e = lane + 32 * j;
      if (e < E) logits[static_cast<int64_t>(t) * E + e] = acc[i][j] + (b_r ? __ldg(b_r + e) : 0.0f);
    }
  }
}

// ------------------------------------------------------------------ a2 + a3
// (value, index) order of reading S3: a beats b <=> va > vb or (va == vb and ia < ib).
// An index < 0 marks "no candidate" and loses to everything.
__device__ __forceinline__ bool beats(float va, int ia, float vb, int ib) {
  if (ia < 0) return false;
  if (ib < 0) return true;
  return (va > vb) || (va == vb && ia < ib);
}

template <int NE>
__global__ void __launch_bounds__(256) topk_hist_kernel(const float* __restrict__ logits, int T, int E, int k,
                                                        int tokens_per_block, int32_t* __restrict__ topk_idx,
                                                        float* __restrict__ topk_w,
                                                        int32_t* __restrict__ block_counts) {
  __shared__ int hist[MAX_E];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int e = threadIdx.x; e < E; e += 256) hist[e] = 0;
  __syncthreads();
  const int t_begin = blockIdx.x * tokens_per_block;
  const int t_end = min(T, t_begin + tokens_per_block);
  for (int t = t_begin + warp; t < t_end; t += 8) {
    float v[NE];
    bool taken[NE];
    #pragma unroll
    for (int j = 0; j < NE; ++j) {
      const int e = lane + 32 * j;
      v[j] = (e < E) ? __ldg(logits + static_cast<int64_t>(t) * E + e) : 0.0f;
      taken[j] = !(e < E);
    }
    float sel_v[MAX_K];
    int sel_i[MAX_K];
    #pragma unroll
    for (int s = 0; s < MAX_K; ++s) {
      sel_v[s] = 0.0f;
      sel_i[s] = 0;
      if (s < k) {
        float bv = 0.0f;
        int bi = -1;
        #pragma unroll
        for (int j = 0; j < NE; ++j)
          if (!taken[j] && beats(v[j], lane + 32 * j, bv, bi)) { bv = v[j]; bi = lane + 32 * j; }
        #pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
          const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
          if (beats(ov, oi, bv, bi)) { bv = ov; bi = oi; }
        }
        // every lane now holds the same winner
        #pragma unroll
        for (int j = 0; j < NE; ++j)
          if (bi == lane + 32 * j) taken[j] = true;
        sel_v[s] = bv;
        sel_i[s] = bi;
      }
    }
    // gates: softmax over the k selected logits, slot 0 holds the maximum (reading S2)
    float ex[MAX_K], denom = 0.0f;
    #pragma unroll
    for (int s = 0; s < MAX_K; ++s) {
      ex[s] = (s < k) ? expf(sel_v[s] - sel_v[0]) : 0.0f;
      denom += ex[s];
    }
    #pragma unroll
    for (int s = 0; s < MAX_K; ++s) {
      if (s < k && lane == s) {
        topk_idx[static_cast<int64_t>(t) * k + s] = sel_i[s];
        topk_w[static_cast<int64_t>(t) * k + s] = ex[s] / denom;
        atomicAdd(&hist[sel_i[s]], 1);
      }
    }
  }
  __syncthreads();
  for (int e = threadIdx.x; e < E; e += 256) block_counts[static_cast<int64_t>(blockIdx.x) * E + e] = hist[e];
}

// Recount per-block histograms from topk_idx (split API: bg_moe_permute gets only idx + offsets).
__global__ void __launch_bounds__(256) block_hist_kernel(const int32_t* __restrict__ topk_idx, int T, int E, int k,
                                                         int tokens_per_block,
                                                         int32_t* __restrict__ block_counts) {
  __shared__ int hist[MAX_E];
  for (int e = threadIdx.x; e < E; e += 256) hist[e] = 0;
  __syncthreads();
  const int64_t i0 = static_cast<int64_t>(blockIdx.x) * tokens_per_block * k;
  const int64_t n = min(static_cast<int64_t>(tokens_per_block) * k, static_cast<int64_t>(T) * k - i0);
  if (threadIdx.x < n) {
    const int e = __ldg(topk_idx + i0 + threadIdx.x);
    if (e >= 0 && e < E) atomicAdd(&hist[e], 1);
  }
  __syncthreads();
  for (int e = threadIdx.x; e < E; e += 256) block_counts[static_cast<int64_t>(blockIdx.x) * E + e] = hist[e];
}

// ------------------------------------------------------------------ a4 scans (one block of 256)
// counts[e] = sum_b block_counts[b][e]; offsets = exclusive scan over e; then
// block_base[b][e] = offsets[e] + sum_{b'<b} block_counts[b'][e]   (first row of block b in expert e)
__global__ void __launch_bounds__(256) scan_kernel(const int32_t* __restrict__ block_counts, int nblk, int E,
                                                   int32_t* __restrict__ block_base,
                                                   int32_t* __restrict__ counts, int32_t* __restrict__ offsets) {
  __shared__ int warp_tot[8];
  const int e = threadIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int total = 0;
  if (e < E) {
    #pragma unroll 8
    for (int b = 0; b < nblk; ++b) total += __ldg(block_counts + static_cast<int64_t>(b) * E + e);
  }
  int v = total;
  #pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int u = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += u;
  }
  if (lane == 31) warp_tot[warp] = v;
  __syncthreads();
  int add = 0;
  for (int w = 0; w < warp; ++w) add += warp_tot[w];
  const int incl = v + add;
  const int excl = incl - total;
  if (e < E) {
    if (counts) counts[e] = total;
    if (offsets) {
      offsets[e] = excl;
      if (e == E - 1) offsets[E] = incl;
    }
    int run = excl;
    #pragma unroll 8
    for (int b = 0; b < nblk; ++b) {
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
__global__ void __launch_bounds__(256) rank_kernel(const int32_t* __restrict__ topk_idx,
                                                   const int32_t* __restrict__ block_base, int T, int E, int k,
                                                   int tokens_per_block, int32_t* __restrict__ row_src,
                                                   int32_t* __restrict__ inv_perm) {
  __shared__ int wcnt[8][MAX_E];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < 8 * MAX_E; i += 256) (&wcnt[0][0])[i] = 0;
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
  }
}

}  // namespace

cudaError_t launch_router_logits(const void* hidden, const float* W_r, const float* b_r, int T, int d, int E,
                                 float* logits, cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  const __nv_bfloat16* h = static_cast<const __nv_bfloat16*>(hidden);
  const int grid = (T + RT_TOK - 1) / RT_TOK;
  const int ne = (E + 31) / 32;
  switch (ne) {
    case 1: router_logits_kernel<1><<<grid, 256, 0, st>>>(h, W_r, b_r, T, d, E, logits); break;
    case 2: router_logits_kernel<2><<<grid, 256, 0, st>>>(h, W_r, b_r, T, d, E, logits); break;
    case 3: case 4: router_logits_kernel<4><<<grid, 256, 0, st>>>(h, W_r, b_r, T, d, E, logits); break;
    default: router_logits_kernel<8><<<grid, 256, 0, st>>>(h, W_r, b_r, T, d, E, logits); break;
  }
  return cudaGetLastError();
}

cudaError_t launch_topk_hist(const float* logits, int T, int E, int k, int32_t* topk_idx, float* topk_w,
                             int32_t* block_counts, cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  const int tb = route_tokens_per_block(k), grid = route_num_blocks(T, k);
  const int ne = (E + 31) / 32;
  switch (ne) {
    case 1: topk_hist_kernel<1><<<grid, 256, 0, st>>>(logits, T, E, k, tb, topk_idx, topk_w, block_counts); break;
    case 2: topk_hist_kernel<2><<<grid, 256, 0, st>>>(logits, T, E, k, tb, topk_idx, topk_w, block_counts); break;
    case 3: case 4: topk_hist_kernel<4><<<grid, 256, 0, st>>>(logits, T, E, k, tb, topk_idx, topk_w, block_counts); break;
    default: topk_hist_kernel<8><<<grid, 256, 0, st>>>(logits, T, E, k, tb, topk_idx, topk_w, block_counts); break;
  }
  return cudaGetLastError();
}

cudaError_t launch_block_hist(const int32_t* topk_idx, int T, int E, int k, int32_t* block_counts,
                              cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  block_hist_kernel<<<route_num_blocks(T, k), 256, 0, st>>>(topk_idx, T, E, k, route_tokens_per_block(k),
                                                             block_counts);
  return cudaGetLastError();
}

cudaError_t launch_scan(const int32_t* block_counts, int nblk, int E, int32_t* block_base, int32_t* counts,
                        int32_t* offsets, cudaStream_t st) {
  scan_kernel<<<1, 256, 0, st>>>(block_counts, nblk, E, block_base, counts, offsets);
  return cudaGetLastError();
}

cudaError_t launch_rank(const int32_t* topk_idx, const int32_t* block_base, int T, int E, int k,
                        int32_t* row_src, int32_t* inv_perm, cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  rank_kernel<<<route_num_blocks(T, k), 256, 0, st>>>(topk_idx, block_base, T, E, k, route_tokens_per_block(k),
                                                       row_src, inv_perm);
  return cudaGetLastError();
}

}  // namespace bg
