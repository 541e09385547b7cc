// routing.cu -- the stand-alone routing kernels of the SPLIT API.  The fused chain and
// bg_moe_route(hidden) run steps a1-a4 inside router_fused.cu; these kernels serve the calls that start from
// something other than hidden states:
//   topk_tile_kernel   bg_moe_route(logits_in = ...): a2 top-k + gates, a3 per-tile histogram, tile-local rank
//   tile_rank_kernel   bg_moe_permute(topk_idx, offsets): per-tile histogram + tile-local rank from given indices
//   scan_kernel        a4 over tiles and experts (the fused router does this in its last tile)
// BASELINE.json north_star: "fp32 router top-k over all yielded tokens, a per-expert histogram and exclusive
// scan, a token permutation into expert-contiguous rows"; "ties broken by the lower expert index"; routing
// artefacts bit-exact given the same fp32 logits.
#include "kernels.h"
#include "ptx_sm100.cuh"
#include "routing_common.cuh"

namespace bg {
namespace {

__device__ __forceinline__ void bar128() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

// One block per 128-token tile, 4 warps; each warp takes the tile's tokens w, w+4, ...: (logit, expert) is packed
// into one 64-bit key whose unsigned order IS the order of reading S3 (larger logit first, equal logits -> lower
// expert index first); lane l holds the keys of experts l, l+32, ...; k rounds of a warp arg-max.
template <int NE>
__global__ void __launch_bounds__(ROUTE_TILE) topk_tile_kernel(const float* __restrict__ logits, int T, int E, int k,
                                                               int32_t* __restrict__ topk_idx,
                                                               float* __restrict__ topk_w,
                                                               int32_t* __restrict__ tile_rank,
                                                               int32_t* __restrict__ tile_counts) {
  pdl_wait_then_trigger();
  __shared__ int idx_tile[ROUTE_TILE * ROUTE_MAX_K];
  __shared__ uint32_t mask[ROUTE_MAX_E * 4];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < ROUTE_MAX_E * 4; i += ROUTE_TILE) mask[i] = 0u;
  for (int row = warp; row < ROUTE_TILE; row += 4) {
    const int t = blockIdx.x * ROUTE_TILE + row;
    if (t >= T) {
      if (lane < ROUTE_MAX_K) idx_tile[row * ROUTE_MAX_K + lane] = -1;
      continue;
    }
    unsigned long long key[NE];
    #pragma unroll
    for (int j = 0; j < NE; ++j) {
      const int e = lane + 32 * j;
      key[j] = 0ull;                                  // 0 = "no candidate": below every real key
      if (e < E)
        key[j] = (static_cast<unsigned long long>(float_to_ordered(__ldg(logits + static_cast<int64_t>(t) * E + e))) << 32) |
                 (0xFFFFFFFFu - static_cast<uint32_t>(e));
    }
    int my_e = -1;
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
    }
    if (lane < ROUTE_MAX_K) idx_tile[row * ROUTE_MAX_K + lane] = (lane < k) ? my_e : -1;
  }
  __syncthreads();
  const int row = threadIdx.x, t = blockIdx.x * ROUTE_TILE + row;
  int e[ROUTE_MAX_K], rk[ROUTE_MAX_K];
  #pragma unroll
  for (int s = 0; s < ROUTE_MAX_K; ++s) e[s] = idx_tile[row * ROUTE_MAX_K + s];
  tile_rank_and_counts(mask, row, e, k, E, rk, tile_counts + static_cast<int64_t>(blockIdx.x) * E, threadIdx.x,
                       [] { bar128(); });
  #pragma unroll
  for (int s = 0; s < ROUTE_MAX_K; ++s)
    if (s < k && e[s] >= 0) tile_rank[static_cast<int64_t>(t) * k + s] = rk[s];
}

// Per-tile histogram and tile-local rank from caller-supplied indices (entries outside [0,E) are skipped).
// Unlike the router's own top-k, a caller's list may name the same expert in several slots of one token, so the
// single bit per (expert, token) of tile_rank_and_counts is not enough here: one bit plane per SLOT.  Bit `row` of
// plane[s][e] is set iff entry (row, s) goes to expert e; the stable rank of entry (row, s) -- entries ordered by
// flat index t*k+s -- is the number of entries of e in lower rows (any slot) plus the number of lower slots of the
// same row that name e, and counts[e] is the number of ENTRIES, not of tokens.
__global__ void __launch_bounds__(ROUTE_TILE) tile_rank_kernel(const int32_t* __restrict__ topk_idx, int T, int E, int k,
                                                               int32_t* __restrict__ tile_rank,
                                                               int32_t* __restrict__ tile_counts) {
  pdl_wait_then_trigger();
  __shared__ uint32_t plane[ROUTE_MAX_K][ROUTE_MAX_E * 4];     // 32 KB
  for (int s = 0; s < k; ++s)
    for (int i = threadIdx.x; i < E * 4; i += ROUTE_TILE) plane[s][i] = 0u;
  const int row = threadIdx.x, t = blockIdx.x * ROUTE_TILE + row;
  int e[ROUTE_MAX_K];
  #pragma unroll
  for (int s = 0; s < ROUTE_MAX_K; ++s) {
    e[s] = -1;
    if (s < k && t < T) {
      const int v = __ldg(topk_idx + static_cast<int64_t>(t) * k + s);
      if (v >= 0 && v < E) e[s] = v;
    }
  }
  __syncthreads();
  #pragma unroll
  for (int s = 0; s < ROUTE_MAX_K; ++s)
    if (s < k && e[s] >= 0) atomicOr(&plane[s][e[s] * 4 + (row >> 5)], 1u << (row & 31));
  __syncthreads();
  const int w = row >> 5;
  const uint32_t below = (1u << (row & 31)) - 1u;
  #pragma unroll
  for (int s = 0; s < ROUTE_MAX_K; ++s)
    if (s < k && e[s] >= 0) {
      int r = 0;
      for (int s2 = 0; s2 < k; ++s2) {
        const uint32_t* m = plane[s2] + e[s] * 4;
        r += __popc(m[w] & below);
        #pragma unroll
        for (int j = 0; j < 3; ++j)
          if (j < w) r += __popc(m[j]);
      }
      #pragma unroll
      for (int s2 = 0; s2 < ROUTE_MAX_K; ++s2)
        if (s2 < s && e[s2] == e[s]) ++r;
      tile_rank[static_cast<int64_t>(t) * k + s] = r;
    }
  for (int x = threadIdx.x; x < E; x += ROUTE_TILE) {
    int c = 0;
    for (int s2 = 0; s2 < k; ++s2) {
      const uint32_t* m = plane[s2] + x * 4;
      c += __popc(m[0]) + __popc(m[1]) + __popc(m[2]) + __popc(m[3]);
    }
    tile_counts[static_cast<int64_t>(blockIdx.x) * E + x] = c;
  }
}

__global__ void __launch_bounds__(256) scan_kernel(const int32_t* __restrict__ tile_counts, int n_tiles, int E,
                                                   int32_t* __restrict__ tile_base, int32_t* __restrict__ counts,
                                                   int32_t* __restrict__ offsets) {
  pdl_wait_then_trigger();
  __shared__ int scratch[2 * 256 + 8];
  scan_tiles_block256(tile_counts, n_tiles, E, tile_base, counts, offsets, scratch);
}

}  // namespace

cudaError_t launch_topk_tile(const float* logits, int T, int E, int k, int32_t* topk_idx, float* topk_w,
                             int32_t* tile_rank, int32_t* tile_counts, cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  const int ne = (E + 31) / 32;
#define BG_TOPK(NE_) launch_pdl(topk_tile_kernel<NE_>, route_num_tiles(T), ROUTE_TILE, 0, st, logits, T, E, k, topk_idx, \
                                topk_w, tile_rank, tile_counts)
  switch (ne) {
    case 1: BG_TOPK(1); break;
    case 2: BG_TOPK(2); break;
    case 3: case 4: BG_TOPK(4); break;
    default: BG_TOPK(8); break;
  }
#undef BG_TOPK
  return cudaGetLastError();
}

cudaError_t launch_tile_rank(const int32_t* topk_idx, int T, int E, int k, int32_t* tile_rank, int32_t* tile_counts,
                             cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  launch_pdl(tile_rank_kernel, route_num_tiles(T), ROUTE_TILE, 0, st, topk_idx, T, E, k, tile_rank, tile_counts);
  return cudaGetLastError();
}

cudaError_t launch_scan(const int32_t* tile_counts, int n_tiles, int E, int32_t* tile_base, int32_t* counts,
                        int32_t* offsets, cudaStream_t st) {
  launch_pdl(scan_kernel, 1, 256, 0, st, tile_counts, n_tiles, E, tile_base, counts, offsets);
  return cudaGetLastError();
}

}  // namespace bg
