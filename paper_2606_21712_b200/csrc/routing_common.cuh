// routing_common.cuh -- device helpers shared by the fused router kernel (router_fused.cu) and the
// stand-alone routing kernels (routing.cu): the sortable key of reading S3, the tile-local stable rank
// (step a5, first half) and the scan over tiles and experts (step a4).
//
// Routing works on TILES of 128 consecutive tokens (the router GEMM's M tile).  For every tile the kernels
// produce counts[tile][e] and, for every (token, slot), its stable rank among the tile's entries of the same
// expert; a single scan over (tiles x experts) then gives base[tile][e] = offsets[e] + sum of the earlier
// tiles' counts, and row(t, s) = base[t/128][idx[t,s]] + rank(t, s).  That is the stable counting sort of
// DESIGN.md §1 (a3-a5) split so that only the scan needs all tiles.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bg {

constexpr int ROUTE_TILE = 128;      // tokens per routing tile
constexpr int ROUTE_MAX_E = 256;
constexpr int ROUTE_MAX_K = 8;

// (logit -> uint32) whose unsigned order is the logit order; -0.0 and +0.0 map to the same key (they tie).
// 0 is below every key a non-NaN logit can produce and serves as "no candidate".
__device__ __forceinline__ uint32_t float_to_ordered(float f) {
  f = f + 0.0f;                                    // canonicalise -0.0 to +0.0
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ordered_to_float(uint32_t o) {
  return __uint_as_float((o & 0x80000000u) ? (o ^ 0x80000000u) : ~o);
}

// Tile-local stable rank and histogram.  Called by the 128 threads that own the tile's token rows
// (row = 0..127) with the token's k selected experts in e[] (-1 = no entry: token past T or invalid index).
// mask: shared [E][4] words, zeroed by the caller before the barrier that precedes this call; bit `row` of
// mask[e] is set iff token `row` selected expert e (integer OR: independent of arrival order).  A token's k
// experts are distinct, so the stable rank of entry (row, s) among the tile's entries of expert e -- entries
// ordered by flat index -- is the number of lower rows that selected e.
// `sync128` is a barrier over exactly those 128 threads.
template <typename Sync>
__device__ __forceinline__ void tile_rank_and_counts(uint32_t* mask, int row, const int* e, int k, int E,
                                                     int32_t* rank_out /*[k] of this token, or nullptr*/,
                                                     int32_t* counts_out /*[E] of this tile*/, int tid128,
                                                     Sync sync128) {
  #pragma unroll
  for (int s = 0; s < ROUTE_MAX_K; ++s)
    if (s < k && e[s] >= 0) atomicOr(&mask[e[s] * 4 + (row >> 5)], 1u << (row & 31));
  sync128();
  const int w = row >> 5;
  const uint32_t below = (1u << (row & 31)) - 1u;
  #pragma unroll
  for (int s = 0; s < ROUTE_MAX_K; ++s)
    if (s < k && e[s] >= 0) {
      const uint32_t* m = mask + e[s] * 4;
      int r = __popc(m[w] & below);
      #pragma unroll
      for (int j = 0; j < 3; ++j)
        if (j < w) r += __popc(m[j]);
      rank_out[s] = r;
    }
  for (int x = tid128; x < E; x += ROUTE_TILE) {
    const uint32_t* m = mask + x * 4;
    counts_out[x] = __popc(m[0]) + __popc(m[1]) + __popc(m[2]) + __popc(m[3]);
  }
}

// Step a4 for all tiles, by ONE block of 256 threads:
//   counts[e] = sum_tiles tile_counts[tile][e];  offsets = exclusive scan over e, offsets[E] = total;
//   tile_base[tile][e] = offsets[e] + sum_{tile' < tile} tile_counts[tile'][e].
// scratch: shared, >= 2 * 256 + 8 ints.  counts / offsets may be nullptr.
__device__ __forceinline__ void scan_tiles_block256(const int32_t* tile_counts, int n_tiles, int E,
                                                    int32_t* tile_base, int32_t* counts, int32_t* offsets,
                                                    int* scratch) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int EW = 32;
  while (EW < E) EW <<= 1;                       // lanes per tile row (power of two, <= 256)
  const int G = 256 / EW;                        // tile groups
  const int g = tid / EW, e = tid - g * EW;
  const int per = (n_tiles + G - 1) / G;
  const int b0 = min(n_tiles, g * per), b1 = min(n_tiles, b0 + per);
  int* gsum = scratch;                           // [G][EW] = 256
  int* excl = scratch + 256;                     // [256]
  int* wtot = scratch + 512;                     // [8]
  int part = 0;
  if (e < E) {
    #pragma unroll 8
    for (int b = b0; b < b1; ++b) part += __ldcg(tile_counts + static_cast<int64_t>(b) * E + e);
  }
  gsum[tid] = part;
  __syncthreads();
  int total = 0;
  if (tid < EW)
    for (int gg = 0; gg < G; ++gg) total += gsum[gg * EW + tid];
  int v = total;                                 // threads >= EW (or e >= E) contribute 0
  #pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int u = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += u;
  }
  if (lane == 31) wtot[warp] = v;
  __syncthreads();
  int add = 0;
  for (int w = 0; w < warp; ++w) add += wtot[w];
  const int incl = v + add;
  excl[tid] = incl - total;
  if (tid < E) {
    if (counts) counts[tid] = total;
    if (offsets) {
      offsets[tid] = incl - total;
      if (tid == E - 1) offsets[E] = incl;
    }
  }
  __syncthreads();
  if (e < E) {
    int run = excl[e];
    for (int gg = 0; gg < g; ++gg) run += gsum[gg * EW + e];
    #pragma unroll 8
    for (int b = b0; b < b1; ++b) {
      const int64_t at = static_cast<int64_t>(b) * E + e;
      tile_base[at] = run;
      run += __ldcg(tile_counts + at);
    }
  }
}

}  // namespace bg
