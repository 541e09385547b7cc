// route_noalloc.cu -- bg_moe_route_logits_noalloc: routing steps a2-a4 (top-k + gates, per-expert histogram,
// exclusive scan) from given fp32 logits, for callers that must not allocate device memory.
//
// Who that is.  Every other routing call of this library needs a bg_moe_ctx, and bg_moe_create cudaMallocs the
// context's workspace.  Two kinds of caller cannot do that:
//   * a serving runtime that has already handed the whole of HBM to pools it manages itself -- the paper's runtime
//     is one: KV cache plus the ring parameter buffer are sized to fill the device (§5.2) --
//     so a cudaMalloc from a library it loads would simply fail, or take memory its planner counted on;
//   * code on a latency-critical path (a scheduler tick between two module launches) where cudaMalloc / cudaFree
//     are off limits because they serialise with everything in flight on the device.
// For them the per-tile histograms and the tile ticket -- the only global memory this kernel needs beyond its
// inputs and outputs -- live in a fixed array that is part of the library image (g_scratch below).  Its size fixes
// the largest call: BG_MOE_NOALLOC_MAX_TOKENS tokens, E <= 256.  Every GPU on which the library's module is loaded
// holds its own copy of the array (128 KiB + 256 B = 131,328 bytes) until the process exits.
//
// This file is self-contained on purpose: the array, the one place that asks the runtime for its device address and
// the kernel that uses it must be in ONE translation unit (the array has internal linkage), and nothing here touches
// a bg_moe_ctx, the workspace code in api.cu or the kernels of routing.cu.  The arithmetic is that of
// routing.cu:topk_tile_kernel (same key order -- reading S3 -- same expf / division), so the results carry the same
// bits as bg_moe_route(logits_in = ...).
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <mutex>
#include "../../include/bg_moe.h"
#include "routing_common.cuh"

namespace {

constexpr int NA_MAX_TILES = BG_MOE_NOALLOC_MAX_TOKENS / bg::ROUTE_TILE;        // 128 tiles of 128 tokens
constexpr size_t NA_TICKET_BYTES = 256;                                         // one int, on a line of its own
constexpr size_t NA_COUNTS_BYTES = sizeof(int32_t) * NA_MAX_TILES * bg::ROUTE_MAX_E;
constexpr size_t NA_SCRATCH_BYTES = NA_TICKET_BYTES + NA_COUNTS_BYTES;          // 131,328 bytes
static_assert(BG_MOE_NOALLOC_MAX_TOKENS % bg::ROUTE_TILE == 0, "whole tiles");
constexpr int NA_MAX_DEVICES = 64;

// The scratch itself.  In HOST code this name is only a handle for the runtime's symbol calls -- it is not a
// device address and must never be handed to a kernel as a pointer (a kernel given &g_scratch[0] taken on the
// host faults, or on a machine where the GPU can reach host memory quietly scribbles over the wrong bytes).
// Host code gets the real address from cudaGetSymbolAddress (scratch_for_current_device).
//   [0, 256)      ticket: number of tiles that have published their histogram in the running call
//   [256, ...)    tile_counts int32 [n_tiles][E] of the running call
static __device__ __align__(256) unsigned char g_scratch[NA_SCRATCH_BYTES];

std::mutex g_mu;
void* g_scratch_addr[NA_MAX_DEVICES] = {};      // per device ordinal: device address of that GPU's copy
thread_local char g_err[256] = "";

int fail(int status, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess)
    snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
  else
    snprintf(g_err, sizeof g_err, "%s", what);
  return status;
}

// Set-up, once per device, with that device current: the address of THIS device's copy of g_scratch.
// cudaGetSymbolAddress may load the library's module onto the device the first time (the runtime's own work, not
// something to do in the middle of a stream capture); afterwards the address comes from the table.
int scratch_for_current_device(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(BG_ERR_CUDA, "cudaGetDevice", e);
  if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(BG_ERR_UNSUPPORTED, "device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_mu);
  if (g_scratch_addr[dev] == nullptr) {
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail(BG_ERR_CUDA, "cudaDeviceGetAttribute", e);
    if (major != 10) return fail(BG_ERR_UNSUPPORTED, "device is not sm_100 (there is no CPU fallback)");
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_scratch);
    if (e != cudaSuccess || p == nullptr) return fail(BG_ERR_CUDA, "cudaGetSymbolAddress(g_scratch)", e);
    g_scratch_addr[dev] = p;
  }
  *out = static_cast<unsigned char*>(g_scratch_addr[dev]);
  return BG_OK;
}

// One block of 128 threads per 128-token tile (grid = max(1, number of tiles)).
//   phase 1  top-k + gates per token, one warp per token, 64-bit (ordered logit, ~expert) keys: as topk_tile_kernel
//   phase 2  the tile's histogram (shared integer atomics: order-independent) -> scratch tile_counts[tile][.]
//   phase 3  the tile takes a ticket; the tile that draws the last one sums the histograms over tiles in tile
//            order, scans over experts, writes counts / offsets, and puts the ticket back to zero
// `scratch` is the DEVICE address of g_scratch (device code could also name g_scratch directly; taking it as an
// argument keeps the kernel honest about what it touches).
template <int NE>
__global__ void __launch_bounds__(bg::ROUTE_TILE)
route_logits_noalloc_kernel(const float* __restrict__ logits, int T, int E, int k, int32_t* __restrict__ topk_idx,
                            float* __restrict__ topk_w, int32_t* __restrict__ counts, int32_t* __restrict__ offsets,
                            unsigned char* __restrict__ scratch) {
  using namespace bg;
  __shared__ int hist[ROUTE_MAX_E];
  __shared__ int wsum[4], wsum1[4];
  __shared__ int is_last;
  int* ticket = reinterpret_cast<int*>(scratch);
  int32_t* tile_counts = reinterpret_cast<int32_t*>(scratch + NA_TICKET_BYTES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_tiles = gridDim.x;
  for (int i = threadIdx.x; i < ROUTE_MAX_E; i += ROUTE_TILE) hist[i] = 0;
  __syncthreads();

  for (int row = warp; row < ROUTE_TILE; row += 4) {
    const int t = blockIdx.x * ROUTE_TILE + row;
    if (t >= T) break;                                  // rows of a warp ascend: nothing further in this tile
    unsigned long long key[NE];
    #pragma unroll
    for (int j = 0; j < NE; ++j) {
      const int e = lane + 32 * j;
      key[j] = 0ull;                                    // "no candidate": below every real key
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
        if (key[j] == best) key[j] = 0ull;              // taken
      const float val = ordered_to_float(static_cast<uint32_t>(best >> 32));
      if (s == 0) v_max = val;
      if (lane == s) { my_e = static_cast<int>(0xFFFFFFFFu - static_cast<uint32_t>(best)); my_v = val; }
    }
    const float ex = (lane < k) ? expf(my_v - v_max) : 0.0f;
    float denom = 0.0f;
    for (int s = 0; s < k; ++s) denom += __shfl_sync(0xffffffffu, ex, s);      // slot order
    if (lane < k) {
      topk_idx[static_cast<int64_t>(t) * k + lane] = my_e;
      topk_w[static_cast<int64_t>(t) * k + lane] = ex / denom;
      atomicAdd(&hist[my_e], 1);
    }
  }
  __syncthreads();

  // publish this tile's histogram, then take a ticket
  for (int e = threadIdx.x; e < E; e += ROUTE_TILE) tile_counts[static_cast<int64_t>(blockIdx.x) * E + e] = hist[e];
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = (atomicAdd(ticket, 1) == n_tiles - 1);
  __syncthreads();
  if (!is_last) return;
  __threadfence();

  // the last tile: counts over tiles (thread x owns experts x and x + 128), exclusive scan over experts
  int c0 = 0, c1 = 0;
  const int e0 = threadIdx.x, e1 = threadIdx.x + ROUTE_TILE;
  for (int b = 0; b < n_tiles; ++b) {
    if (e0 < E) c0 += __ldcg(tile_counts + static_cast<int64_t>(b) * E + e0);
    if (e1 < E) c1 += __ldcg(tile_counts + static_cast<int64_t>(b) * E + e1);
  }
  // inclusive scan of c0 over the 128 threads; the c1 half follows after the total of the c0 half
  int v0 = c0, v1 = c1;
  #pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int u0 = __shfl_up_sync(0xffffffffu, v0, o), u1 = __shfl_up_sync(0xffffffffu, v1, o);
    if (lane >= o) { v0 += u0; v1 += u1; }
  }
  if (lane == 31) { wsum[warp] = v0; wsum1[warp] = v1; }
  __syncthreads();
  int add0 = 0, add1 = 0, total0 = 0;
  for (int w = 0; w < 4; ++w) {
    if (w < warp) { add0 += wsum[w]; add1 += wsum1[w]; }
    total0 += wsum[w];
  }
  const int incl0 = v0 + add0, incl1 = total0 + v1 + add1;
  if (e0 < E) {
    counts[e0] = c0;
    offsets[e0] = incl0 - c0;
    if (e0 == E - 1) offsets[E] = incl0;
  }
  if (e1 < E) {
    counts[e1] = c1;
    offsets[e1] = incl1 - c1;
    if (e1 == E - 1) offsets[E] = incl1;
  }
  if (threadIdx.x == 0) *ticket = 0;                    // the next call starts from zero
}

}  // namespace

extern "C" int bg_moe_route_logits_noalloc(const float* logits, int32_t T, int32_t E, int32_t k, int32_t* topk_idx,
                                           float* topk_w, int32_t* counts, int32_t* offsets, void* stream) {
  g_err[0] = '\0';
  if (T < 0 || E < 1 || k < 1 || k > E) return fail(BG_ERR_INVALID_ARG, "need T >= 0, E >= 1, 1 <= k <= E");
  if (E > bg::ROUTE_MAX_E || k > bg::ROUTE_MAX_K) return fail(BG_ERR_UNSUPPORTED, "E > 256 or k > 8");
  if (T > BG_MOE_NOALLOC_MAX_TOKENS) {
    snprintf(g_err, sizeof g_err,
             "T = %d exceeds BG_MOE_NOALLOC_MAX_TOKENS = %d: the fixed scratch array holds the histograms of at most "
             "%d tiles; split the batch or use bg_moe_route with a context",
             T, BG_MOE_NOALLOC_MAX_TOKENS, NA_MAX_TILES);
    return BG_ERR_INVALID_ARG;
  }
  if (!counts || !offsets) return fail(BG_ERR_INVALID_ARG, "counts / offsets is NULL");
  if (T > 0 && (!logits || !topk_idx || !topk_w)) return fail(BG_ERR_INVALID_ARG, "logits / topk_idx / topk_w is NULL");
  unsigned char* scratch = nullptr;
  int rc = scratch_for_current_device(&scratch);
  if (rc != BG_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // The array is shared by every call and keeps what the last one left.  The histograms are fully rewritten for
  // the tiles of this call before anything reads them; the ticket is the one word that must start at zero.  The
  // kernel re-arms it, and it is cleared here as well so that a call cut short (a failed launch, a faulted
  // predecessor) cannot leave a count behind for the next one.
  cudaError_t e = cudaMemsetAsync(scratch, 0, NA_TICKET_BYTES, st);
  if (e != cudaSuccess) return fail(BG_ERR_CUDA, "cudaMemsetAsync(ticket)", e);
  const int grid = T > 0 ? (T + bg::ROUTE_TILE - 1) / bg::ROUTE_TILE : 1;
  const int ne = (E + 31) / 32;
#define BG_NA_LAUNCH(NE_) \
  route_logits_noalloc_kernel<NE_><<<grid, bg::ROUTE_TILE, 0, st>>>(logits, T, E, k, topk_idx, topk_w, counts, offsets, scratch)
  switch (ne) {
    case 1: BG_NA_LAUNCH(1); break;
    case 2: BG_NA_LAUNCH(2); break;
    case 3: case 4: BG_NA_LAUNCH(4); break;
    default: BG_NA_LAUNCH(8); break;
  }
#undef BG_NA_LAUNCH
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(BG_ERR_CUDA, "launch route_logits_noalloc_kernel", e);
  return BG_OK;
}

extern "C" const char* bg_moe_noalloc_last_error(void) { return g_err; }
