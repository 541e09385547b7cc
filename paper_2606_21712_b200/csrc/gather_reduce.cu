// gather_reduce.cu -- the two HBM-bound row movers of the combined MoE layer:
//   a5'' + a6    row r of entry i = t*k+s from the tile bases and tile-local ranks (inv_perm, row_src, w_perm),
//                x_perm[r,:] = hidden[row_src[r]/k,:]   written as x_perm[inv_perm[i],:] = hidden[i/k,:]
//   a9 reduce    out[t,:]    = sum_{s<k} (w[t,s]) * Y[inv_perm[t*k+s],:]     slot order, fp32, RNE->bf16
// BASELINE.json north_star: "a gather kernel with 16-byte vectorised, coalesced row copies" and "a
// gate-weighted un-permute that sums each token's top-k results", atomic-free.
// One warp moves one row at a time; consecutive lanes touch consecutive 16-byte vectors, several
// vectors in flight per lane.  Grid = a multiple of the SM count, warps stride over rows.
#include "kernels.h"
#include "ptx_sm100.cuh"
#include <cuda_bf16.h>

namespace bg {
namespace {

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(uint4* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w) : "memory");
}

// a5 (second half) + a6 as a scatter: one warp per TOKEN.  Lane s < k finishes the permutation of entry
// i = t*k + s -- row r = tile_base[t/128][idx] + tile_rank[i] (routing_common.cuh), inv_perm[i] = r,
// row_src[r] = i, w_perm[r] = topk_w[i] -- then the warp reads the token's hidden row once (registers) and writes
// it to its k expert-order rows: x_perm[inv_perm[t*k+s]] = hidden[t] is the same assignment as
// x_perm[r] = hidden[row_src[r]/k], with 1 load + k stores per vector instead of k loads + k stores.
struct PermArgs {
  const int32_t* topk_idx;    // [T,k]
  const int32_t* tile_rank;   // [T,k]
  const int32_t* tile_base;   // [n_tiles,E]
  const float* topk_w;        // [T,k] or nullptr
  int32_t* row_src;           // [T*k]
  int32_t* inv_perm;          // [T*k]
  float* w_perm;              // [T*k] or nullptr
  int E;
};

template <int KMAX>
__global__ void __launch_bounds__(256) gather_kernel(const uint4* __restrict__ hidden, const PermArgs pa, int T, int k,
                                                     int vec_per_row, uint4* __restrict__ x_perm, const SegTable seg,
                                                     int parts) {
  pdl_wait_then_trigger();
  const int lane = threadIdx.x & 31;
  const int warps_total = gridDim.x * (blockDim.x >> 5);
  // `parts` warps share a token (a power of two; > 1 at small T, where one warp per token leaves the SMs a few dozen
  // warps each and the kernel latency-bound): warp unit u moves columns [part, part + 1) * vec_per_row / parts of token
  // u / parts; part 0 also records the permutation.
  const int units = T * parts;
  const int span = (vec_per_row + parts - 1) / parts;
  for (int u = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); u < units; u += warps_total) {
    const int t = u / parts, part = u - t * parts;
    const int c_begin = part * span, c_end = min(vec_per_row, c_begin + span);
    int r = -1;
    if (lane < k) {
      const int64_t i = static_cast<int64_t>(t) * k + lane;
      const int e = __ldg(pa.topk_idx + i);
      if (e >= 0 && e < pa.E) {
        r = __ldg(pa.tile_base + static_cast<int64_t>(t >> 7) * pa.E + e) + __ldg(pa.tile_rank + i);
        if (part == 0) {
          pa.inv_perm[i] = r;
          pa.row_src[r] = static_cast<int32_t>(i);
          if (pa.w_perm != nullptr) pa.w_perm[r] = __ldg(pa.topk_w + i);
        }
      }
    }
    if (x_perm == nullptr) continue;
    const uint4* src;
    if (seg.n > 0) {               // zero-copy COMBINE: the token's row inside its coroutine's own buffer
      const int sg = seg_of(seg.start, seg.n, t);
      src = static_cast<const uint4*>(seg.hidden[sg]) + static_cast<int64_t>(t - __ldg(seg.start + sg)) * vec_per_row;
    } else {
      src = hidden + static_cast<int64_t>(t) * vec_per_row;
    }
    uint4* dst[KMAX];
    bool ok[KMAX];
    #pragma unroll
    for (int s = 0; s < KMAX; ++s) {
      const int rs = __shfl_sync(0xffffffffu, r, s);
      ok[s] = s < k && rs >= 0;
      dst[s] = x_perm + static_cast<int64_t>(ok[s] ? rs : 0) * vec_per_row;
    }
    int c = c_begin + lane;
    for (; c + 96 < c_end; c += 128) {
      const uint4 a0 = ld_stream(src + c), a1 = ld_stream(src + c + 32), a2 = ld_stream(src + c + 64),
                  a3 = ld_stream(src + c + 96);
      #pragma unroll
      for (int s = 0; s < KMAX; ++s)
        if (ok[s]) {
          st_stream(dst[s] + c, a0);
          st_stream(dst[s] + c + 32, a1);
          st_stream(dst[s] + c + 64, a2);
          st_stream(dst[s] + c + 96, a3);
        }
    }
    for (; c < c_end; c += 32) {
      const uint4 a = ld_stream(src + c);
      #pragma unroll
      for (int s = 0; s < KMAX; ++s)
        if (ok[s]) st_stream(dst[s] + c, a);
    }
  }
}

__device__ __forceinline__ void accum8(float* acc, const uint4& v, float w) {
  const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v);
  #pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float2 f = __bfloat1622float2(h[i]);
    acc[2 * i] = fmaf(w, f.x, acc[2 * i]);
    acc[2 * i + 1] = fmaf(w, f.y, acc[2 * i + 1]);
  }
}

template <int KMAX>
__global__ void __launch_bounds__(256) unpermute_kernel(const uint4* __restrict__ y_perm,
                                                        const int32_t* __restrict__ inv_perm,
                                                        const float* __restrict__ weights, int T, int k,
                                                        int vec_per_row, uint4* __restrict__ out, const SegTable seg,
                                                        int parts) {
  pdl_wait_then_trigger();
  const int lane = threadIdx.x & 31;
  const int warps_total = gridDim.x * (blockDim.x >> 5);
  const int units = T * parts;                 // `parts` warps share a token, each a column range (see gather_kernel)
  const int span = (vec_per_row + parts - 1) / parts;
  for (int u = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); u < units; u += warps_total) {
    const int t = u / parts, part = u - t * parts;
    const int c_begin = part * span, c_end = min(vec_per_row, c_begin + span);
    const uint4* rows[KMAX];
    float w[KMAX];
    #pragma unroll
    for (int s = 0; s < KMAX; ++s) {
      rows[s] = y_perm;
      w[s] = 0.0f;
      if (s < k) {
        rows[s] = y_perm + static_cast<int64_t>(__ldg(inv_perm + static_cast<int64_t>(t) * k + s)) * vec_per_row;
        w[s] = weights ? __ldg(weights + static_cast<int64_t>(t) * k + s) : 1.0f;
      }
    }
    uint4* dst;
    if (seg.n > 0) {               // zero-copy split: the result goes back to the token's coroutine
      const int sg = seg_of(seg.start, seg.n, t);
      dst = static_cast<uint4*>(seg.out[sg]) + static_cast<int64_t>(t - __ldg(seg.start + sg)) * vec_per_row;
    } else {
      dst = out + static_cast<int64_t>(t) * vec_per_row;
    }
    for (int c = c_begin + lane; c < c_end; c += 32) {
      uint4 v[KMAX];
      #pragma unroll
      for (int s = 0; s < KMAX; ++s)
        if (s < k) v[s] = ld_stream(rows[s] + c);
      float acc[8];
      #pragma unroll
      for (int i = 0; i < 8; ++i) acc[i] = 0.0f;
      #pragma unroll
      for (int s = 0; s < KMAX; ++s)       // slot order s = 0..k-1 (reading S11)
        if (s < k) accum8(acc, v[s], w[s]);
      uint4 o;
      __nv_bfloat162 p;
      p = __floats2bfloat162_rn(acc[0], acc[1]); o.x = *reinterpret_cast<uint32_t*>(&p);
      p = __floats2bfloat162_rn(acc[2], acc[3]); o.y = *reinterpret_cast<uint32_t*>(&p);
      p = __floats2bfloat162_rn(acc[4], acc[5]); o.z = *reinterpret_cast<uint32_t*>(&p);
      p = __floats2bfloat162_rn(acc[6], acc[7]); o.w = *reinterpret_cast<uint32_t*>(&p);
      st_stream(dst + c, o);
    }
  }
}

// Warps per token: enough warps for ~48 per SM, each keeping at least one warp-wide pass of 16-byte vectors.
inline int row_mover_parts(int T, int vec_per_row, int num_sms) {
  int parts = 1;
  while (parts < 8 && static_cast<int64_t>(T) * parts < 48ll * num_sms && vec_per_row / (2 * parts) >= 32) parts *= 2;
  return parts;
}

inline int row_mover_grid(int rows, int num_sms) {
  const int blocks_needed = (rows + 7) / 8;
  const int cap = num_sms * 8;     // 8 resident blocks of 256 threads per SM
  return blocks_needed < cap ? (blocks_needed > 0 ? blocks_needed : 1) : cap;
}

}  // namespace

cudaError_t launch_gather(const void* hidden, const PermLaunch& pl, int T, int E, int k, int d, void* x_perm,
                          int num_sms, cudaStream_t st, const SegTable* segp) {
  const SegTable seg = segp ? *segp : SegTable{nullptr, nullptr, nullptr, 0};
  if (T == 0) return cudaSuccess;
  PermArgs pa;
  pa.topk_idx = pl.topk_idx; pa.tile_rank = pl.tile_rank; pa.tile_base = pl.tile_base; pa.topk_w = pl.topk_w;
  pa.row_src = pl.row_src; pa.inv_perm = pl.inv_perm; pa.w_perm = pl.w_perm; pa.E = E;
  const int parts = row_mover_parts(T, d / 8, num_sms);
  const int grid = row_mover_grid(T * parts, num_sms);
  if (k <= 2)
    launch_pdl(gather_kernel<2>, grid, 256, 0, st, static_cast<const uint4*>(hidden), pa, T, k, d / 8,
                                           static_cast<uint4*>(x_perm), seg, parts);
  else if (k <= 4)
    launch_pdl(gather_kernel<4>, grid, 256, 0, st, static_cast<const uint4*>(hidden), pa, T, k, d / 8,
                                           static_cast<uint4*>(x_perm), seg, parts);
  else
    launch_pdl(gather_kernel<8>, grid, 256, 0, st, static_cast<const uint4*>(hidden), pa, T, k, d / 8,
                                           static_cast<uint4*>(x_perm), seg, parts);
  return cudaGetLastError();
}

cudaError_t launch_unpermute(const void* y_perm, const int32_t* inv_perm, const float* weights, int T, int k,
                             int d, void* out, int num_sms, cudaStream_t st, const SegTable* segp) {
  const SegTable seg = segp ? *segp : SegTable{nullptr, nullptr, nullptr, 0};
  if (T == 0) return cudaSuccess;
  const int parts = row_mover_parts(T, d / 8, num_sms);
  const int grid = row_mover_grid(T * parts, num_sms);
  if (k <= 2)
    launch_pdl(unpermute_kernel<2>, grid, 256, 0, st, static_cast<const uint4*>(y_perm), inv_perm, weights, T, k, d / 8,
                                              static_cast<uint4*>(out), seg, parts);
  else if (k <= 4)
    launch_pdl(unpermute_kernel<4>, grid, 256, 0, st, static_cast<const uint4*>(y_perm), inv_perm, weights, T, k, d / 8,
                                              static_cast<uint4*>(out), seg, parts);
  else
    launch_pdl(unpermute_kernel<8>, grid, 256, 0, st, static_cast<const uint4*>(y_perm), inv_perm, weights, T, k, d / 8,
                                              static_cast<uint4*>(out), seg, parts);
  return cudaGetLastError();
}

}  // namespace bg
