// fp8_quant.cu -- quantisation kernels of the FP8 (e4m3) gate/up path (DESIGN.md §2 readings
// F1-F4; the paper's MoE GEMMs are FP8: PAPER.md:384, 442, 476-478).
//
//   F1  e4m3 ("fn": no infinities, max 448), round to nearest even, saturating    (__NV_SATFINITE, __NV_E4M3)
//   F2  activations: sx[r] = fl32(max_j |x[r,j]| / 448) (1 for a zero row); xq[r,j] = e4m3(fl32(x[r,j] / sx[r]))
//   F3  weights: sw[e,n] = fl32(max_k |W[e,k,n]| / 448) (1 for a zero channel); Wq[e,n,k] = e4m3(fl32(W[e,k,n] / sw[e,n])),
//       stored [E, N, K] (k contiguous) so that both GEMM operands are K-major
// The divisions are IEEE fp32 (__fdiv_rn): the precision in which the oracle takes the same decision, so the codes
// are compared bit for bit.
#include "kernels.h"
#include "ptx_sm100.cuh"
#include <cuda_bf16.h>
#include <cuda_fp8.h>

namespace bg {
namespace {

__device__ __forceinline__ uint8_t to_e4m3(float v) {
  return static_cast<uint8_t>(__nv_cvt_float_to_fp8(v, __NV_SATFINITE, __NV_E4M3));
}

// ---- weights: one block per (expert, 32 output channels); 256 threads = 32 channels x 8 k-lanes
__global__ void __launch_bounds__(256) quantize_weights_kernel(const __nv_bfloat16* __restrict__ W, int K, int N,
                                                               uint8_t* __restrict__ Wq, float* __restrict__ sw) {
  __shared__ float red[8][33];
  __shared__ float scale[32];
  __shared__ __align__(16) uint8_t tile[32][36];                        // [channel][k within a 32-row slab] (+4: bank spread)
  const int e = blockIdx.y, n0 = blockIdx.x * 32;
  const int cn = threadIdx.x & 31, kl = threadIdx.x >> 5; // channel within the block, k lane 0..7
  const int n = n0 + cn;
  const __nv_bfloat16* We = W + static_cast<int64_t>(e) * K * N;
  float amax = 0.0f;
  if (n < N)
    for (int k = kl; k < K; k += 8) amax = fmaxf(amax, fabsf(__bfloat162float(We[static_cast<int64_t>(k) * N + n])));
  red[kl][cn] = amax;
  __syncthreads();
  if (kl == 0) {
    float m = red[0][cn];
    #pragma unroll
    for (int i = 1; i < 8; ++i) m = fmaxf(m, red[i][cn]);
    const float s = m == 0.0f ? 1.0f : __fdiv_rn(m, 448.0f);
    scale[cn] = s;
    if (n < N) sw[static_cast<int64_t>(e) * N + n] = s;
  }
  __syncthreads();
  const float s = scale[cn];
  uint8_t* Wqe = Wq + static_cast<int64_t>(e) * N * K;
  for (int k0 = 0; k0 < K; k0 += 32) {
    // read 32 k-rows x 32 channels (channels contiguous in global), write 32 channels x 32 k (k contiguous)
    #pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int k = k0 + kl + 8 * i;
      uint8_t q = 0;
      if (n < N && k < K) q = to_e4m3(__fdiv_rn(__bfloat162float(We[static_cast<int64_t>(k) * N + n]), s));
      tile[cn][kl + 8 * i] = q;
    }
    __syncthreads();
    {
      const int c2 = threadIdx.x >> 3, k4 = (threadIdx.x & 7) * 4;      // 32 channels x 8 groups of 4 k
      const int nn = n0 + c2, kk = k0 + k4;
      if (nn < N && kk < K) {                                           // K is a multiple of 8 (bg_moe_create)
        const uint32_t v = *reinterpret_cast<const uint32_t*>(&tile[c2][k4]);
        *reinterpret_cast<uint32_t*>(Wqe + static_cast<int64_t>(nn) * K + kk) = v;
      }
    }
    __syncthreads();
  }
}

struct PermArgs {
  const int32_t* topk_idx;
  const int32_t* tile_rank;
  const int32_t* tile_base;
  const float* topk_w;
  int32_t* row_src;
  int32_t* inv_perm;
  float* w_perm;
  int E;
};

// ---- activations: the gather of gather_reduce.cu with the row quantised on the way.  One warp per token: the
// permutation entries of its k slots (as in gather_kernel), the row maximum (first pass over the row), then the
// e4m3 row written to the token's k expert-order rows (second pass; the row is 4-14 KB and stays in L1/L2).
template <int KMAX>
__global__ void __launch_bounds__(256) gather_fp8_kernel(const uint4* __restrict__ hidden, const PermArgs pa, int T, int k,
                                                         int vec_per_row, uint2* __restrict__ xq_perm,
                                                         float* __restrict__ sx_perm, unsigned* __restrict__ hmax,
                                                         const SegTable seg) {
  pdl_wait_then_trigger();
  const int lane = threadIdx.x & 31;
  const int warps_total = gridDim.x * (blockDim.x >> 5);
  for (int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); t < T; t += warps_total) {
    int r = -1;
    if (lane < k) {
      const int64_t i = static_cast<int64_t>(t) * k + lane;
      const int e = __ldg(pa.topk_idx + i);
      if (e >= 0 && e < pa.E) {
        r = __ldg(pa.tile_base + static_cast<int64_t>(t >> 7) * pa.E + e) + __ldg(pa.tile_rank + i);
        pa.inv_perm[i] = r;
        pa.row_src[r] = static_cast<int32_t>(i);
        if (pa.w_perm != nullptr) pa.w_perm[r] = __ldg(pa.topk_w + i);
      }
    }
    const uint4* src;
    if (seg.n > 0) {
      const int sg = seg_of(seg.start, seg.n, t);
      src = static_cast<const uint4*>(seg.hidden[sg]) + static_cast<int64_t>(t - __ldg(seg.start + sg)) * vec_per_row;
    } else {
      src = hidden + static_cast<int64_t>(t) * vec_per_row;
    }
    // pass 1: row maximum
    float amax = 0.0f;
    for (int c = lane; c < vec_per_row; c += 32) {
      const uint4 a = __ldg(src + c);
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&a);
      #pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float2 f = __bfloat1622float2(h[i]);
        amax = fmaxf(amax, fmaxf(fabsf(f.x), fabsf(f.y)));
      }
    }
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const float sx = amax == 0.0f ? 1.0f : __fdiv_rn(amax, 448.0f);
    uint2* dst[KMAX];
    bool ok[KMAX];
    #pragma unroll
    for (int s = 0; s < KMAX; ++s) {
      const int rs = __shfl_sync(0xffffffffu, r, s);
      ok[s] = s < k && rs >= 0;
      dst[s] = xq_perm + static_cast<int64_t>(ok[s] ? rs : 0) * vec_per_row;
      if (ok[s] && lane == 0) {
        sx_perm[rs] = sx;
        if (hmax != nullptr) hmax[rs] = 0u;
      }
    }
    // pass 2: quantise 8 values per vector -> 8 bytes
    for (int c = lane; c < vec_per_row; c += 32) {
      const uint4 a = __ldg(src + c);
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&a);
      uint32_t w[2] = {0u, 0u};
      #pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float2 f = __bfloat1622float2(h[i]);
        const uint32_t lo = to_e4m3(__fdiv_rn(f.x, sx)), hi = to_e4m3(__fdiv_rn(f.y, sx));
        w[i >> 1] |= (lo | (hi << 8)) << (16 * (i & 1));
      }
      #pragma unroll
      for (int s = 0; s < KMAX; ++s)
        if (ok[s]) dst[s][c] = make_uint2(w[0], w[1]);
    }
  }
}

// ---- H rows (reading F5): one warp per expert-order row
__global__ void __launch_bounds__(256) quantize_h_kernel(const uint4* __restrict__ H, const unsigned* __restrict__ hmax,
                                                         const float* __restrict__ w_perm, int64_t rows, int vec_per_row,
                                                         uint2* __restrict__ Hq, float* __restrict__ sh,
                                                         float* __restrict__ sc) {
  pdl_wait_then_trigger();
  const int lane = threadIdx.x & 31;
  const int64_t warps_total = static_cast<int64_t>(gridDim.x) * (blockDim.x >> 5);
  for (int64_t r = static_cast<int64_t>(blockIdx.x) * (blockDim.x >> 5) + (threadIdx.x >> 5); r < rows; r += warps_total) {
    const float amax = __uint_as_float(__ldg(hmax + r));
    const float s = amax == 0.0f ? 1.0f : __fdiv_rn(amax, 448.0f);
    if (lane == 0) {
      sh[r] = s;
      sc[r] = w_perm != nullptr ? s * __ldg(w_perm + r) : s;
    }
    const uint4* src = H + r * vec_per_row;
    uint2* dst = Hq + r * vec_per_row;
    for (int c = lane; c < vec_per_row; c += 32) {
      const uint4 a = __ldg(src + c);
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&a);
      uint32_t w[2] = {0u, 0u};
      #pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float2 f = __bfloat1622float2(h[i]);
        const uint32_t lo = to_e4m3(__fdiv_rn(f.x, s)), hi = to_e4m3(__fdiv_rn(f.y, s));
        w[i >> 1] |= (lo | (hi << 8)) << (16 * (i & 1));
      }
      dst[c] = make_uint2(w[0], w[1]);
    }
  }
}

}  // namespace

cudaError_t launch_quantize_h(const void* H, const unsigned* hmax, const float* w_perm, int64_t rows, int f, void* Hq,
                              float* sh, float* sc, int num_sms, cudaStream_t st) {
  if (rows == 0) return cudaSuccess;
  const int64_t blocks_needed = (rows + 7) / 8, cap = static_cast<int64_t>(num_sms) * 8;
  const int grid = static_cast<int>(blocks_needed < cap ? blocks_needed : cap);
  launch_pdl(quantize_h_kernel, grid, 256, 0, st, static_cast<const uint4*>(H), hmax, w_perm, rows, f / 8,
             static_cast<uint2*>(Hq), sh, sc);
  return cudaGetLastError();
}

cudaError_t launch_quantize_weights(const void* W, int E, int K, int N, void* Wq, float* sw, cudaStream_t st) {
  dim3 grid((N + 31) / 32, E);
  quantize_weights_kernel<<<grid, 256, 0, st>>>(static_cast<const __nv_bfloat16*>(W), K, N, static_cast<uint8_t*>(Wq), sw);
  return cudaGetLastError();
}

cudaError_t launch_gather_fp8(const void* hidden, const PermLaunch& pl, int T, int E, int k, int d, void* xq_perm,
                              float* sx_perm, unsigned* hmax, int num_sms, cudaStream_t st, const SegTable* segp) {
  const SegTable seg = segp ? *segp : SegTable{nullptr, nullptr, nullptr, 0};
  if (T == 0) return cudaSuccess;
  PermArgs pa;
  pa.topk_idx = pl.topk_idx; pa.tile_rank = pl.tile_rank; pa.tile_base = pl.tile_base; pa.topk_w = pl.topk_w;
  pa.row_src = pl.row_src; pa.inv_perm = pl.inv_perm; pa.w_perm = pl.w_perm; pa.E = E;
  const int blocks_needed = (T + 7) / 8, cap = num_sms * 8;
  const int grid = blocks_needed < cap ? blocks_needed : cap;
  if (k <= 2)
    launch_pdl(gather_fp8_kernel<2>, grid, 256, 0, st, static_cast<const uint4*>(hidden), pa, T, k, d / 8,
               static_cast<uint2*>(xq_perm), sx_perm, hmax, seg);
  else if (k <= 4)
    launch_pdl(gather_fp8_kernel<4>, grid, 256, 0, st, static_cast<const uint4*>(hidden), pa, T, k, d / 8,
               static_cast<uint2*>(xq_perm), sx_perm, hmax, seg);
  else
    launch_pdl(gather_fp8_kernel<8>, grid, 256, 0, st, static_cast<const uint4*>(hidden), pa, T, k, d / 8,
               static_cast<uint2*>(xq_perm), sx_perm, hmax, seg);
  return cudaGetLastError();
}

}  // namespace bg
