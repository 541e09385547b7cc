// grouped_gemm.cu -- steps a7 / a8 of the combined MoE layer on sm_100a tensor cores.
//
//   a7: H[r,:] = silu(x_perm[r,:] W_gate[e]) (.) (x_perm[r,:] W_up[e])      rows r of expert e
//   a8: Y[r,:] = (w[row_src[r]]) * (H[r,:] W_down[e])
// (BASELINE.json north_star "grouped SwiGLU expert FFN".)
//
// One persistent kernel template serves both GEMMs: a 128 x 256 fp32 accumulator tile in TMEM,
// tcgen05.mma (kind::f16, M=128, N=256, K=16) issued by one thread, operands staged by TMA into
// 128B-swizzled shared memory through a 4-stage mbarrier ring, two TMEM accumulator stages so the
// epilogue of tile i overlaps the main loop of tile i+1.
//   A operand: activations [rows, K] bf16, K contiguous  -> K-major,  TMA box {64 k, 128 rows}
//   B operand: weights [E, K, N] bf16, N contiguous      -> MN-major, TMA boxes {64 n, 64 k, 1}
// The weights are consumed in the layout the layer is given (reading S14): no transpose/prepack.
// For a7 the 256 accumulator columns are [gate n0..n0+128 | up n0..n0+128] so that SiLU(g)*u is
// an epilogue over one thread's registers; for a8 they are 256 consecutive output columns.
//
// Tile scheduler: M-tiles never straddle experts.  Expert e owns ceil(n_e/128) M-tiles; its tiles
// are ordered n-tile-major / m-tile-minor so that the CTAs running at the same time share one
// weight strip through L2.  Tile t -> CTA (t mod gridDim.x).  Experts with no rows own no tiles
// and their weights are never touched.  Rows past the end of an expert inside a tile are computed
// (they belong to the next expert or are TMA zero fill) but never stored.
#include "kernels.h"
#include "ptx_sm100.cuh"

namespace bg {
namespace {

constexpr int BM = 128;            // rows per tile (UMMA M)
constexpr int BN = 256;            // accumulator columns per tile (UMMA N)
constexpr int BK = 64;             // k per pipeline stage = one 128-byte swizzle span of bf16
constexpr int UK = 16;             // UMMA K for 16-bit inputs
constexpr int STAGES = 4;
constexpr int A_BYTES = BM * BK * 2;          // 16 KB
constexpr int B_BLK_BYTES = 64 * BK * 2;      // 8 KB: one 64-column block of B
constexpr int B_BYTES = (BN / 64) * B_BLK_BYTES;   // 32 KB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;     // 48 KB
constexpr int NUM_THREADS = 256;   // warp 0 TMA, warp 1 MMA, warp 2 TMEM alloc, warps 4-7 epilogue
constexpr int MAX_E = 256;
// Epilogue staging: each epilogue warp transposes 32 rows x 64 bf16 columns through its own
// padded shared-memory buffer (row pitch 144 B: conflict-free 16-byte accesses) so that global
// stores are whole 128-byte lines instead of 32 scattered 16-byte pieces.
constexpr int EPI_PITCH = 144;
constexpr int EPI_WARP_BYTES = 32 * EPI_PITCH;               // 4608 B
constexpr int TABLE_BYTES = 2064;                            // 2 x (MAX_E + 1) ints, 16-byte padded
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/ + TABLE_BYTES +
                           4 * EPI_WARP_BYTES;

constexpr uint32_t IDESC = umma_idesc_bf16(BM, BN, /*A K-major*/ 0, /*B MN-major*/ 1);
// A: K-major SW128: 8-row groups 1024 B apart (SBO); LBO unused inside one swizzle span.
constexpr uint64_t ADESC_HI = umma_desc_sw128(16, 1024);
// B: MN-major SW128: 64-column blocks B_BLK_BYTES apart (LBO); 8-k-row groups 1024 B apart (SBO).
constexpr uint64_t BDESC_HI = umma_desc_sw128(B_BLK_BYTES, 1024);

struct Params {
  const int32_t* offsets;
  int E, K, N;
  __nv_bfloat16* out;
  const float* row_scale;
  const int32_t* row_src;
  bool w4d;                    // tm_b0 / tm_b1 are the 4-D block views (kernels.h)
};

struct TileCoord {
  int e, row0, rows_valid, n_tile;
};

// tile_start[e] = first linear tile index of expert e (tile_start[E] = total);
// m_tiles[e] = M-tiles of expert e.  Both live in shared memory.
__device__ __forceinline__ TileCoord decode_tile(int t, const int* tile_start, const int* m_tiles,
                                                 const int32_t* offsets, int E) {
  int lo = 0, hi = E;              // largest e with tile_start[e] <= t
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (tile_start[mid] <= t) lo = mid; else hi = mid;
  }
  // experts with zero tiles share tile_start with their successor: the search above lands on the
  // last expert whose start <= t, which is the one that owns t (its successors start later).
  const int e = lo;
  const int local = t - tile_start[e];
  const int mt = m_tiles[e];
  const int n_tile = local / mt;
  const int m_tile = local - n_tile * mt;
  const int beg = __ldg(offsets + e), end = __ldg(offsets + e + 1);
  TileCoord c;
  c.e = e;
  c.row0 = beg + m_tile * BM;
  c.rows_valid = min(BM, end - c.row0);
  c.n_tile = n_tile;
  return c;
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

__device__ __forceinline__ float silu_mul(float g, float u) {
  return __fdividef(g, 1.0f + __expf(-g)) * u;
}

// GATEUP = true : a7 (B = [W_gate strip | W_up strip], SwiGLU epilogue, 128 output columns / tile)
// GATEUP = false: a8 (B = W_down strip, optional row scale, 256 output columns / tile)
template <bool GATEUP>
__global__ void __launch_bounds__(NUM_THREADS, 1)
grouped_gemm_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_b0,
                    const __grid_constant__ CUtensorMap tm_b1, const Params p) {
  constexpr int OUT_COLS = GATEUP ? BN / 2 : BN;     // output columns per tile
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;       // SW128 tiles need 1024-byte alignment
  uint8_t* smem = smem_raw + (base - raw);
  const uint32_t bar_base = base + STAGES * STAGE_BYTES;
  // barriers: full[0..S), empty[0..S), tmem_full[0..2), tmem_empty[0..2); then the TMEM address
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + STAGES * STAGE_BYTES + 8 * (2 * STAGES + 4));
  int* tile_start = reinterpret_cast<int*>(smem + STAGES * STAGE_BYTES + 256);
  int* m_tiles = tile_start + (MAX_E + 1);
  uint8_t* epi_smem = smem + STAGES * STAGE_BYTES + 256 + TABLE_BYTES;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int E = p.E;
  const int n_tiles = (p.N + OUT_COLS - 1) / OUT_COLS;
  const int k_blocks = (p.K + BK - 1) / BK;

  pdl_wait_then_trigger();
  // ---- per-CTA tile table: inclusive scan of per-expert tile counts (E <= 256 = blockDim)
  {
    int mt = 0;
    if (threadIdx.x < E) {
      const int cnt = __ldg(p.offsets + threadIdx.x + 1) - __ldg(p.offsets + threadIdx.x);
      mt = (cnt + BM - 1) / BM;
      m_tiles[threadIdx.x] = mt;
    }
    int v = mt * n_tiles;
    // warp inclusive scan, then scan of warp totals
    #pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v += u;
    }
    __shared__ int warp_tot[NUM_THREADS / 32];
    if (lane == 31) warp_tot[warp] = v;
    __syncthreads();
    int add = 0;
    for (int w = 0; w < warp; ++w) add += warp_tot[w];
    v += add;                                   // inclusive prefix for thread's expert
    if (threadIdx.x < E) tile_start[threadIdx.x + 1] = v;
    if (threadIdx.x == 0) tile_start[0] = 0;
  }

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_a);
    tma_prefetch_desc(&tm_b0);
    if (GATEUP) tma_prefetch_desc(&tm_b1);
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull_bar(a), 1);
      mbar_init(tempty_bar(a), 128);
    }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc(smem_u32(tmem_slot), 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int total_tiles = tile_start[E];

  if (warp == 0) {
    // ===================== TMA producer (one thread) =====================
    // (A tile::gather4 load of the rows straight from `hidden` was measured and rejected: 32 gather4
    //  operations per k-block cost ~40 ns each and made this kernel 3.4x slower.)
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
        const TileCoord c = decode_tile(t, tile_start, m_tiles, p.offsets, E);
        const int n0 = c.n_tile * OUT_COLS;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(empty_bar(s), ph ^ 1u);
          const uint32_t sa = base + s * STAGE_BYTES;
          const uint32_t sb = sa + A_BYTES;
          mbar_expect_tx(full_bar(s), STAGE_BYTES);
          tma_load_2d(sa, &tm_a, full_bar(s), kb * BK, c.row0);
          if (p.w4d) {
            // one operation per weight tensor: 64-column blocks in [block][k][64 n] order (kernels.h)
            if (GATEUP) {
              tma_load_4d(sb, &tm_b0, full_bar(s), 0, kb * BK, n0 >> 6, c.e);
              tma_load_4d(sb + 2 * B_BLK_BYTES, &tm_b1, full_bar(s), 0, kb * BK, n0 >> 6, c.e);
            } else {
              tma_load_4d(sb, &tm_b0, full_bar(s), 0, kb * BK, n0 >> 6, c.e);
            }
          } else if (GATEUP) {
            tma_load_3d(sb + 0 * B_BLK_BYTES, &tm_b0, full_bar(s), n0, kb * BK, c.e);
            tma_load_3d(sb + 1 * B_BLK_BYTES, &tm_b0, full_bar(s), n0 + 64, kb * BK, c.e);
            tma_load_3d(sb + 2 * B_BLK_BYTES, &tm_b1, full_bar(s), n0, kb * BK, c.e);
            tma_load_3d(sb + 3 * B_BLK_BYTES, &tm_b1, full_bar(s), n0 + 64, kb * BK, c.e);
          } else {
            #pragma unroll
            for (int j = 0; j < 4; ++j)
              tma_load_3d(sb + j * B_BLK_BYTES, &tm_b0, full_bar(s), n0 + 64 * j, kb * BK, c.e);
          }
          if (++s == STAGES) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (one thread) =====================
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      int it = 0;
      for (int t = blockIdx.x; t < total_tiles; t += gridDim.x, ++it) {
        const int as = it & 1;
        const uint32_t aph = (it >> 1) & 1u;
        mbar_wait(tempty_bar(as), aph ^ 1u);          // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * BN;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(full_bar(s), ph);
          tc_fence_after();
          const uint32_t sa = base + s * STAGE_BYTES;
          const uint32_t sb = sa + A_BYTES;
          const uint64_t ad = ADESC_HI | ((sa >> 4) & 0x3FFFu);
          const uint64_t bd = BDESC_HI | ((sb >> 4) & 0x3FFFu);
          #pragma unroll
          for (int kk = 0; kk < BK / UK; ++kk) {
            // A: +16 k = +32 bytes inside the swizzle span; B: +16 k = two 8-row groups = +2048 bytes
            umma_f16(d_tmem, ad + ((kk * UK * 2) >> 4), bd + ((kk * UK * 128) >> 4), IDESC,
                     (kb | kk) != 0 ? 1u : 0u);
          }
          umma_commit(empty_bar(s));                  // smem slot free once these MMAs retire
          if (++s == STAGES) { s = 0; ph ^= 1u; }
        }
        umma_commit(tfull_bar(as));                   // accumulator complete -> epilogue
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: TMEM -> registers -> global =====================
    const int q = warp & 3;                            // TMEM lane quarter this warp may read
    int it = 0;
    for (int t = blockIdx.x; t < total_tiles; t += gridDim.x, ++it) {
      const TileCoord c = decode_tile(t, tile_start, m_tiles, p.offsets, E);
      const int as = it & 1;
      const uint32_t aph = (it >> 1) & 1u;
      const int row_in_tile = q * 32 + lane;
      const bool row_ok = row_in_tile < c.rows_valid;
      const int64_t grow = static_cast<int64_t>(c.row0) + row_in_tile;
      const int n0 = c.n_tile * OUT_COLS;
      float scale = 1.0f;
      if (!GATEUP && p.row_scale != nullptr && row_ok) scale = __ldg(p.row_scale + __ldg(p.row_src + grow));
      mbar_wait(tfull_bar(as), aph);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + as * BN;
      uint8_t* stage_buf = epi_smem + q * EPI_WARP_BYTES;
      const uint32_t my_row_smem = smem_u32(stage_buf) + lane * EPI_PITCH;
      // transposed read-out: lane -> (row = lane/8 + 4*j, 16-byte piece = lane%8)
      const int piece = lane & 7, sub_row = lane >> 3;
      #pragma unroll 1
      for (int ch = 0; ch < OUT_COLS / 64; ++ch) {            // 64 output columns per round
        #pragma unroll
        for (int half = 0; half < 2; ++half) {
          const int c32 = ch * 64 + half * 32;               // first of 32 output columns
          uint32_t packed[16];
          if (GATEUP) {
            uint32_t g[32], u[32];
            tmem_ld_32x32(taddr + c32, g);
            tmem_ld_32x32(taddr + BN / 2 + c32, u);
            tmem_ld_wait();
            #pragma unroll
            for (int j = 0; j < 16; ++j)
              packed[j] = pack_bf16(silu_mul(__uint_as_float(g[2 * j]), __uint_as_float(u[2 * j])),
                                    silu_mul(__uint_as_float(g[2 * j + 1]), __uint_as_float(u[2 * j + 1])));
          } else {
            uint32_t a[32];
            tmem_ld_32x32(taddr + c32, a);
            tmem_ld_wait();
            #pragma unroll
            for (int j = 0; j < 16; ++j)
              packed[j] = pack_bf16(__uint_as_float(a[2 * j]) * scale, __uint_as_float(a[2 * j + 1]) * scale);
          }
          #pragma unroll
          for (int v = 0; v < 4; ++v)
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(my_row_smem + half * 64 + v * 16),
                         "r"(packed[4 * v]), "r"(packed[4 * v + 1]), "r"(packed[4 * v + 2]), "r"(packed[4 * v + 3])
                         : "memory");
        }
        __syncwarp();
        const int col = n0 + ch * 64 + piece * 8;
        if (col + 8 <= p.N) {
          #pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int r = sub_row + 4 * j;                   // row inside this warp's 32
            if (q * 32 + r < c.rows_valid) {
              const uint4 val = *reinterpret_cast<const uint4*>(stage_buf + r * EPI_PITCH + piece * 16);
              *reinterpret_cast<uint4*>(p.out + (static_cast<int64_t>(c.row0) + q * 32 + r) * p.N + col) = val;
            }
          }
        }
        __syncwarp();
      }
      tc_fence_before();
      mbar_arrive(tempty_bar(as));
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

Params make_params(const GemmLaunch& g) {
  Params p;
  p.offsets = g.offsets;
  p.E = g.E;
  p.K = g.K;
  p.N = g.N;
  p.out = static_cast<__nv_bfloat16*>(g.out);
  p.row_scale = g.row_scale;
  p.row_src = g.row_src;
  p.w4d = g.w4d;
  return p;
}

}  // namespace

cudaError_t gemm_kernels_init() {
  cudaError_t e = cudaFuncSetAttribute(grouped_gemm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(grouped_gemm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              SMEM_BYTES);
}

cudaError_t launch_gateup_swiglu(const GemmLaunch& g, cudaStream_t st) {
  launch_pdl(grouped_gemm_kernel<true>, g.num_sms, NUM_THREADS, SMEM_BYTES, st, g.tm_act.m[15], g.w4d ? g.tm_b0_4d : g.tm_b0, g.w4d ? g.tm_b1_4d : g.tm_b1, make_params(g));
  return cudaGetLastError();
}

cudaError_t launch_down(const GemmLaunch& g, cudaStream_t st) {
  launch_pdl(grouped_gemm_kernel<false>, g.num_sms, NUM_THREADS, SMEM_BYTES, st, g.tm_act.m[15], g.w4d ? g.tm_b0_4d : g.tm_b0, g.w4d ? g.tm_b0_4d : g.tm_b0, make_params(g));
  return cudaGetLastError();
}

}  // namespace bg
