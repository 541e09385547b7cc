// grouped_gemm.cu -- steps a7 / a8 (and, fused, a6) of the combined MoE layer on sm_100a tensor cores.
//
//   a7: H[r,:] = silu(x_perm[r,:] W_gate[e]) (.) (x_perm[r,:] W_up[e])      rows r of expert e
//   a8: Y[r,:] = (w[row_src[r]]) * (H[r,:] W_down[e])
// (BASELINE.json north_star "grouped SwiGLU expert FFN".)
//
// "Swap-AB" orientation: the WEIGHTS sit on the UMMA M axis (128 output features per tile) and the
// TOKENS on the UMMA N axis, because N is the only tile dimension tcgen05 lets us size finely
// (any multiple of 16 up to 256 at M = 128).  Per-expert row counts are whatever the router
// produced (a few rows for a cold expert, a ragged tail for every expert), so the token extent
// of a tile is ceil16(rows) and the tensor-core time of a tile is proportional to the rows it
// really has, not to a padded 128-row block.
//
//   A operand: weights [E, K, N_out] bf16, N_out contiguous -> MN-major, TMA boxes {64 n, 64 k, 1}
//              a7: M rows 0..63 = 64 W_gate columns, M rows 64..127 = the same 64 W_up columns
//              a8: M rows 0..127 = 128 consecutive W_down columns
//   B operand: activations [rows, K] bf16, K contiguous     -> K-major,  TMA box {64 k, NT rows}
//   D (TMEM) : [128 lanes = features] x [NT columns = tokens] fp32, two stages of 256 columns
// The weights are consumed in the layout the layer is given (reading S14): no transpose/prepack.
//
// Warp roles (one persistent 256-thread CTA per SM, + 128 threads when the gather is fused):
//   warp 0  lane 0: TMA producer of the A (weight) ring        -- 6 stages x 16 KB, streams from HBM
//   warp 3  lane 0: TMA producer of the B (activation) ring    -- 3 stages x 32 KB, mostly L2 hits
//   warp 1  lane 0: tcgen05.mma issuer (waits on both rings)
//   warp 2        : TMEM allocator
//   warps 4-7     : epilogue (TMEM -> registers -> SwiGLU | gate weight -> bf16 -> global)
//   warps 8-11    : fused gather (a6 inside a7): the B ring is filled with 16-byte cp.async copies of
//                   hidden[row_src[r]/k, :] in the 128B-swizzled layout TMA would have produced;
//                   x_perm is never written.
// The two operand rings are separate because their latencies differ: weight strips come from HBM
// and want depth, activation tiles are re-read by every feature tile and come from L2.
//
// a7 epilogue: gate and up accumulators of one feature live in different TMEM lane quarters
// (lanes f and 64+f), i.e. in different warps.  Warp pairs (0,2) and (1,3) exchange 32-token chunks
// through shared memory: for chunks (2i, 2i+1) the up-warp hands its chunk 2i to the gate-warp
// and the gate-warp hands its chunk 2i+1 to the up-warp, so both warps do half of the SiLU work.
//
// Tile scheduler: token tiles never straddle experts.  Expert e with n_e rows owns
// tt_e = ceil(n_e/256) token tiles of `base_e` = ceil16(ceil(n_e/tt_e)) rows (the last one shorter)
// times ceil(N_out/OUT_FEATS) feature tiles, ordered feature-tile-major / token-tile-minor so the
// CTAs running at the same time share weight strips through L2.  Tile t -> CTA (t mod gridDim.x).
// Experts with no rows own no tiles and their weights are never touched.
#include "kernels.h"
#include "ptx_sm100.cuh"

namespace bg {
namespace {

constexpr int BM = 128;            // UMMA M: weight-side rows of a tile
constexpr int BN_MAX = 256;        // UMMA N max: tokens per tile
constexpr int BK = 64;             // k per pipeline stage = one 128-byte swizzle span of bf16
constexpr int UK = 16;             // UMMA K for 16-bit inputs
#ifndef BG_A_STAGES
#define BG_A_STAGES 6
#endif
#ifndef BG_B_STAGES
#define BG_B_STAGES 3
#endif
constexpr int A_STAGES = BG_A_STAGES;
constexpr int B_STAGES = BG_B_STAGES;
constexpr int A_BLK_BYTES = 64 * BK * 2;            // 8 KB: one 64-feature block of weights
constexpr int A_BYTES = 2 * A_BLK_BYTES;            // 16 KB
constexpr int B_BYTES = BN_MAX * BK * 2;            // 32 KB
constexpr int NUM_THREADS = 256;
constexpr int GATHER_THREADS = 128;
constexpr int GATHER_LAG = 2;      // cp.async groups kept in flight per gather thread (< B_STAGES)
constexpr int MAX_E = 256;
constexpr int XCH_PITCH = 36;                       // words per lane row of an exchange buffer (conflict-free v4)
constexpr int XCH_BYTES = 32 * XCH_PITCH * 4;       // 4608 B
constexpr int BAR_BYTES = 256;
constexpr int TABLE_BYTES = 2064;                   // 2 x (MAX_E + 1) ints, 16-byte padded
constexpr int STAGE_TILE_BYTES = 32 * 64;            // per-warp output staging: [32 tokens][32 features] bf16
// epilogue scratch: [4 exchange buffers (a7) | 4 x 256 gate weights (a8)] then the 4 staging tiles
constexpr int EPI_BYTES = 4 * XCH_BYTES + 4 * STAGE_TILE_BYTES;
constexpr int SMEM_BYTES = A_STAGES * A_BYTES + B_STAGES * B_BYTES + 1024 /*align slack*/ + BAR_BYTES +
                           TABLE_BYTES + EPI_BYTES;

// M = 128, A MN-major (weights), B K-major (tokens); the N field is filled in per tile.
constexpr uint32_t IDESC_BASE = umma_idesc_bf16(BM, 0, /*A MN-major*/ 1, /*B K-major*/ 0);
// A: MN-major SW128: 64-feature blocks A_BLK_BYTES apart (LBO); 8-k-row groups 1024 B apart (SBO).
constexpr uint64_t ADESC_HI = umma_desc_sw128(A_BLK_BYTES, 1024);
// B: K-major SW128: 8-token groups 1024 B apart (SBO); LBO unused inside one swizzle span.
constexpr uint64_t BDESC_HI = umma_desc_sw128(16, 1024);

struct Params {
  const int32_t* offsets;
  int E, K, N;                 // N = output features (f for a7, d for a8)
  __nv_bfloat16* out;
  const float* row_scale;
  const int32_t* row_src;
  const uint8_t* gather_src;   // hidden (bf16 [T,K]) when the B rows are gathered in-kernel
  int k;
};

__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

struct TileCoord {
  int e, row0, rows_valid, nt, f_tile;
};

// tile_start[e] = first linear tile index of expert e (tile_start[E] = total);
// t_tiles[e] = token tiles of expert e.  Both live in shared memory.
__device__ __forceinline__ TileCoord decode_tile(int t, const int* tile_start, const int* t_tiles,
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
  const int tt = t_tiles[e];
  const int f_tile = local / tt;
  const int t_tile = local - f_tile * tt;
  const int beg = __ldg(offsets + e), end = __ldg(offsets + e + 1);
  const int n_e = end - beg;
  const int base = (((n_e + tt - 1) / tt) + 15) & ~15;      // rows per token tile, multiple of 16, <= 256
  TileCoord c;
  c.e = e;
  c.row0 = beg + t_tile * base;
  c.rows_valid = min(base, end - c.row0);
  c.nt = (c.rows_valid + 15) & ~15;
  c.f_tile = f_tile;
  return c;
}

// silu(g) * u with silu(g) = g / (1 + exp(-g)) = h + h tanh(h), h = g/2 (the same function; one
// MUFU instead of two; tanh.approx has 2^-11 relative error, far below the bf16 rounding of H).
__device__ __forceinline__ float silu_mul(float g, float u) {
  const float h = 0.5f * g;
  float th;
  asm("tanh.approx.f32 %0, %1;" : "=f"(th) : "f"(h));
  return fmaf(h, th, h) * u;
}

__device__ __forceinline__ void st_shared_bf16(uint32_t addr, float v) {
#ifdef BG_DBG_NO_STORE
  if (v == 123456.789f)
#endif
  {
    const __nv_bfloat16 b = __float2bfloat16_rn(v);
    asm volatile("st.shared.b16 [%0], %1;" ::"r"(addr), "h"(*reinterpret_cast<const uint16_t*>(&b)) : "memory");
  }
}

// GATEUP = true : a7 (A = [64 W_gate columns | 64 W_up columns], SwiGLU epilogue, 64 output features / tile)
// GATEUP = false: a8 (A = 128 W_down columns, optional per-token scale, 128 output features / tile)
// GATHER (a7 only): B rows come from hidden through row_src (cp.async), not from x_perm by TMA
template <bool GATEUP, bool GATHER>
__global__ void __launch_bounds__(NUM_THREADS + (GATHER ? GATHER_THREADS : 0), 1)
grouped_gemm_kernel(const __grid_constant__ ActMaps tm_act, const __grid_constant__ CUtensorMap tm_w0,
                    const __grid_constant__ CUtensorMap tm_w1, const Params p) {
  constexpr int OUT_FEATS = GATEUP ? BM / 2 : BM;    // output features per tile
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;       // SW128 tiles need 1024-byte alignment
  uint8_t* smem = smem_raw + (base - raw);
  const uint32_t a_base = base;
  const uint32_t b_base = base + A_STAGES * A_BYTES;
  constexpr int RING_BYTES = A_STAGES * A_BYTES + B_STAGES * B_BYTES;
  const uint32_t bar_base = base + RING_BYTES;
  // barriers: fullA[6] emptyA[6] fullB[3] emptyB[3] tmem_full[2] tmem_empty[2]; then the TMEM address
  auto fullA = [&](int s) { return bar_base + 8u * s; };
  auto emptyA = [&](int s) { return bar_base + 8u * (A_STAGES + s); };
  auto fullB = [&](int s) { return bar_base + 8u * (2 * A_STAGES + s); };
  auto emptyB = [&](int s) { return bar_base + 8u * (2 * A_STAGES + B_STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * A_STAGES + 2 * B_STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * A_STAGES + 2 * B_STAGES + 2 + a); };
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + RING_BYTES + 8 * (2 * A_STAGES + 2 * B_STAGES + 4));
  int* tile_start = reinterpret_cast<int*>(smem + RING_BYTES + BAR_BYTES);
  int* t_tiles = tile_start + (MAX_E + 1);
  uint8_t* epi_smem = smem + RING_BYTES + BAR_BYTES + TABLE_BYTES;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int E = p.E;
  const int f_tiles = (p.N + OUT_FEATS - 1) / OUT_FEATS;
  const int k_blocks = (p.K + BK - 1) / BK;

  // ---- per-CTA tile table: inclusive scan of per-expert tile counts (E <= 256)
  {
    int tt = 0;
    if (threadIdx.x < E) {
      const int cnt = __ldg(p.offsets + threadIdx.x + 1) - __ldg(p.offsets + threadIdx.x);
      tt = (cnt + BN_MAX - 1) / BN_MAX;
      t_tiles[threadIdx.x] = tt;
    }
    int v = tt * f_tiles;
    #pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v += u;
    }
    __shared__ int warp_tot[NUM_THREADS / 32];
    if (lane == 31 && warp < NUM_THREADS / 32) warp_tot[warp] = v;
    __syncthreads();
    int add = 0;
    for (int w = 0; w < warp && w < NUM_THREADS / 32; ++w) add += warp_tot[w];
    v += add;                                   // inclusive prefix for thread's expert
    if (threadIdx.x < E) tile_start[threadIdx.x + 1] = v;
    if (threadIdx.x == 0) tile_start[0] = 0;
  }

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_w0);
    if (GATEUP) tma_prefetch_desc(&tm_w1);
    for (int s = 0; s < A_STAGES; ++s) { mbar_init(fullA(s), 1); mbar_init(emptyA(s), 1); }
    for (int s = 0; s < B_STAGES; ++s) { mbar_init(fullB(s), GATHER ? GATHER_THREADS : 1); mbar_init(emptyB(s), 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 128); }
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
    // ===================== A producer: weight strips, TMA (one thread) =====================
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
        const TileCoord c = decode_tile(t, tile_start, t_tiles, p.offsets, E);
        const int n0 = c.f_tile * OUT_FEATS;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(emptyA(s), ph ^ 1u);
          const uint32_t sa = a_base + s * A_BYTES;
          mbar_expect_tx(fullA(s), A_BYTES);
          if (GATEUP) {
            tma_load_3d(sa, &tm_w0, fullA(s), n0, kb * BK, c.e);
            tma_load_3d(sa + A_BLK_BYTES, &tm_w1, fullA(s), n0, kb * BK, c.e);
          } else {
            tma_load_3d(sa, &tm_w0, fullA(s), n0, kb * BK, c.e);
            tma_load_3d(sa + A_BLK_BYTES, &tm_w0, fullA(s), n0 + 64, kb * BK, c.e);
          }
          if (++s == A_STAGES) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == 3) {
    // ===================== B producer: activation rows, TMA (one thread) =====================
    if (!GATHER && lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
        const TileCoord c = decode_tile(t, tile_start, t_tiles, p.offsets, E);
        // the smallest power-of-two box (>= 16 rows) that covers the tile's rows; rows of the slot
        // past the box keep stale data, which only feeds accumulator columns that are never stored
        const int box = c.rows_valid <= 16 ? 16 : 1 << (32 - __clz(c.rows_valid - 1));
        const CUtensorMap* tm_b = &tm_act.m[27 - __clz(box)];          // log2(box) - 4
        const uint32_t tx = box * BK * 2;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(emptyB(s), ph ^ 1u);
          mbar_expect_tx(fullB(s), tx);
          tma_load_2d(b_base + s * B_BYTES, tm_b, fullB(s), kb * BK, c.row0);
          if (++s == B_STAGES) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (one thread) =====================
    if (lane == 0) {
      int sa = 0, sb = 0;
      uint32_t pha = 0, phb = 0;
      int it = 0;
      for (int t = blockIdx.x; t < total_tiles; t += gridDim.x, ++it) {
        const TileCoord c = decode_tile(t, tile_start, t_tiles, p.offsets, E);
        const uint32_t idesc = IDESC_BASE | (static_cast<uint32_t>(c.nt >> 3) << 17);
        const int as = it & 1;
        const uint32_t aph = (it >> 1) & 1u;
        mbar_wait(tempty_bar(as), aph ^ 1u);          // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * BN_MAX;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(fullA(sa), pha);
          mbar_wait(fullB(sb), phb);
          tc_fence_after();
          const uint32_t a_addr = a_base + sa * A_BYTES;
          const uint32_t b_addr = b_base + sb * B_BYTES;
          const uint64_t ad = ADESC_HI | ((a_addr >> 4) & 0x3FFFu);
          const uint64_t bd = BDESC_HI | ((b_addr >> 4) & 0x3FFFu);
          #pragma unroll
          for (int kk = 0; kk < BK / UK; ++kk) {
            // A (MN-major): +16 k = two 8-row groups = +2048 bytes; B (K-major): +16 k = +32 bytes in the span
            umma_f16(d_tmem, ad + ((kk * UK * 128) >> 4), bd + ((kk * UK * 2) >> 4), idesc,
                     (kb | kk) != 0 ? 1u : 0u);
          }
          umma_commit(emptyA(sa));                    // slots free once these MMAs retire
          umma_commit(emptyB(sb));
          if (++sa == A_STAGES) { sa = 0; pha ^= 1u; }
          if (++sb == B_STAGES) { sb = 0; phb ^= 1u; }
        }
        umma_commit(tfull_bar(as));                   // accumulator complete -> epilogue
      }
    }
  } else if (warp >= 4 && warp < 8) {
    // ===================== epilogue: TMEM -> registers -> shared (transpose) -> global ==========
    // A thread owns one feature (TMEM lane) and reads 32 tokens (columns) at a time; the output is
    // token-major, so each warp turns its 32 feature x 32 token block around in a private 2 KB
    // staging tile ([token][32 features] bf16) and stores 16 bytes per lane, 64 contiguous bytes
    // per token.  Instruction count matters here: the four epilogue warps sit alone on their SM
    // sub-partitions, so every instruction is exposed.
    const int q = warp & 3;                            // TMEM lane quarter this warp may read
    uint8_t* stage = epi_smem + 4 * XCH_BYTES + q * STAGE_TILE_BYTES;
    const uint32_t stage_wr = smem_u32(stage) + lane * 2;                       // + token * 64
    const uint32_t stage_rd = smem_u32(stage) + (lane >> 2) * 64 + (lane & 3) * 16;   // + i * 512
    float* sc_smem = reinterpret_cast<float*>(epi_smem) + q * BN_MAX;           // a8: this warp's copy
    const int feat0 = (GATEUP ? (q & 1) : q) * 32;     // first of this warp's 32 output features in the tile
    int it = 0;
    for (int t = blockIdx.x; t < total_tiles; t += gridDim.x, ++it) {
      const TileCoord c = decode_tile(t, tile_start, t_tiles, p.offsets, E);
      const int as = it & 1;
      const uint32_t aph = (it >> 1) & 1u;
      const int n_chunks = (c.nt + 31) >> 5;           // 32-token chunks (the last may be half used)
      const int col = c.f_tile * OUT_FEATS + feat0 + (lane & 3) * 8;            // this lane's 8 output columns
      const bool col_ok = col < p.N;                   // N is a multiple of 8
      __nv_bfloat16* out_tile = p.out + static_cast<int64_t>(c.row0) * p.N + col;
      if (!GATEUP) {
        // gate weights of the tile's tokens -> shared memory, fetched before the accumulator is
        // awaited so the two dependent loads hide behind the main loop
        __syncwarp();
        #pragma unroll
        for (int i = 0; i < BN_MAX / 32; ++i) {
          float sc = 1.0f;
          if (p.row_scale != nullptr && i * 32 + lane < c.rows_valid)
            sc = __ldg(p.row_scale + __ldg(p.row_src + c.row0 + i * 32 + lane));
          sc_smem[i * 32 + lane] = sc;
        }
        __syncwarp();
      }
      mbar_wait(tfull_bar(as), aph);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + as * BN_MAX;
      // token-major write-out of the staged 32 x 32 block of chunk cc
      auto flush_chunk = [&](int cc) {
        __syncwarp();
        const int n_tok = c.rows_valid - cc * 32;
        #pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int r = (lane >> 2) + 8 * i;
          uint4 val;
          asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                       : "=r"(val.x), "=r"(val.y), "=r"(val.z), "=r"(val.w) : "r"(stage_rd + i * 512));
          if (col_ok && r < n_tok)
            *reinterpret_cast<uint4*>(out_tile + static_cast<int64_t>(cc * 32 + r) * p.N) = val;
        }
        __syncwarp();
      };
      if (GATEUP) {
        // pair (q&1): gate warp q in {0,1} and up warp q+2 hold the same 32 features
        const bool is_up = q >= 2;
        float* xch_g2u = reinterpret_cast<float*>(epi_smem + (q & 1) * 2 * XCH_BYTES);   // gate -> up warp
        float* xch_u2g = xch_g2u + XCH_BYTES / 4;                                         // up -> gate warp
        float* my_out = (is_up ? xch_u2g : xch_g2u) + lane * XCH_PITCH;
        const float* my_in = (is_up ? xch_g2u : xch_u2g) + lane * XCH_PITCH;
        const int bar_id = 1 + (q & 1);
        #pragma unroll 1
        for (int c0 = 0; c0 < n_chunks; c0 += 2) {
          uint32_t v0[32], v1[32];
          tmem_ld_32x32(taddr + c0 * 32, v0);
          if (c0 + 1 < n_chunks) tmem_ld_32x32(taddr + (c0 + 1) * 32, v1);
          tmem_ld_wait();
          // hand over the chunk the partner finishes: up warp gives chunk c0, gate warp gives chunk c0+1
          #pragma unroll
          for (int j = 0; j < 32; j += 4)
            *reinterpret_cast<uint4*>(my_out + j) =
                is_up ? make_uint4(v0[j], v0[j + 1], v0[j + 2], v0[j + 3])
                      : make_uint4(v1[j], v1[j + 1], v1[j + 2], v1[j + 3]);
          named_bar_sync(bar_id, 64);
          const int cc = is_up ? c0 + 1 : c0;            // the chunk this warp finishes
          if (cc < n_chunks) {
            #pragma unroll
            for (int j = 0; j < 32; j += 4) {
              const uint4 o = *reinterpret_cast<const uint4*>(my_in + j);
              const uint32_t other[4] = {o.x, o.y, o.z, o.w};
              #pragma unroll
              for (int i = 0; i < 4; ++i) {
                const float g = __uint_as_float(is_up ? other[i] : v0[j + i]);
                const float u = __uint_as_float(is_up ? v1[j + i] : other[i]);
                st_shared_bf16(stage_wr + (j + i) * 64, silu_mul(g, u));
              }
            }
            flush_chunk(cc);
          }
          named_bar_sync(bar_id, 64);                    // exchange buffers free for the next round
        }
      } else {
        #pragma unroll 1
        for (int cc = 0; cc < n_chunks; ++cc) {
          uint32_t v[32];
          tmem_ld_32x32(taddr + cc * 32, v);
          tmem_ld_wait();
          #pragma unroll
          for (int j = 0; j < 32; j += 4) {
            const float4 s4 = *reinterpret_cast<const float4*>(sc_smem + cc * 32 + j);   // broadcast
            st_shared_bf16(stage_wr + (j + 0) * 64, __uint_as_float(v[j + 0]) * s4.x);
            st_shared_bf16(stage_wr + (j + 1) * 64, __uint_as_float(v[j + 1]) * s4.y);
            st_shared_bf16(stage_wr + (j + 2) * 64, __uint_as_float(v[j + 2]) * s4.z);
            st_shared_bf16(stage_wr + (j + 3) * 64, __uint_as_float(v[j + 3]) * s4.w);
          }
          flush_chunk(cc);
        }
      }
      tc_fence_before();
      mbar_arrive(tempty_bar(as));
    }
  } else if (GATHER && warp >= 8) {
    // ===================== fused gather (a6): hidden rows -> swizzled B slot, cp.async ============
    // Eight consecutive lanes copy the eight 16-byte chunks of one row's 128-byte k-span (full
    // sectors); a warp instruction covers 4 rows, the four warps 16 rows, nt/16 rounds the tile.
    // Chunk c of row r lands at r*128 + ((c ^ (r & 7)) << 4): the 128B swizzle TMA applies.
    // cp.async writes through the generic proxy and tcgen05.mma reads through the async proxy, so
    // every thread waits for its own copies of a stage (wait_group, GATHER_LAG stages behind the one
    // it is about to issue), makes them visible with fence.proxy.async, and only then arrives on fullB.
    const int gw = warp - 8, sub = lane >> 3, chunk = lane & 7;
    const int r_in16 = gw * 4 + sub;                                  // row inside a 16-row round
    const uint32_t dst0 = r_in16 * 128 + ((chunk ^ (r_in16 & 7)) << 4);
    const int64_t row_bytes = static_cast<int64_t>(p.K) * 2;
    int s = 0;
    uint32_t ph = 0;
    int issued = 0, pub_s = 0;                                         // stages issued / next stage to publish
    for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
      const TileCoord c = decode_tile(t, tile_start, t_tiles, p.offsets, E);
      const int rounds = c.nt >> 4;
      int tok[16];
      #pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int rr = j * 16 + r_in16;
        tok[j] = (rr < c.rows_valid) ? __ldg(p.row_src + c.row0 + rr) / p.k : -1;
      }
      for (int kb = 0; kb < k_blocks; ++kb) {
        // publish the stage issued GATHER_LAG iterations ago before blocking on a free slot, so the
        // MMA warp always finds the next stage ready while GATHER_LAG stages are in flight
        if (issued >= GATHER_LAG) {
          cp_async_wait<GATHER_LAG - 1>();
          fence_proxy_async();
          mbar_arrive(fullB(pub_s));
          if (++pub_s == B_STAGES) pub_s = 0;
        }
        mbar_wait(emptyB(s), ph ^ 1u);
        const uint32_t sb = b_base + s * B_BYTES + dst0;
        const bool k_ok = kb * BK + chunk * 8 < p.K;                   // k past K must read as zero
        const uint8_t* src_k = p.gather_src + kb * (BK * 2) + chunk * 16;
        #pragma unroll
        for (int j = 0; j < 16; ++j) {
          if (j < rounds) {
            const bool ok = k_ok && tok[j] >= 0;
            cp_async_16(sb + j * 2048, src_k + (ok ? tok[j] * row_bytes : 0), ok ? 16u : 0u);
          }
        }
        cp_async_commit();
        ++issued;
        if (++s == B_STAGES) { s = 0; ph ^= 1u; }
      }
    }
    cp_async_wait<0>();
    fence_proxy_async();
    for (int i = issued > GATHER_LAG ? GATHER_LAG : issued; i > 0; --i) {
      mbar_arrive(fullB(pub_s));
      if (++pub_s == B_STAGES) pub_s = 0;
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
  p.gather_src = static_cast<const uint8_t*>(g.gather_src);
  p.k = g.k;
  return p;
}

}  // namespace

cudaError_t gemm_kernels_init() {
  cudaError_t e = cudaFuncSetAttribute(grouped_gemm_kernel<true, false>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(grouped_gemm_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(grouped_gemm_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              SMEM_BYTES);
}

cudaError_t launch_gateup_swiglu(const GemmLaunch& g, cudaStream_t st) {
  if (g.gather_src != nullptr)
    grouped_gemm_kernel<true, true><<<g.num_sms, NUM_THREADS + GATHER_THREADS, SMEM_BYTES, st>>>(
        g.tm_act, g.tm_b0, g.tm_b1, make_params(g));
  else
    grouped_gemm_kernel<true, false><<<g.num_sms, NUM_THREADS, SMEM_BYTES, st>>>(g.tm_act, g.tm_b0, g.tm_b1,
                                                                                 make_params(g));
  return cudaGetLastError();
}

cudaError_t launch_down(const GemmLaunch& g, cudaStream_t st) {
  grouped_gemm_kernel<false, false><<<g.num_sms, NUM_THREADS, SMEM_BYTES, st>>>(g.tm_act, g.tm_b0, g.tm_b0,
                                                                                  make_params(g));
  return cudaGetLastError();
}

}  // namespace bg
