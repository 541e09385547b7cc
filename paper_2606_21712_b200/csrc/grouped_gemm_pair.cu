// grouped_gemm_pair.cu -- steps a7 / a8 of the combined MoE layer on sm_100a tensor cores, CTA-pair form.
//
//   a7: H[r,:] = silu(x_perm[r,:] W_gate[e]) (.) (x_perm[r,:] W_up[e])      rows r of expert e
//   a8: Y[r,:] = (w[row_src[r]]) * (H[r,:] W_down[e])
// (BASELINE.json north_star "grouped SwiGLU expert FFN".)
//
// Orientation ("swap-AB"): the WEIGHTS sit on the UMMA M axis and the TOKENS on the UMMA N axis,
// because N is the only tile dimension tcgen05 sizes finely (multiples of 16 up to 256).  Per-expert
// row counts are whatever the router produced (a few rows for a cold expert, a ragged tail for every
// expert); with tokens on N the tensor-core time of a tile follows the rows it really has instead of
// a padded 128-row block.
//
// CTA pair (tcgen05 cta_group::2): two CTAs of a cluster run ONE MMA of M = 256.  Each CTA stages
// 128 weight columns (its half of M) and HALF of the tile's tokens (its half of N) in its own shared
// memory and owns 128 accumulator lanes x N columns in its own TMEM.  Per CTA and 64-wide k-block
// that is 16 KB of weights + <= 16 KB of tokens for 128 x 256 x 64 MACs: two thirds of the L2->SM
// traffic of the 1-CTA 128 x 256 tile (48 KB), which ncu showed running at 17 TB/s (profiles/r01).
//
//   A operand: weights [E, K, N_out] bf16, N_out contiguous -> MN-major, TMA boxes {64 n, 64 k, 1}
//              a7: M rows 0..63 = 64 W_gate columns, rows 64..127 = the same 64 W_up columns (per CTA)
//              a8: M rows 0..127 = 128 consecutive W_down columns (per CTA)
//   B operand: activations [rows, K] bf16, K contiguous     -> K-major,  ONE TMA box {64 k, nt/2 rows}
//              (sixteen tensor maps, one per multiple of 8 rows) -- the TMA unit costs ~40 ns per
//              operation whatever its size, so a k-block is 2 (a8) or 3 (a7) operations per CTA
//   D (TMEM) : [128 lanes = features] x [nt columns = tokens] fp32 per CTA, two stages of 256 columns
// The weights are consumed in the layout the layer is given (reading S14): no transpose/prepack.
//
// Warp roles (persistent, one CTA per SM, 74 clusters; every launch uses programmatic dependent launch):
//   warp 0       : TMA producer, one elected lane issues (both CTAs; transaction bytes of both land on the leader's barrier)
//   warp 1       : tcgen05.mma issuer, one elected lane issues (leader CTA only); commits are multicast to both CTAs
//   warp 2       : TMEM allocator
//   warp 3 lane 0: tile scheduler (leader only): ticket counter -> 4-slot ring in both CTAs' shared memory
//   warps 4-7    : epilogue (TMEM -> registers -> SwiGLU | gate weight -> bf16 -> smem transpose -> global);
//                  a8 adds warps 8-11 (384 threads): its k loops are short, two warps serve each TMEM lane quarter
//
// a7 epilogue: gate and up accumulators of one feature live in TMEM lanes f and 64+f, i.e. in
// different warps.  Warp pairs (0,2) and (1,3) exchange 32-token chunks through shared memory: for
// chunks (2i, 2i+1) the up-warp hands chunk 2i to the gate-warp and the gate-warp hands chunk 2i+1 to
// the up-warp, so both warps do half of the SiLU work.
//
// Tile scheduler: token tiles never straddle experts.  Expert e with n_e rows owns
// tt_e = ceil(n_e/256) token tiles of ceil16(ceil(n_e/tt_e)) rows (the last one shorter) times
// ceil(N_out/OUT_FEATS) feature tiles, ordered feature-tile-major / token-tile-minor so that the
// clusters running at the same time share weight strips through L2.  Tiles are drawn in that order from a
// global ticket counter (dynamic feed, see `feed_tile`), so the neighbours really run concurrently and a strip
// is read from HBM once; bg_moe_set_debug(static_tile_feed) keeps the fixed map tile t -> cluster (t mod #clusters).
// Experts with no rows own no tiles and their weights are never touched.
#include "kernels.h"
#include "ptx_sm100.cuh"

namespace bg {
namespace {

constexpr int BN_MAX = 256;        // UMMA N max: tokens per tile
constexpr int BK = 64;             // k per pipeline stage = one 128-byte swizzle span of bf16
constexpr int UK = 16;             // UMMA K for 16-bit inputs
constexpr int STAGES = 6;
constexpr int SCHED_SLOTS = 4;     // tiles published ahead by the dynamic scheduler
constexpr int SLOT_WORDS = 8;      // a published tile: ticket, expert, row0, rows_valid, f_tile, t_tile, token tiles of the expert
constexpr int A_BLK_BYTES = 64 * BK * 2;            // 8 KB: one 64-feature block of weights
constexpr int A_BYTES = 2 * A_BLK_BYTES;            // 16 KB: this CTA's 128 M rows
constexpr int B_BYTES = (BN_MAX / 2) * BK * 2;      // 16 KB: this CTA's half of the tokens
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;      // 32 KB
constexpr int RING_BYTES = STAGES * STAGE_BYTES;    // 192 KB
constexpr int MAX_THREADS = 384;             // 4 role warps + 4 (a7) or 8 (a8) epilogue warps
constexpr int MAX_E = 256;
constexpr int XCH_PITCH = 36;                       // words per lane row of an exchange buffer (conflict-free v4)
constexpr int XCH_BYTES = 32 * XCH_PITCH * 4;       // 4608 B
constexpr int BAR_BYTES = 512;
constexpr int TABLE_BYTES = 3104;                   // 3 x (MAX_E + 1) ints (tile_start, t_tiles, offsets), 16-byte padded
constexpr int STAGE_TILE_BYTES = 32 * 64;           // per-warp output staging: [32 tokens][32 features] bf16
// epilogue scratch: [4 exchange buffers (a7) | 4 x 256 gate weights (a8)] then the 4 staging tiles
constexpr int EPI_BYTES = 4 * XCH_BYTES + 4 * STAGE_TILE_BYTES + BN_MAX * 4;   // a8: 2 KB of scales + 8 staging tiles = 18 KB; FP8 a7: + 1 KB of token scales
static_assert(EPI_BYTES >= 2 * BN_MAX * 4 + 8 * STAGE_TILE_BYTES, "a8 epilogue scratch");
constexpr int SMEM_BYTES = RING_BYTES + 1024 /*align slack*/ + BAR_BYTES + TABLE_BYTES + EPI_BYTES;
static_assert(SMEM_BYTES <= 227 * 1024, "shared memory budget");

// M = 256 (pair), A MN-major (weights), B K-major (tokens); the N field is filled in per tile.
constexpr uint32_t IDESC_BASE = umma_idesc_bf16(256, 0, /*A MN-major*/ 1, /*B K-major*/ 0);
// FP8 gate/up: e4m3 x e4m3, both operands K-major (the quantised weights are stored [E, N, K], reading F3)
constexpr uint32_t IDESC_FP8 = umma_idesc_e4m3(256, 0, 0, 0);
// A: MN-major SW128: 64-feature blocks A_BLK_BYTES apart (LBO); 8-k-row groups 1024 B apart (SBO).
constexpr uint64_t ADESC_HI = umma_desc_sw128(A_BLK_BYTES, 1024);
// B: K-major SW128: 8-token groups 1024 B apart (SBO); LBO unused inside one swizzle span.
constexpr uint64_t BDESC_HI = umma_desc_sw128(16, 1024);

struct Params {
  const int32_t* offsets;
  int E, K, N;                 // N = output features (f for a7, d for a8)
  __nv_bfloat16* out;
  const float* row_scale;      // a8, fused path: gate weight per expert-order row (w_perm[r]); nullptr = 1
  bool w4d;                    // tm_w0 / tm_w1 are the 4-D block views (kernels.h)
  int sg_max;                  // 0 = derive the super-group size from K
  int* tile_counter;           // dynamic feed: [2] = ticket counter, clusters-finished counter (zero between launches); nullptr = static feed
  // FP8 gate/up (reading F4): dequantisation scales
  const float* sx;             // [rows]  per expert-order token row
  const float* sw0;            // [E, N]  per expert and output channel, W_gate
  const float* sw1;            // [E, N]  W_up
  unsigned* hmax;              // a7, FP8 down GEMM downstream (reading F5): [rows] running max |H| (float bits), or nullptr
};

__device__ __forceinline__ void named_bar_sync(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

struct TileCoord {
  int e, row0, rows_valid, nt, f_tile, t_tile, tt;
};

// tile_start[e] = first linear tile index of expert e (tile_start[E] = total);
// t_tiles[e] = token tiles of expert e.  Both live in shared memory.
// Inside an expert the order is feature-tile-major / token-tile-minor, so the token tiles that share a
// weight strip run at the same time.  When an expert's token matrix is too large to stay in L2 between
// two feature tiles (DeepSeek-shaped hot experts: thousands of rows x 14 KB), that order re-streams the
// tokens from HBM once per feature tile; such experts are cut into super-groups of `sg_max` token tiles
// (sized to ~48 MB of tokens) and each super-group runs through all feature tiles before the next starts:
// the tokens stay in L2 and the expert's weights are streamed once per super-group instead.
__device__ __forceinline__ TileCoord decode_tile(int t, const int* tile_start, const int* t_tiles,
                                                 const int32_t* offsets, int E, int sg_max) {
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
  int f_tile, t_tile;
  if (tt <= sg_max) {
    f_tile = local / tt;
    t_tile = local - f_tile * tt;
  } else {
    const int f_tiles = (tile_start[e + 1] - tile_start[e]) / tt;
    const int n_sg = (tt + sg_max - 1) / sg_max;
    const int g = (tt + n_sg - 1) / n_sg;             // balanced super-group size; the last may be smaller
    const int per_sg = g * f_tiles;
    const int sg = local / per_sg;
    const int r = local - sg * per_sg;
    const int g_here = min(g, tt - sg * g);
    f_tile = r / g_here;
    t_tile = sg * g + (r - f_tile * g_here);
  }
  const int beg = offsets[e], end = offsets[e + 1];    // the CTA's shared-memory copy (a global load here sits on every role's path at every tile)
  const int n_e = end - beg;
  const int base = (((n_e + tt - 1) / tt) + 15) & ~15;      // rows per token tile, multiple of 16, <= 256
  TileCoord c;
  c.e = e;
  c.row0 = beg + t_tile * base;
  c.rows_valid = min(base, end - c.row0);
  c.nt = (c.rows_valid + 15) & ~15;
  c.f_tile = f_tile;
  c.t_tile = t_tile;
  c.tt = tt;
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
  const __nv_bfloat16 b = __float2bfloat16_rn(v);
  asm volatile("st.shared.b16 [%0], %1;" ::"r"(addr), "h"(*reinterpret_cast<const uint16_t*>(&b)) : "memory");
}

// GATEUP = true : a7 (per CTA A = [64 W_gate columns | 64 W_up columns], SwiGLU epilogue, 128 output features / pair tile)
// GATEUP = false: a8 (per CTA A = 128 W_down columns, optional per-token scale, 256 output features / pair tile)
// FP8 (a7 only): operands are e4m3 bytes, a k-block is 128 elements (the same 128-byte swizzle span), both K-major;
//                 the epilogue multiplies the accumulators by sx[token] * sw[expert, feature] before the SwiGLU.
template <bool GATEUP, bool FP8 = false>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(GATEUP ? 256 : 384, 1)
pair_gemm_kernel(const __grid_constant__ ActMaps tm_act, const __grid_constant__ CUtensorMap tm_w0,
                 const __grid_constant__ CUtensorMap tm_w1, const Params p) {
  constexpr int CTA_FEATS = GATEUP ? 64 : 128;       // output features per CTA and tile
  constexpr int OUT_FEATS = 2 * CTA_FEATS;           // output features per pair tile
  // a8 has short k loops (K = f), so its epilogue gets two warps per TMEM lane quarter
  constexpr int EPI_WARPS = GATEUP ? 4 : 8;
  constexpr int STAGE_OFF = GATEUP ? 4 * XCH_BYTES : 2 * BN_MAX * 4;   // staging tiles follow the exchange / scale area
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;       // SW128 tiles need 1024-byte alignment
  uint8_t* smem = smem_raw + (base - raw);
  const uint32_t bar_base = base + RING_BYTES;
  // barriers: full[S] empty[S] tmem_full[2] tmem_empty[2]; then the TMEM address
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  // tile feed (dynamic scheduler): sched_full[SCHED_SLOTS] per CTA, sched_empty[SCHED_SLOTS] on the leader
  auto sfull_bar = [&](int i) { return bar_base + 8u * (2 * STAGES + 4 + i); };
  auto sempty_bar = [&](int i) { return bar_base + 8u * (2 * STAGES + 4 + SCHED_SLOTS + i); };
  constexpr int NBAR = 2 * STAGES + 4 + 2 * SCHED_SLOTS;
  static_assert(8 * NBAR + 16 + 4 * SLOT_WORDS * SCHED_SLOTS <= BAR_BYTES, "barrier area");
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + RING_BYTES + 8 * NBAR);
  volatile int* tile_slot = reinterpret_cast<volatile int*>(smem + RING_BYTES + 8 * NBAR + 16);
  constexpr int N_CONSUMERS = 3 + 2 * EPI_WARPS;      // two producers, the MMA thread, every epilogue warp of the pair
  int* tile_start = reinterpret_cast<int*>(smem + RING_BYTES + BAR_BYTES);
  int* t_tiles = tile_start + (MAX_E + 1);
  int* offs = t_tiles + (MAX_E + 1);                  // offsets[0..E], copied once
  uint8_t* epi_smem = smem + RING_BYTES + BAR_BYTES + TABLE_BYTES;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();            // 0 = leader
  const int cluster_id = blockIdx.x >> 1, num_clusters = gridDim.x >> 1;
  const int E = p.E;
  const int f_tiles = (p.N + OUT_FEATS - 1) / OUT_FEATS;
  constexpr int BKE = FP8 ? 2 * BK : BK;             // elements per k-block (128 bytes either way)
  const int k_blocks = (p.K + BKE - 1) / BKE;
  // token tiles whose rows fit ~48 MB of L2 (p.sg_max > 0: override, used by the tests to reach this path on small shapes)
  const int sg_max = p.sg_max > 0 ? p.sg_max : max(1, (48 << 20) / (BN_MAX * 2 * p.K));

  // ---- independent of the previous kernel: barriers and TMEM
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_w0);
    if (GATEUP) tma_prefetch_desc(&tm_w1);
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    // tmem_empty (used on the leader only): one arrival per epilogue warp of both CTAs
    for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 2 * EPI_WARPS); }
    for (int i = 0; i < SCHED_SLOTS; ++i) { mbar_init(sfull_bar(i), 1); mbar_init(sempty_bar(i), N_CONSUMERS); }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc_pair(smem_u32(tmem_slot), 512);
    tmem_relinquish_pair();
  }
  // ---- everything below reads what the previous kernels wrote (offsets, activations)
  pdl_wait_then_trigger();
  // ---- per-CTA tile table: inclusive scan of per-expert tile counts (E <= 256 = blockDim)
  {
    int tt = 0;
    if (threadIdx.x < E) {
      const int o0 = __ldg(p.offsets + threadIdx.x), o1 = __ldg(p.offsets + threadIdx.x + 1);
      const int cnt = o1 - o0;
      tt = (cnt + BN_MAX - 1) / BN_MAX;
      t_tiles[threadIdx.x] = tt;
      offs[threadIdx.x] = o0;
      if (threadIdx.x == E - 1) offs[E] = o1;
    }
    int v = tt * f_tiles;
    #pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v += u;
    }
    __shared__ int warp_tot[MAX_THREADS / 32];
    if (lane == 31) warp_tot[warp] = v;
    __syncthreads();
    int add = 0;
    for (int w = 0; w < warp; ++w) add += warp_tot[w];
    v += add;                                   // inclusive prefix for thread's expert
    if (threadIdx.x < E) tile_start[threadIdx.x + 1] = v;
    if (threadIdx.x == 0) tile_start[0] = 0;
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                 // the peer's barriers are initialised, its TMEM allocated
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const int total_tiles = tile_start[E];

  // ---- tile feed.  Static (tile_counter == nullptr): cluster c takes tiles c, c + 74, ...  Dynamic: tiles
  // are handed out in linear order from a global ticket counter by one thread of the leader CTA (warp 3),
  // written to a 4-slot ring in BOTH CTAs' shared memory and published through sched_full; every consumer
  // (the two TMA producers, the MMA thread, each epilogue warp) reads the ticket and hands the slot back on
  // the leader's sched_empty.  -1 ends the stream.  With tickets drawn in real time the token tiles that
  // share a weight strip stay concurrent however unequal the tiles of a launch are.
  const bool dyn = p.tile_counter != nullptr;
  struct Feed { int slot; uint32_t ph; int t; };
  // Next tile of this cluster into `c`; false = the stream has ended.  Dynamic feed: the scheduler thread has already
  // DECODED the ticket (binary search over the experts, the divisions of the tile order): a consumer reads seven words
  // instead of repeating ~0.3 us of dependent integer work at the head of every tile -- the k loops of the down GEMM are
  // 12 k-blocks (3-5 us) long.
  auto feed_tile = [&](Feed& f, TileCoord& c) -> bool {
    if (!dyn) {
      f.t = (f.t < 0) ? cluster_id : f.t + num_clusters;
      if (f.t >= total_tiles) return false;
      c = decode_tile(f.t, tile_start, t_tiles, offs, E, sg_max);
      return true;
    }
    mbar_wait_cluster(sfull_bar(f.slot), f.ph);
    const volatile int* w = tile_slot + f.slot * SLOT_WORDS;
    const int t = w[0];
    c.e = w[1]; c.row0 = w[2]; c.rows_valid = w[3]; c.f_tile = w[4]; c.t_tile = w[5]; c.tt = w[6];
    c.nt = (c.rows_valid + 15) & ~15;
    // Hand the slot back with a RELAXED arrive whose address depends on the words just read (so it cannot
    // pass the reads): a releasing arrive is a fence that waits for the thread's outstanding work -- the
    // epilogue's global stores, the MMA thread's in-flight tcgen05 operations -- once per tile.
    uint32_t zero;
    asm volatile("and.b32 %0, %1, 0;" : "=r"(zero) : "r"(t | c.e | c.row0 | c.rows_valid | c.f_tile | c.t_tile | c.tt));
    __syncwarp();                                      // all 32 lanes have read; one lane arrives
    if (lane == 0) mbar_arrive_cluster_relaxed(sempty_bar(f.slot) + zero, 0);
    if (++f.slot == SCHED_SLOTS) { f.slot = 0; f.ph ^= 1u; }
    return t >= 0;
  };

  // The TMA and MMA roles run WARP-WIDE with one elected lane issuing (elect.sync): inside `if (lane == 0)` ptxas
  // cannot tell that a single lane is active and wraps every asm statement in an elect / branch loop, and the
  // MMA issue loop is instruction-bound (ncu: ~0.25 us of issue work per 0.30 us k-block on C2), so those extra
  // instructions cost tensor time.
  if (warp == 0) {
    // ===================== TMA producer (one warp per CTA, one elected lane issues) =====================
    int s = 0;
    uint32_t ph = 0;
    Feed feed = {0, 0, -1};
    TileCoord c;
    while (feed_tile(feed, c)) {
      const int n0 = c.f_tile * OUT_FEATS + static_cast<int>(rank) * CTA_FEATS;
      const int half = c.nt >> 1;                    // this CTA's tokens (multiple of 8, <= 128)
      const int brow0 = c.row0 + static_cast<int>(rank) * half;
      const uint32_t tx_pair = 2u * (A_BYTES + static_cast<uint32_t>(half) * (BK * 2));
      const CUtensorMap* tm_b = &tm_act.m[(half >> 3) - 1];
      // An expert with ONE token tile uses each weight byte exactly once: its strips are loaded with an L2
      // evict-first policy so that they do not displace what is reused (token tiles, routing tables, W_r pieces).
      // Measured: C3 at T = 64 / 1024 0.220 -> 0.213 / 0.254 -> 0.247 ms, T = 4096 and C2 unchanged; the same hint on
      // experts with two token tiles, or evict-last on the x_perm / H / Y stores, was slower.
      const bool once = c.tt == 1;
      const uint64_t pol = l2_policy_evict_first();
      // a8 with an expert's weight matrix larger than ~half of L2 (Mixtral: 117 MB): every feature tile streams 7 MB of
      // weights past the expert's H tiles, which all later feature tiles need again -- the H tiles are loaded evict-last.
      // Measured on C2: down reads 1.66-1.80 GB per launch instead of 1.73-2.02 GB (ncu, four captures; algorithmic 1.17 GB),
      // step 2.103 / 2.102 -> 2.095 / 2.086 ms (same call, alternating builds).
      // With small experts (C3: 3 MB) the sticky lines only crowd the next kernels' data (C3 T=16384 1.181 -> 1.186 ms).
      const uint64_t pol_last = l2_policy_evict_last();
      const bool keep_tokens = !GATEUP && static_cast<int64_t>(p.K) * p.N * 2 > (48ll << 20);
      for (int kb = 0; kb < k_blocks; ++kb) {
        mbar_wait(empty_bar(s), ph ^ 1u);            // this CTA's slot is free (multicast commit)
        if (elect_one()) {
          const uint32_t sa = base + s * STAGE_BYTES;
          const uint32_t sb = sa + A_BYTES;
          const uint32_t fb = leader_bar(full_bar(s));
          if (rank == 0) mbar_expect_tx(full_bar(s), tx_pair);   // the bytes of both CTAs
          if (FP8 && GATEUP) {
            // quantised weights [E, N, K] bytes: box {128 k, 64 features, 1}: K-major, 8 KB per tensor
            tma_load_3d_pair(sa, &tm_w0, fb, kb * BKE, n0, c.e);
            tma_load_3d_pair(sa + A_BLK_BYTES, &tm_w1, fb, kb * BKE, n0, c.e);
          } else if (FP8) {
            tma_load_3d_pair(sa, &tm_w0, fb, kb * BKE, n0, c.e);      // W_down codes: box {128 k, 128 features, 1}
          } else if (p.w4d && once) {
            tma_load_4d_pair_hint(sa, &tm_w0, fb, 0, kb * BK, n0 >> 6, c.e, pol);
            if (GATEUP) tma_load_4d_pair_hint(sa + A_BLK_BYTES, &tm_w1, fb, 0, kb * BK, n0 >> 6, c.e, pol);
          } else if (p.w4d) {
            // one operation per weight tensor: nblk 64-column blocks in [block][k][64 n] order
            tma_load_4d_pair(sa, &tm_w0, fb, 0, kb * BK, n0 >> 6, c.e);
            if (GATEUP) tma_load_4d_pair(sa + A_BLK_BYTES, &tm_w1, fb, 0, kb * BK, n0 >> 6, c.e);
          } else if (GATEUP) {
            tma_load_3d_pair(sa, &tm_w0, fb, n0, kb * BK, c.e);
            tma_load_3d_pair(sa + A_BLK_BYTES, &tm_w1, fb, n0, kb * BK, c.e);
          } else {
            tma_load_3d_pair(sa, &tm_w0, fb, n0, kb * BK, c.e);
            tma_load_3d_pair(sa + A_BLK_BYTES, &tm_w0, fb, n0 + 64, kb * BK, c.e);
          }
          // this CTA's half of the tokens: one box of exactly `half` rows
          if (keep_tokens && c.tt > 1) tma_load_2d_pair_hint(sb, tm_b, fb, kb * BKE, brow0, pol_last);
          else tma_load_2d_pair(sb, tm_b, fb, kb * BKE, brow0);
        }
        __syncwarp();
        if (++s == STAGES) { s = 0; ph ^= 1u; }
      }
    }
  } else if (warp == 3) {
    // ===================== tile scheduler (dynamic feed only; one thread of the leader CTA) ==========
    if (dyn && lane == 0 && rank == 0) {
      int slot = 0;
      uint32_t ph = 0;
      while (true) {
        mbar_wait(sempty_bar(slot), ph ^ 1u);          // every consumer has read this slot's previous ticket
        int t = atomicAdd(p.tile_counter, 1);
        if (t >= total_tiles) t = -1;
        int w[7] = {t, 0, 0, 0, 0, 0, 0};
        if (t >= 0) {
          const TileCoord c = decode_tile(t, tile_start, t_tiles, offs, E, sg_max);
          w[1] = c.e; w[2] = c.row0; w[3] = c.rows_valid; w[4] = c.f_tile; w[5] = c.t_tile; w[6] = c.tt;
        }
        #pragma unroll
        for (int i = 0; i < 7; ++i) {
          tile_slot[slot * SLOT_WORDS + i] = w[i];
          st_shared_cluster_u32(smem_u32(const_cast<int*>(tile_slot + slot * SLOT_WORDS + i)), 1, static_cast<uint32_t>(w[i]));
        }
        mbar_arrive(sfull_bar(slot));                  // release.cta: the local store above
        mbar_arrive_cluster(sfull_bar(slot), 1);       // release.cluster: the remote store above
        if (t < 0) break;
        if (++slot == SCHED_SLOTS) { slot = 0; ph ^= 1u; }
      }
      // the last cluster to run dry re-arms the counters for the next launch
      if (atomicAdd(p.tile_counter + 1, 1) == num_clusters - 1) {
        p.tile_counter[0] = 0;
        p.tile_counter[1] = 0;
        __threadfence();
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (one warp of the leader CTA, one elected lane issues) =====================
    if (rank == 0) {
      int s = 0;
      uint32_t ph = 0;
      int it = 0;
      Feed feed = {0, 0, -1};
      TileCoord c;
      for (; feed_tile(feed, c); ++it) {
        const uint32_t idesc = (FP8 ? IDESC_FP8 : IDESC_BASE) | (static_cast<uint32_t>(c.nt >> 3) << 17);
        const int as = it & 1;
        const uint32_t aph = (it >> 1) & 1u;
        mbar_wait(tempty_bar(as), aph ^ 1u);          // both CTAs' epilogues have drained this accumulator
        const uint32_t d_tmem = tmem_base + as * BN_MAX;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(full_bar(s), ph);
          tc_fence_after();
          if (elect_one()) {
            const uint32_t a_addr = base + s * STAGE_BYTES;
            const uint32_t b_addr = a_addr + A_BYTES;
            const uint64_t ad = (FP8 ? BDESC_HI : ADESC_HI) | ((a_addr >> 4) & 0x3FFFu);   // FP8: A is K-major too
            const uint64_t bd = BDESC_HI | ((b_addr >> 4) & 0x3FFFu);
            #pragma unroll
            for (int kk = 0; kk < BK / UK; ++kk) {
              if (FP8) {
                // both K-major: +32 k (one MMA of 8-bit inputs) = +32 bytes in the span
                umma_f8_pair(d_tmem, ad + ((kk * 32) >> 4), bd + ((kk * 32) >> 4), idesc, (kb | kk) != 0 ? 1u : 0u);
              } else {
                // A (MN-major): +16 k = two 8-row groups = +2048 bytes; B (K-major): +16 k = +32 bytes in the span
                umma_f16_pair(d_tmem, ad + ((kk * UK * 128) >> 4), bd + ((kk * UK * 2) >> 4), idesc,
                              (kb | kk) != 0 ? 1u : 0u);
              }
            }
            umma_commit_pair(empty_bar(s));           // both CTAs' slots free once these MMAs retire
            if (kb + 1 == k_blocks) umma_commit_pair(tfull_bar(as));   // accumulator complete -> both epilogues
          }
          __syncwarp();
          if (++s == STAGES) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: TMEM -> registers -> shared (transpose) -> global ==========
    // A thread owns one feature (TMEM lane) and reads 32 tokens (columns) at a time; the output is
    // token-major, so each warp turns its 32 feature x 32 token block around in a private 2 KB
    // staging tile ([token][32 features] bf16) and stores 16 bytes per lane, 64 contiguous bytes
    // per token.
    const int q = warp & 3;                            // TMEM lane quarter this warp may read
    const int ew = warp - 4, sub = ew >> 2;            // a8: warps 4-7 take even chunks, warps 8-11 odd chunks
    uint8_t* stage = epi_smem + STAGE_OFF + ew * STAGE_TILE_BYTES;
    const uint32_t stage_wr = smem_u32(stage) + lane * 2;                       // + token * 64
    const uint32_t stage_rd = smem_u32(stage) + (lane >> 2) * 64 + (lane & 3) * 16;   // + i * 512
    float* sc_smem = reinterpret_cast<float*>(epi_smem);                        // a8: [2][BN_MAX] gate weights, double-buffered
    const int feat0 = static_cast<int>(rank) * CTA_FEATS + (GATEUP ? (q & 1) : q) * 32;   // in the pair tile
    Feed feed = {0, 0, -1};
    TileCoord c, cn;
    bool have = feed_tile(feed, c);
    if (!GATEUP && have) {                           // gate weights of the first tile -> buffer 0
      float sc = 1.0f;
      if (p.row_scale != nullptr && ew * 32 + lane < c.rows_valid) sc = __ldg(p.row_scale + c.row0 + ew * 32 + lane);
      sc_smem[ew * 32 + lane] = sc;
    }
    int it = 0;
    for (; have; ++it) {
      const bool have_next = feed_tile(feed, cn);      // this cluster's next tile (false: none)
      const int as = it & 1;
      const uint32_t aph = (it >> 1) & 1u;
      const int n_chunks = (c.nt + 31) >> 5;           // 32-token chunks (the last may be half used)
      const int col = c.f_tile * OUT_FEATS + feat0 + (lane & 3) * 8;            // this lane's 8 output columns
      const bool col_ok = col < p.N;                   // N is a multiple of 8
      __nv_bfloat16* out_tile = p.out + static_cast<int64_t>(c.row0) * p.N + col;
      float sc_next = 1.0f;
      if (!GATEUP) {
        // Gate weights (already in expert order: w_perm[r]) of the NEXT tile: warp ew fetches tokens
        // ew*32 .. +31 now and parks them in the other buffer after this tile's chunks, so the load
        // latency never sits on the epilogue's critical path.  The barrier makes this tile's buffer
        // (written by all eight warps at the end of the previous tile) visible.
        if (have_next && p.row_scale != nullptr) {
          if (ew * 32 + lane < cn.rows_valid) sc_next = __ldg(p.row_scale + cn.row0 + ew * 32 + lane);
        }
        named_bar_sync(3, 32 * EPI_WARPS);
      }
      float swg = 1.0f, swu = 1.0f;                    // FP8: this thread's feature's weight scales
      float* sx_smem = reinterpret_cast<float*>(epi_smem + 4 * XCH_BYTES + 4 * STAGE_TILE_BYTES);   // FP8: [BN_MAX] token scales
      if (FP8 && GATEUP) {
        const int n = c.f_tile * OUT_FEATS + feat0 + lane;                    // this thread's output feature
        if (n < p.N) {
          swg = __ldg(p.sw0 + static_cast<int64_t>(c.e) * p.N + n);
          swu = __ldg(p.sw1 + static_cast<int64_t>(c.e) * p.N + n);
        }
        named_bar_sync(5, 32 * EPI_WARPS);             // every warp is done with the previous tile's token scales
        for (int i = ew * 32 + lane; i < c.nt; i += 32 * EPI_WARPS)
          sx_smem[i] = i < c.rows_valid ? __ldg(p.sx + c.row0 + i) : 0.0f;
        named_bar_sync(5, 32 * EPI_WARPS);
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
          if (GATEUP && p.hmax != nullptr) {
            // row maximum of |H| for the FP8 down GEMM's per-row scale: integer max on the float bits of
            // non-negative values (order-independent, hence deterministic); 4 lanes share a token row
            const __nv_bfloat162* hv = reinterpret_cast<const __nv_bfloat162*>(&val);
            float m = 0.0f;
            if (col_ok && r < n_tok) {
              #pragma unroll
              for (int x = 0; x < 4; ++x) {
                const float2 f2 = __bfloat1622float2(hv[x]);
                m = fmaxf(m, fmaxf(fabsf(f2.x), fabsf(f2.y)));
              }
            }
            m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 1));
            m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
            if ((lane & 3) == 0 && r < n_tok) atomicMax(p.hmax + c.row0 + cc * 32 + r, __float_as_uint(m));
          }
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
                float g = __uint_as_float(is_up ? other[i] : v0[j + i]);
                float u = __uint_as_float(is_up ? v1[j + i] : other[i]);
                if (FP8) {                               // dequantise: sx[token] * sw[expert, feature] (reading F4)
                  const float st = sx_smem[cc * 32 + j + i];
                  g *= st * swg;
                  u *= st * swu;
                }
                st_shared_bf16(stage_wr + (j + i) * 64, silu_mul(g, u));
              }
            }
            flush_chunk(cc);
          }
          named_bar_sync(bar_id, 64);                    // exchange buffers free for the next round
        }
      } else {
        float swf = 1.0f;                              // FP8: this thread's output channel's weight scale (reading F5)
        if (FP8) {
          const int n = c.f_tile * OUT_FEATS + feat0 + lane;
          if (n < p.N) swf = __ldg(p.sw0 + static_cast<int64_t>(c.e) * p.N + n);
        }
        #pragma unroll 1
        for (int cc = sub; cc < n_chunks; cc += 2) {
          uint32_t v[32];
          tmem_ld_32x32(taddr + cc * 32, v);
          tmem_ld_wait();
          #pragma unroll
          for (int j = 0; j < 32; j += 4) {
            float4 s4 = *reinterpret_cast<const float4*>(sc_smem + (it & 1) * BN_MAX + cc * 32 + j);   // broadcast
            if (FP8) { s4.x *= swf; s4.y *= swf; s4.z *= swf; s4.w *= swf; }
            st_shared_bf16(stage_wr + (j + 0) * 64, __uint_as_float(v[j + 0]) * s4.x);
            st_shared_bf16(stage_wr + (j + 1) * 64, __uint_as_float(v[j + 1]) * s4.y);
            st_shared_bf16(stage_wr + (j + 2) * 64, __uint_as_float(v[j + 2]) * s4.z);
            st_shared_bf16(stage_wr + (j + 3) * 64, __uint_as_float(v[j + 3]) * s4.w);
          }
          flush_chunk(cc);
        }
      }
      if (!GATEUP) sc_smem[((it + 1) & 1) * BN_MAX + ew * 32 + lane] = sc_next;
      // accumulator drained: one arrival per warp on the LEADER's tmem_empty barrier
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster_relaxed(tempty_bar(as), 0);   // relaxed: must not wait for the stores
      c = cn;
      have = have_next;
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync_all();          // the peer may still read this CTA's shared memory / signal its barriers
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc_pair(tmem_base, 512);
  }
}

Params make_params(const GemmLaunch& g) {
  Params p;
  p.offsets = g.offsets;
  p.E = g.E;
  p.K = g.K;
  p.N = g.N;
  p.out = static_cast<__nv_bfloat16*>(g.out);
  p.row_scale = g.row_scale_perm;
  p.w4d = g.w4d;
  p.sg_max = g.sg_max;
  p.tile_counter = g.tile_counter;
  p.sx = g.sx; p.sw0 = g.sw0; p.sw1 = g.sw1;
  p.hmax = g.hmax;
  return p;
}

}  // namespace

cudaError_t pair_kernels_init() {
  cudaError_t e = cudaFuncSetAttribute(pair_gemm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(pair_gemm_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(pair_gemm_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(pair_gemm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
}

cudaError_t launch_gateup_swiglu_pair(const GemmLaunch& g, cudaStream_t st) {
  launch_pdl(pair_gemm_kernel<true>, g.num_sms & ~1, 256, SMEM_BYTES, st, g.tm_act, g.w4d ? g.tm_b0_4d : g.tm_b0, g.w4d ? g.tm_b1_4d : g.tm_b1, make_params(g));
  return cudaGetLastError();
}

// FP8 gate/up: tm_act over the e4m3 rows [rows, K bytes], tm_b0 / tm_b1 over the quantised weights [E, N, K bytes]
cudaError_t launch_gateup_swiglu_pair_fp8(const GemmLaunch& g, cudaStream_t st) {
  launch_pdl(pair_gemm_kernel<true, true>, g.num_sms & ~1, 256, SMEM_BYTES, st, g.tm_act, g.tm_b0, g.tm_b1, make_params(g));
  return cudaGetLastError();
}

// FP8 down: tm_act over the e4m3 H rows [rows, K bytes], tm_b0 over the quantised W_down [E, N, K bytes] (box of 128 rows)
cudaError_t launch_down_pair_fp8(const GemmLaunch& g, cudaStream_t st) {
  launch_pdl(pair_gemm_kernel<false, true>, g.num_sms & ~1, 384, SMEM_BYTES, st, g.tm_act, g.tm_b0, g.tm_b0, make_params(g));
  return cudaGetLastError();
}

cudaError_t launch_down_pair(const GemmLaunch& g, cudaStream_t st) {
  launch_pdl(pair_gemm_kernel<false>, g.num_sms & ~1, 384, SMEM_BYTES, st, g.tm_act, g.w4d ? g.tm_b0_4d : g.tm_b0, g.w4d ? g.tm_b0_4d : g.tm_b0, make_params(g));
  return cudaGetLastError();
}

}  // namespace bg
