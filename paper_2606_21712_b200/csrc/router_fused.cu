// router_fused.cu -- steps a1-a4 and the tile-local half of a5 in ONE kernel per call (DESIGN.md §4 K1):
//
//   a1  L[t,e] = sum_j float(hidden[t,j]) * W_r[j,e] (+ b_r[e])     tcgen05, fp32-exact products
//   a2  top-k under (logit desc, expert index asc), gates = softmax over the k selected logits
//   a3  per-tile expert histogram        a5' stable rank of every (token, slot) inside its 128-token tile
//   a4  exclusive scan over tiles and experts, by the last tile to finish
// (BASELINE.json north_star "fp32 router top-k over all yielded tokens, a per-expert histogram and exclusive
// scan"; routing artefacts bit-exact given the fp32 logits.)
//
// a1 on tensor cores.  hidden is bf16 and an fp32 W_r[j,e] (24-bit significand) is EXACTLY the sum of three
// bf16 values hi + mid + lo (8 significand bits each, reading S6), so hidden * W_r = hidden * hi + hidden * mid
// + hidden * lo with every bf16 x bf16 product exact in the fp32 accumulator; only the accumulation order
// differs from a scalar fp32 loop.  (A single TF32 pass would round W_r to 10 bits and is not used.)  The three
// pieces are produced once per bg_moe_set_weights by split_wr_kernel.
//
// One CLUSTER per 128-token tile; the cluster's `nch` CTAs split K into nch contiguous chunks of k-blocks.
// nch depends on d ONLY (router_nch), never on T: the fp32 summation order of a logit is then the same
// whatever the token was combined with, so forward(concat(S1,S2)) == concat(forward(S1), forward(S2)) bit for
// bit.  Each CTA: tcgen05.mma kind::f16, M = 128 tokens, N = round_up(E,16),
// A = hidden (K-major, TMA), B = the three W_r pieces (MN-major, one 4-D TMA box per k-block), accumulator in
// TMEM.  Then, through distributed shared memory:
//   1. reduce-scatter: CTA c sends rows [r*128/nch, (r+1)*128/nch) of its partial tile to CTA r; CTA r adds the
//      nch partials in ascending chunk order (+ bias) -> the logits of its 128/nch tokens (written to HBM once);
//   2. top-k of those tokens in registers: 256 / (128/nch) adjacent lanes per token scan interleaved groups of four
//      experts keeping a sorted k-list (branch-free insertion on sortable uint32 keys); the lists are merged by k
//      rounds of a shuffle tournament;
//   3. the selected experts go to the cluster's leader, which builds the tile's [E] x 128-bit selection mask
//      (integer OR), from it every entry's stable rank inside the tile and the tile's histogram;
//   4. the last tile to finish (a global counter) scans the tile histograms into counts / offsets / per-tile
//      bases and re-arms the counters.
// No partial logits, no per-block histogram and no separate top-k / scan / rank launches touch HBM.
//
// Two forms of the same arithmetic (SEQ template flag), chosen on the host from T:
//   cluster form (above): nch CTAs per tile; used while the grid fits about one wave (small / mid T, where the
//     layer is latency-bound and K must be spread over SMs) and whenever nch accumulators do not fit in TMEM;
//   sequential form: ONE CTA per tile runs the nch chunks one after the other into nch separate TMEM
//     accumulators (nch * round_up(E,16) <= 512 columns) and adds them in the same ascending order in its
//     epilogue -- the same partial sums, hence bit-identical logits, with no cluster traffic and a quarter of
//     the CTAs; the summed rows go to shared memory and through the same top-k code (two lanes per token).
#include "kernels.h"
#include "ptx_sm100.cuh"
#include "routing_common.cuh"

namespace bg {
namespace {

constexpr int BM = ROUTE_TILE, BK = 64, UK = 16, MAX_STAGES = 6;
constexpr int A_BYTES = BM * BK * 2;             // 16 KB
constexpr int B_BLK_BYTES = 64 * BK * 2;         // 8 KB per 64 experts of one piece
// A stage = one k-block: the hidden tile ONCE plus all three W_r pieces (3 x n_blk x 8 KB) when three such
// stages fit (E <= 128), else one piece per stage (E <= 256: 4 stages of 48 KB).
constexpr int RING_BYTES = 208 * 1024;
constexpr int BAR_BYTES = 256;
constexpr int IDX_TILE_BYTES = BM * ROUTE_MAX_K * 4;     // leader: the tile's selected experts
constexpr int MASK_BYTES = ROUTE_MAX_E * 4 * 4;          // leader: [E][4] selection mask
constexpr int SMEM_BYTES = RING_BYTES + 1024 + BAR_BYTES + IDX_TILE_BYTES + MASK_BYTES;
constexpr int NUM_THREADS = 256;                 // warp 0 TMA, warp 1 MMA, warp 2 TMEM alloc, warps 4-7 epilogue
// epilogue scratch that reuses the ring once every MMA of the cluster has retired
constexpr int RECV_BYTES = BM * (ROUTE_MAX_E + 4) * 4;   // [nch][128/nch][n_mma + 4] fp32 partial rows
constexpr int SCAN_BYTES = (2 * 256 + 8) * 4;
constexpr int XPOSE_PITCH = 36;                          // floats per row of a warp's 32 x 32 transposition tile
constexpr int XPOSE_BYTES = 8 * 32 * XPOSE_PITCH * 4;    // one tile per warp
static_assert(RECV_BYTES + SCAN_BYTES + XPOSE_BYTES <= RING_BYTES, "epilogue scratch must fit in the ring");
static_assert(SMEM_BYTES <= 227 * 1024, "shared memory budget");

constexpr uint64_t ADESC_HI = umma_desc_sw128(16, 1024);
constexpr uint64_t BDESC_HI = umma_desc_sw128(B_BLK_BYTES, 1024);

// pieces: [3][d][E_ld] bf16, E_ld = round_up(E,16), zero padded (TMA needs 16-byte row strides).
__global__ void split_wr_kernel(const float* __restrict__ W_r, int d, int E, int E_ld,
                                __nv_bfloat16* __restrict__ pieces) {
  const int64_t n = static_cast<int64_t>(d) * E_ld;
  const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int j = static_cast<int>(i / E_ld), e = static_cast<int>(i - static_cast<int64_t>(j) * E_ld);
  const float w = (e < E) ? W_r[static_cast<int64_t>(j) * E + e] : 0.0f;
  const __nv_bfloat16 hi = __float2bfloat16_rn(w);
  const float r1 = w - __bfloat162float(hi);                 // exact
  const __nv_bfloat16 mid = __float2bfloat16_rn(r1);
  const float r2 = r1 - __bfloat162float(mid);               // exact
  const __nv_bfloat16 lo = __float2bfloat16_rn(r2);          // exact: <= 8 significant bits remain
  pieces[i] = hi;
  pieces[n + i] = mid;
  pieces[2 * n + i] = lo;
}

__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

struct RouterParams {
  int T, d, E, k, nch;
  const float* b_r;
  float* logits_out;        // [T,E]
  int32_t* topk_idx;        // [T,k]
  float* topk_w;            // [T,k]
  int32_t* tile_rank;       // [T,k]  stable rank of the entry among its tile's entries of the same expert
  int32_t* tile_counts;     // [n_tiles,E]
  int32_t* tile_base;       // [n_tiles,E]
  int32_t* counts;          // [E]
  int32_t* offsets;         // [E+1]
  int32_t* done_counter;    // zero on entry; the last tile re-arms it
  int32_t* gemm_counters;   // 8 ints (ticket counters of the two grouped GEMMs) zeroed by the last tile; may be null
  const void* const* seg_hidden;
  const int32_t* seg_start;
  int n_segs;
};

#ifdef BG_ROUTER_TRACE
__device__ unsigned long long g_router_trace[8 * 16];   // development builds only: globaltimer stamps of CTAs 0..7
#endif

// Sorted insertion of (x, xe) into the descending list (bk, be): after every entry that `wins` against it.
// TIE_BY_INDEX = false: entries arrive in ascending expert order, so an equal key already in the list has the
// lower index and stays ahead (strict >).  true (merging lists of different threads): equal keys order by index.
template <int KMAX, bool TIE_BY_INDEX>
__device__ __forceinline__ void klist_insert(uint32_t (&bk)[KMAX], int (&be)[KMAX], uint32_t x, int xe) {
  bool c[KMAX];
  #pragma unroll
  for (int s = 0; s < KMAX; ++s)
    c[s] = TIE_BY_INDEX ? (x > bk[s] || (x == bk[s] && xe < be[s])) : (x > bk[s]);
  #pragma unroll
  for (int s = KMAX - 1; s >= 0; --s) {
    const bool up = s > 0 && c[s - 1];           // the entry above moves down into this slot
    const uint32_t nk = up ? bk[s > 0 ? s - 1 : 0] : x;
    const int ne = up ? be[s > 0 ? s - 1 : 0] : xe;
    bk[s] = c[s] ? nk : bk[s];
    be[s] = c[s] ? ne : be[s];
  }
}

// Gates (reading S2: softmax over the k selected logits, slot 0 holds the maximum), the token's rows of
// topk_idx / topk_w, and its selected experts into the tile table `dst` (this CTA's or the leader's).
template <int KMAX, typename Store>
__device__ __forceinline__ void finish_token(const uint32_t (&bk)[KMAX], const int (&be)[KMAX], int k, int t, int T,
                                             const RouterParams& p, Store store_idx) {
  const float v0 = ordered_to_float(bk[0]);
  float ex[KMAX];
  float denom = 0.0f;
  #pragma unroll
  for (int s = 0; s < KMAX; ++s) {
    ex[s] = (s < k) ? expf(ordered_to_float(bk[s]) - v0) : 0.0f;
    denom += ex[s];                                // slot order
  }
  #pragma unroll
  for (int s = 0; s < KMAX; ++s)
    if (s < k) {
      if (t < T) {
        p.topk_idx[static_cast<int64_t>(t) * k + s] = be[s];
        p.topk_w[static_cast<int64_t>(t) * k + s] = ex[s] / denom;
      }
      store_idx(s, t < T ? be[s] : -1);
    }
}

// ROWS = false: A (hidden tile) by TMA from one contiguous [T, d] matrix (tm_h).
// ROWS = true : A rows fetched through per-row pointers (segments, zero-copy COMBINE) by the four epilogue
//               warps with 16-byte cp.async copies into the 128B-swizzled layout TMA would have produced;
//               cp.async writes through the generic proxy and tcgen05.mma reads through the async proxy, so
//               every loader thread waits for its own copies, fences the proxies, and only then arrives on
//               the stage's full barrier.
// SEQ = false : cluster form, one K chunk per CTA (cluster size = p.nch), partials reduced through DSMEM.
// SEQ = true  : sequential form, one CTA per tile, chunk c accumulates in TMEM columns [c * n_mma, (c+1) * n_mma).
template <bool ROWS, bool SEQ, int KMAX>
__global__ void __launch_bounds__(NUM_THREADS, 1)
router_fused_kernel(const __grid_constant__ CUtensorMap tm_h, const __grid_constant__ CUtensorMap tm_w,
                    const __grid_constant__ CUtensorMap tm_w1, const RouterParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (base - raw);
  const uint32_t bar_base = base + RING_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (MAX_STAGES + s); };
  const uint32_t done_bar = bar_base + 8u * (2 * MAX_STAGES);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + RING_BYTES + 8 * (2 * MAX_STAGES + 1));
  int* last_flag = reinterpret_cast<int*>(smem + RING_BYTES + 8 * (2 * MAX_STAGES + 1) + 8);
  int* idx_tile = reinterpret_cast<int*>(smem + RING_BYTES + BAR_BYTES);                       // [128][8]
  uint32_t* mask = reinterpret_cast<uint32_t*>(smem + RING_BYTES + BAR_BYTES + IDX_TILE_BYTES);   // [E][4]
  // ring reuse after the main loop
  float* recv = reinterpret_cast<float*>(smem);
  int* scan_scratch = reinterpret_cast<int*>(smem + RECV_BYTES);
  float* xpose = reinterpret_cast<float*>(smem + RECV_BYTES + SCAN_BYTES);           // [8 warps][32][XPOSE_PITCH]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int T = p.T, d = p.d, E = p.E, k = p.k;
#ifdef BG_ROUTER_TRACE
  auto trace = [&](int slot) {
    if (threadIdx.x == 128 && blockIdx.x < 8) {
      unsigned long long t;
      asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
      g_router_trace[blockIdx.x * 16 + slot] = t;
    }
  };
#else
  auto trace = [](int) {};
#endif
  trace(0);
  const int cs = SEQ ? 1 : p.nch;                            // cluster size
  const int nch = p.nch;                                     // K chunks (a function of d only)
  const uint32_t crank = SEQ ? 0u : cluster_ctarank();
  const int m_tile = blockIdx.x / cs;
  const int n_tiles = gridDim.x / cs;
  const int k_blocks = (d + BK - 1) / BK;
  const int kb_per = (k_blocks + nch - 1) / nch;             // k-blocks per chunk (every chunk has >= 1, see router_nch)
  const int kb0 = SEQ ? 0 : static_cast<int>(crank) * kb_per;
  const int kb1 = SEQ ? k_blocks : min(k_blocks, kb0 + kb_per);
  const int n_kb = max(0, kb1 - kb0);                        // k-blocks of this CTA
  const int n_mma = (E + 15) & ~15;                          // UMMA N (multiple of 16 for M=128)
  const int n_blk = (E + 63) / 64;                           // 64-expert TMA boxes
  const uint32_t piece_bytes = n_blk * B_BLK_BYTES;
  const int pps = (3 * (A_BYTES + 3 * piece_bytes) <= RING_BYTES) ? 3 : 1;     // pieces per stage
  const int ipk = 3 / pps;                                   // iterations (stages) per k-block
  const int n_iter = n_kb * ipk;
  const uint32_t stage_bytes = A_BYTES + pps * piece_bytes;
  const int n_stages = min(MAX_STAGES, RING_BYTES / static_cast<int>(stage_bytes));
  const bool w4d = (n_mma & 63) == 0;                        // 4-D block view of the pieces (api.cu)
  const uint32_t idesc = umma_idesc_bf16(BM, n_mma, 0, 1);
  const uint32_t tmem_cols = (SEQ && nch * n_mma > 256) ? 512u : 256u;

  // ---- independent of the previous kernel: barriers, TMEM
  if (warp == 0 && lane == 0) {
    if (!ROWS) tma_prefetch_desc(&tm_h);
    tma_prefetch_desc(&tm_w);
    for (int s = 0; s < MAX_STAGES; ++s) { mbar_init(full_bar(s), ROWS ? 1 + 128 : 1); mbar_init(empty_bar(s), 1); }
    mbar_init(done_bar, 1);
    fence_barrier_init();
  }
  if (warp == 2) { tmem_alloc(smem_u32(tmem_slot), tmem_cols); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait_then_trigger();
  trace(1);

  // TMA and MMA roles run warp-wide with one elected lane issuing (elect.sync): under `if (lane == 0)` ptxas wraps
  // every asm statement in an elect / branch loop.
  if (warp == 0) {                                // ---- TMA producer
    int s = 0;
    uint32_t ph = 0;
    for (int it = 0; it < n_iter; ++it) {
      mbar_wait(empty_bar(s), ph ^ 1u);
      if (elect_one()) {
        const int kb = kb0 + it / ipk, pc0 = (it % ipk) * pps;
        const uint32_t sa = base + s * stage_bytes, sb = sa + A_BYTES;
        mbar_expect_tx(full_bar(s), ROWS ? stage_bytes - A_BYTES : stage_bytes);
        if (!ROWS) tma_load_2d(sa, &tm_h, full_bar(s), kb * BK, m_tile * BM);
        if (w4d) {                                  // one operation: [piece][block][k][64 e]
          tma_load_4d(sb, pps == 3 ? &tm_w : &tm_w1, full_bar(s), 0, kb * BK, 0, pc0);
        } else {
          for (int pc = 0; pc < pps; ++pc)
            for (int j = 0; j < n_blk; ++j)
              tma_load_3d(sb + pc * piece_bytes + j * B_BLK_BYTES, &tm_w, full_bar(s), 64 * j, kb * BK, pc0 + pc);
        }
      }
      __syncwarp();
      if (++s == n_stages) { s = 0; ph ^= 1u; }
    }
  } else if (warp == 1) {                         // ---- MMA issuer
    int s = 0;
    uint32_t ph = 0;
    for (int it = 0; it < n_iter; ++it) {
      mbar_wait(full_bar(s), ph);
      tc_fence_after();
      if (elect_one()) {
        const uint32_t sa = base + s * stage_bytes, sb = sa + A_BYTES;
        const uint64_t ad = ADESC_HI | ((sa >> 4) & 0x3FFFu);
        // sequential form: chunk c = kb / kb_per owns its own accumulator, restarted at the chunk's first k-block
        const int kbl = it / ipk;                                   // k-block of this CTA
        const int chunk = SEQ ? kbl / kb_per : 0;
        const bool first = SEQ ? (kbl - chunk * kb_per == 0 && it % ipk == 0) : (it == 0);
        const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(chunk * n_mma);
        for (int pc = 0; pc < pps; ++pc) {        // hidden * hi + hidden * mid + hidden * lo, one accumulator
          const uint64_t bd = BDESC_HI | (((sb + pc * piece_bytes) >> 4) & 0x3FFFu);
          #pragma unroll
          for (int kk = 0; kk < BK / UK; ++kk)
            umma_f16(d_tmem, ad + ((kk * UK * 2) >> 4), bd + ((kk * UK * 128) >> 4), idesc,
                     (first && pc == 0 && kk == 0) ? 0u : 1u);
        }
        umma_commit(empty_bar(s));
        if (it + 1 == n_iter) umma_commit(done_bar);
      }
      __syncwarp();
      if (++s == n_stages) { s = 0; ph ^= 1u; }
    }
    if (n_iter == 0 && elect_one()) umma_commit(done_bar);
  } else if (warp >= 4) {
    if (ROWS) {                                   // ---- row loader (thread <-> one row of the 128-token tile)
      const int LAG = min(4, n_stages - 1);       // stages in flight per thread (n_stages >= 3 always)
      // Eight consecutive lanes copy the eight 16-byte chunks of one row's 128-byte k-span (one full line
      // per row); a warp instruction covers 4 rows, 8 instructions the warp's 32 rows.
      const int lw = warp - 4, sub = lane >> 3, chunk = lane & 7;
      const uint8_t* rowp[8];
      uint32_t dst_off[8];
      #pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int row = lw * 32 + j * 4 + sub;
        const int t = m_tile * BM + row;
        rowp[j] = nullptr;
        if (t < T) {
          const int sg = seg_of(p.seg_start, p.n_segs, t);
          rowp[j] = static_cast<const uint8_t*>(p.seg_hidden[sg]) +
                    static_cast<int64_t>(t - __ldg(p.seg_start + sg)) * d * 2 + chunk * 16;
        }
        dst_off[j] = row * 128 + ((chunk ^ (row & 7)) << 4);   // the 128B swizzle TMA applies
      }
      const uint8_t* dummy = static_cast<const uint8_t*>(p.seg_hidden[0]);
      int s = 0, pub_s = 0, issued = 0;
      uint32_t ph = 0;
      for (int it = 0; it < n_iter; ++it) {
        if (issued >= LAG) {                      // publish the stage issued LAG iterations ago
          if (LAG == 4) asm volatile("cp.async.wait_group 3;" ::: "memory");
          else if (LAG == 3) asm volatile("cp.async.wait_group 2;" ::: "memory");
          else asm volatile("cp.async.wait_group 1;" ::: "memory");
          fence_proxy_async();
          mbar_arrive_relaxed(full_bar(pub_s));
          if (++pub_s == n_stages) pub_s = 0;
        }
        mbar_wait(empty_bar(s), ph ^ 1u);
        const int kb = kb0 + it / ipk;
        const uint32_t sa = base + s * stage_bytes;
        const bool k_ok = kb * BK + chunk * 8 < d;          // k past d must read as zero
        #pragma unroll
        for (int j = 0; j < 8; ++j) {
          const bool ok = k_ok && rowp[j] != nullptr;
          cp_async_16(sa + dst_off[j], ok ? rowp[j] + kb * (BK * 2) : dummy, ok ? 16u : 0u);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        ++issued;
        if (++s == n_stages) { s = 0; ph ^= 1u; }
      }
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      fence_proxy_async();
      for (int i = issued > LAG ? LAG : issued; i > 0; --i) {
        mbar_arrive_relaxed(full_bar(pub_s));
        if (++pub_s == n_stages) pub_s = 0;
      }
    }
  }
  // Every warp takes part in the epilogue (the TMA / MMA / allocator warps are idle by now): two warps share
  // each TMEM lane quarter.
  __syncwarp();
  mbar_wait(done_bar, 0);                         // this CTA's accumulator(s) are complete
  tc_fence_after();
  trace(2);

  const int tid = threadIdx.x - 128;              // epilogue-group thread 0..127 (warps 4-7), used by the rank step
  const int q = warp & 3, half = warp >> 2;       // TMEM lane quarter; which half of the 32-column chunks
  const int EP = n_mma + 4;                       // row pitch (floats) of the partial / logit rows in shared memory
  const int tpc = BM / cs;                        // token rows this CTA finishes (128 in the sequential form)
  const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16);
  if (SEQ) {
    // ===================== sequential form: the nch accumulators added in chunk order, rows to shared memory ====
    const int row = q * 32 + lane;                // (every warp has seen done_bar: the ring is free)
    for (int c0 = half * 32; c0 < n_mma; c0 += 64) {
      uint32_t v[32];
      tmem_ld_32x32(taddr + c0, v);               // chunk 0
      tmem_ld_wait();
      for (int c = 1; c < nch; ++c) {             // + chunk c, ascending: the cluster form's summation order
        uint32_t u[32];
        tmem_ld_32x32(taddr + c * n_mma + c0, u);
        tmem_ld_wait();
        #pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(u[j]));
      }
      #pragma unroll
      for (int j = 0; j < 32; j += 4)
        if (c0 + j < n_mma)
          *reinterpret_cast<uint4*>(recv + row * EP + c0 + j) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
    }
    tc_fence_before();
    for (int i = threadIdx.x; i < ROUTE_MAX_E * 4; i += NUM_THREADS) mask[i] = 0u;
    __syncthreads();
  } else {
    // ===================== cluster form: reduce-scatter over the cluster =====================
    // (A) every CTA of the cluster has retired its MMAs: the rings may be overwritten by peers
    __syncthreads();
    cluster_sync_all();
    trace(3);

    // ---- 1. partial rows to their owners through distributed shared memory.  A thread owns a token row in
    // TMEM, but remote stores must be coalesced (scattered 16-byte stores run at a few percent of the DSMEM
    // bandwidth): each warp turns 32 rows x 32 columns around in a private tile and sends 128-byte row pieces.
    {
      float* tile = xpose + warp * 32 * XPOSE_PITCH;
      const int sub = lane >> 3, cc = (lane & 7) * 4;
      for (int c0 = half * 32; c0 < n_mma; c0 += 64) {
        uint32_t v[32];
        tmem_ld_32x32(taddr + c0, v);             // columns past n_mma are allocated but unused
        tmem_ld_wait();
        #pragma unroll
        for (int j = 0; j < 32; j += 4)
          *reinterpret_cast<uint4*>(tile + lane * XPOSE_PITCH + j) =
              n_kb > 0 ? make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]) : make_uint4(0u, 0u, 0u, 0u);
        __syncwarp();
        if (c0 + cc < n_mma) {
          #pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int r = i * 4 + sub, row = q * 32 + r;
            const int owner = row / tpc, tl = row - owner * tpc;
            const uint4 x = *reinterpret_cast<const uint4*>(tile + r * XPOSE_PITCH + cc);
            const uint32_t dst = mapa_shared(
                base + static_cast<uint32_t>((static_cast<int>(crank) * tpc + tl) * EP + c0 + cc) * 4u,
                static_cast<uint32_t>(owner));
            st_shared_cluster_v4(dst, x.x, x.y, x.z, x.w);
          }
        }
        __syncwarp();
      }
      tc_fence_before();
      trace(4);
    }
    if (crank == 0)
      for (int i = threadIdx.x; i < ROUTE_MAX_E * 4; i += NUM_THREADS) mask[i] = 0u;
    // (B) all partial rows have arrived
    __syncthreads();
    cluster_sync_all();
    trace(5);
  }

  // ===================== logits + top-k of this CTA's tpc tokens, P = 256 / tpc threads per token ==========
  // Thread (tl, part): lanes of one token are adjacent.  It adds the partial rows of experts 4g .. 4g+3,
  // g = part, part + P, ... in ascending chunk order (+ bias), writes those logits, and keeps a sorted k-list
  // (branch-free insertion, ascending expert order inside the thread).  The P lists of a token are then merged
  // by k rounds of a shuffle tournament under the order of reading S3 (key desc, expert index asc).
  {
    const int P = NUM_THREADS / tpc;              // 2 (sequential form) .. 16 (cluster of 8): a power of two
    const int tl = threadIdx.x / P, part = threadIdx.x - tl * P;
    const int row = static_cast<int>(crank) * tpc + tl;        // row of the 128-token tile
    const int t = m_tile * BM + row;
    const int n_sum = SEQ ? 1 : cs;               // partial rows to add (the sequential form added in registers)
    uint32_t bk[KMAX];
    int be[KMAX];
    #pragma unroll
    for (int s = 0; s < KMAX; ++s) { bk[s] = 0u; be[s] = 0x7fffffff; }
    const bool vec_ok = (E & 3) == 0;
    for (int e0 = part * 4; e0 < E; e0 += P * 4) {
      float4 v = *reinterpret_cast<const float4*>(recv + tl * EP + e0);
      for (int c = 1; c < n_sum; ++c) {
        const float4 u = *reinterpret_cast<const float4*>(recv + (c * tpc + tl) * EP + e0);
        v.x += u.x; v.y += u.y; v.z += u.z; v.w += u.w;
      }
      float x[4] = {v.x, v.y, v.z, v.w};
      #pragma unroll
      for (int j = 0; j < 4; ++j)
        if (e0 + j < E) {
          if (p.b_r != nullptr) x[j] += __ldg(p.b_r + e0 + j);
          klist_insert<KMAX, false>(bk, be, float_to_ordered(x[j]), e0 + j);
        }
      if (t < T) {
        float* lrow = p.logits_out + static_cast<int64_t>(t) * E + e0;
        if (vec_ok) {
          *reinterpret_cast<float4*>(lrow) = make_float4(x[0], x[1], x[2], x[3]);
        } else {
          #pragma unroll
          for (int j = 0; j < 4; ++j)
            if (e0 + j < E) lrow[j] = x[j];
        }
      }
    }
    trace(6);
    // tournament: each round every lane offers the head of its list; the winner's owner pops it
    uint32_t rk[KMAX];
    int re[KMAX];
    #pragma unroll
    for (int s = 0; s < KMAX; ++s) {
      uint32_t hk = bk[0];
      int he = be[0];
      for (int o = 1; o < P; o <<= 1) {
        const uint32_t ok = __shfl_xor_sync(0xffffffffu, hk, o);
        const int oe = __shfl_xor_sync(0xffffffffu, he, o);
        if (ok > hk || (ok == hk && oe < he)) { hk = ok; he = oe; }
      }
      rk[s] = hk;
      re[s] = he;
      if (he == be[0]) {                           // expert indices are unique: this lane owns the winner
        #pragma unroll
        for (int i = 0; i + 1 < KMAX; ++i) { bk[i] = bk[i + 1]; be[i] = be[i + 1]; }
        bk[KMAX - 1] = 0u;
        be[KMAX - 1] = 0x7fffffff;
      }
    }
    trace(7);
    if (part == 0) {
      if (SEQ) {
        finish_token<KMAX>(rk, re, k, t, T, p, [&](int s, int e) { idx_tile[row * ROUTE_MAX_K + s] = e; });
      } else {
        const uint32_t lead = mapa_shared(smem_u32(idx_tile) + static_cast<uint32_t>(row * ROUTE_MAX_K) * 4u, 0u);
        finish_token<KMAX>(rk, re, k, t, T, p,
                           [&](int s, int e) { st_shared_cluster_u32_addr(lead + s * 4, static_cast<uint32_t>(e)); });
      }
    }
    trace(8);
  }
  // (C) the tile's selected experts are in idx_tile (of the leader, in the cluster form)
  __syncthreads();
  if (!SEQ) cluster_sync_all();
  trace(9);

  if (crank == 0) {
    if (warp >= 4) {
      // ---- 3. tile-local stable rank + histogram (thread <-> token row)
      const int row = tid, t = m_tile * BM + row;
      int e[ROUTE_MAX_K], rk[ROUTE_MAX_K];
      #pragma unroll
      for (int s = 0; s < ROUTE_MAX_K; ++s) e[s] = (s < k) ? idx_tile[row * ROUTE_MAX_K + s] : -1;
      tile_rank_and_counts(mask, row, e, k, E, rk, p.tile_counts + static_cast<int64_t>(m_tile) * E, tid,
                           [] { named_bar_sync(1, 128); });
      #pragma unroll
      for (int s = 0; s < ROUTE_MAX_K; ++s)
        if (s < k && e[s] >= 0) p.tile_rank[static_cast<int64_t>(t) * k + s] = rk[s];
      __threadfence();
      trace(10);
    }
    __syncthreads();
    if (threadIdx.x == 0) *last_flag = (atomicAdd(p.done_counter, 1) == n_tiles - 1) ? 1 : 0;
    __syncthreads();
    if (*last_flag) {
      // ---- 4. the last tile: scan over tiles and experts; re-arm the counters
      __threadfence();
      scan_tiles_block256(p.tile_counts, n_tiles, E, p.tile_base, p.counts, p.offsets, scan_scratch);
      if (threadIdx.x == 0) {
        *p.done_counter = 0;
        if (p.gemm_counters != nullptr)
          for (int i = 0; i < 8; ++i) p.gemm_counters[i] = 0;
      }
    }
  }
  trace(11);
  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, tmem_cols); }
}

template <bool ROWS, bool SEQ, int KMAX>
cudaError_t launch_one(const CUtensorMap& tm_h, const CUtensorMap& tm_w, const CUtensorMap& tm_w1,
                       const RouterParams& p, cudaStream_t st) {
  auto* kern = router_fused_kernel<ROWS, SEQ, KMAX>;
  const int n_tiles = (p.T + BM - 1) / BM;
  const int cs = SEQ ? 1 : p.nch;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(n_tiles) * cs);
  cfg.blockDim = dim3(NUM_THREADS);
  cfg.dynamicSmemBytes = SMEM_BYTES;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = cs;
  attr[1].val.clusterDim.y = 1;
  attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = SEQ ? 1 : 2;
  return cudaLaunchKernelEx(&cfg, kern, tm_h, tm_w, tm_w1, p);
}

template <bool ROWS, bool SEQ>
cudaError_t launch_k(const CUtensorMap& tm_h, const CUtensorMap& tm_w, const CUtensorMap& tm_w1,
                     const RouterParams& p, cudaStream_t st) {
  if (p.k <= 2) return launch_one<ROWS, SEQ, 2>(tm_h, tm_w, tm_w1, p, st);
  if (p.k <= 4) return launch_one<ROWS, SEQ, 4>(tm_h, tm_w, tm_w1, p, st);
  return launch_one<ROWS, SEQ, 8>(tm_h, tm_w, tm_w1, p, st);
}

template <bool ROWS, bool SEQ, int KMAX>
cudaError_t init_one() {
  return cudaFuncSetAttribute(router_fused_kernel<ROWS, SEQ, KMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              SMEM_BYTES);
}
template <bool ROWS, bool SEQ>
cudaError_t init_k() {
  cudaError_t e;
  if ((e = init_one<ROWS, SEQ, 2>()) != cudaSuccess) return e;
  if ((e = init_one<ROWS, SEQ, 4>()) != cudaSuccess) return e;
  return init_one<ROWS, SEQ, 8>();
}

}  // namespace

cudaError_t router_kernels_init() {
  cudaError_t e;
  if ((e = init_k<false, false>()) != cudaSuccess) return e;
  if ((e = init_k<false, true>()) != cudaSuccess) return e;
  if ((e = init_k<true, false>()) != cudaSuccess) return e;
  return init_k<true, true>();
}

#ifdef BG_ROUTER_TRACE
extern "C" int bg_moe_debug_router_trace(unsigned long long* out) {
  return cudaMemcpyFromSymbol(out, g_router_trace, sizeof(g_router_trace)) == cudaSuccess ? 0 : -3;
}
#endif

cudaError_t launch_split_wr(const float* W_r, int d, int E, void* pieces, cudaStream_t st) {
  const int E_ld = (E + 15) & ~15;
  const int64_t n = static_cast<int64_t>(d) * E_ld;
  split_wr_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, st>>>(W_r, d, E, E_ld,
                                                                          static_cast<__nv_bfloat16*>(pieces));
  return cudaGetLastError();
}

// K chunks (= cluster size) of the router: a function of d ONLY, so that the summation order of a logit never
// depends on the combined-batch size.  Every chunk holds at least one k-block.
int router_nch(int d) {
  const int k_blocks = (d + BK - 1) / BK;
  // At most 4 chunks: with 8 (tried for d >= 6144) a tile's cluster is 8 CTAs and T = 8192 runs 3.5 waves of them, each
  // paying the cluster's two DSMEM barriers and the reduce-scatter for 14 k-blocks of work.  Measured at d = 7168, E = 256
  // (one call, alternating builds): route() 160 -> 112 us at T = 8192, 90 -> 55 us at T = 4096, 59 -> 48 us at T = 2048, and
  // 30 -> 42 us at T <= 1024, where a layer of that width spends milliseconds streaming its expert weights.
  if (k_blocks >= 32) return 4;
  if (k_blocks >= 16) return 2;
  return 1;
}

// Which form runs (both give the same bits): the sequential form needs nch accumulators in TMEM; it is used when
// there is only one chunk anyway, or when the cluster form's grid would exceed about one wave of the machine
// (then K need not be spread over SMs and a quarter of the CTAs do without the cluster traffic).
bool router_sequential(int T, int d, int E, int num_sms) {
  const int nch = router_nch(d);
  if (nch == 1) return true;
  const int n_mma = (E + 15) & ~15;
  if (nch * n_mma > 512) return false;
  const int n_tiles = (T + BM - 1) / BM;
  return n_tiles * nch > num_sms + num_sms / 4;
}

cudaError_t launch_router_fused(const CUtensorMap* tm_h, const CUtensorMap& tm_w, const CUtensorMap& tm_w1,
                                const RouterLaunch& r, const SegTable* seg, cudaStream_t st) {
  if (r.T == 0) return cudaSuccess;
  RouterParams p;
  p.T = r.T; p.d = r.d; p.E = r.E; p.k = r.k; p.nch = router_nch(r.d);
  p.b_r = r.b_r;
  p.logits_out = r.logits_out;
  p.topk_idx = r.topk_idx; p.topk_w = r.topk_w;
  p.tile_rank = r.tile_rank; p.tile_counts = r.tile_counts; p.tile_base = r.tile_base;
  p.counts = r.counts; p.offsets = r.offsets;
  p.done_counter = r.done_counter; p.gemm_counters = r.gemm_counters;
  p.seg_hidden = seg ? seg->hidden : nullptr;
  p.seg_start = seg ? seg->start : nullptr;
  p.n_segs = seg ? seg->n : 0;
  const bool seq = r.force_form == 0 ? router_sequential(r.T, r.d, r.E, r.num_sms)
                                     : (r.force_form == 1 && (p.nch * ((r.E + 15) & ~15) <= 512 || p.nch == 1));
  if (seg != nullptr) return seq ? launch_k<true, true>(tm_w, tm_w, tm_w1, p, st) : launch_k<true, false>(tm_w, tm_w, tm_w1, p, st);
  return seq ? launch_k<false, true>(*tm_h, tm_w, tm_w1, p, st) : launch_k<false, false>(*tm_h, tm_w, tm_w1, p, st);
}

}  // namespace bg
