// router_gemm.cu -- step a1 (router logits) on tensor cores with fp32-exact products.
//
//   L[t,e] = sum_j float(hidden[t,j]) * W_r[j,e]            (BASELINE.json north_star "fp32 router")
//
// hidden is bf16 and an fp32 W_r[j,e] (24-bit significand) is EXACTLY the sum of three bf16 values
// hi + mid + lo (8 significand bits each, reading S6), so
//   hidden * W_r = hidden * hi + hidden * mid + hidden * lo
// with every bf16 x bf16 product exact in the fp32 accumulator; only the accumulation order
// differs from a scalar fp32 loop.  (A single TF32 pass would round W_r to 10 bits and is not used.)
// The three pieces are produced once per bg_moe_set_weights by split_wr_kernel.
//
// Kernel: one CTA per (128-token tile, k-split).  tcgen05.mma kind::f16, M=128, N=round_up(E,16),
// A = hidden [T,d] (K-major, TMA box {64 k,128 rows}), B = pieces [3,d,E_ld] (MN-major, TMA boxes
// {64 n, 64 k, 1}); the pipeline iterates over (k-block, piece).  Split-K keeps the SMs busy when
// T/128 < #SMs: CTA (m, s) writes its fp32 partial tile to partial[s][T][E]; the top-k kernel adds
// the partials in ascending s (a fixed order => bitwise deterministic logits) plus the bias.
#include "kernels.h"
#include "ptx_sm100.cuh"

namespace bg {
namespace {

constexpr int BM = 128, BK = 64, UK = 16, MAX_STAGES = 6;
constexpr int A_BYTES = BM * BK * 2;             // 16 KB
constexpr int B_BLK_BYTES = 64 * BK * 2;         // 8 KB per 64 experts of one piece
// A stage = one k-block: the hidden tile ONCE plus all three W_r pieces (3 x n_blk x 8 KB); the number
// of stages is what fits in RING_BYTES (E <= 64: 5, E <= 128: 3, E <= 256: 2).  The hidden stream comes
// from HBM, so what matters is k-blocks of hidden in flight (one stage per (k-block, piece) re-fetched
// the hidden tile three times and kept 1.3 k-blocks in flight: 25 % of the HBM roofline on C5).
constexpr int RING_BYTES = 224 * 1024;
constexpr int SMEM_BYTES = RING_BYTES + 1024 + 256;
constexpr int NUM_THREADS = 256;                 // warp 0 TMA, warp 1 MMA, warp 2 TMEM alloc, warps 4-7 epilogue

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

// ROWS = false: A (hidden tile) by TMA from one contiguous [T, d] matrix (tm_h).
// ROWS = true : A rows fetched through per-row pointers (segments) by the four epilogue warps with 16-byte
//               cp.async copies into the 128B-swizzled layout TMA would have produced; cp.async writes
//               through the generic proxy and tcgen05.mma reads through the async proxy, so every loader
//               thread waits for its own copies (two stages behind the one it issues), fences the proxies,
//               and only then arrives on the stage's full barrier.
template <bool ROWS>
__global__ void __launch_bounds__(NUM_THREADS, 1)
router_gemm_kernel(const __grid_constant__ CUtensorMap tm_h, const __grid_constant__ CUtensorMap tm_w,
                   const __grid_constant__ CUtensorMap tm_w1, int T, int d,
                   int E, int ksplit, float* __restrict__ partial, int32_t* __restrict__ zero_buf, int zero_n,
                   const void* const* __restrict__ seg_hidden, const int32_t* __restrict__ seg_start, int n_segs) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (base - raw);
  const uint32_t bar_base = base + RING_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (MAX_STAGES + s); };
  const uint32_t done_bar = bar_base + 8u * (2 * MAX_STAGES);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + RING_BYTES + 8 * (2 * MAX_STAGES + 1));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_tile = blockIdx.x, ks = blockIdx.y;
  pdl_wait_then_trigger();
  {  // zero the per-block expert histogram that the top-k kernel (next in the stream) accumulates into
    const int n_cta = gridDim.x * gridDim.y, cta = blockIdx.y * gridDim.x + blockIdx.x;
    const int per = (zero_n + n_cta - 1) / n_cta;
    const int z0 = cta * per, z1 = min(zero_n, z0 + per);
    for (int i = z0 + threadIdx.x; i < z1; i += NUM_THREADS) zero_buf[i] = 0;
  }
  const int k_blocks = (d + BK - 1) / BK;
  const int kb_per = (k_blocks + ksplit - 1) / ksplit;
  const int kb0 = ks * kb_per, kb1 = min(k_blocks, kb0 + kb_per);
  const int n_kb = max(0, kb1 - kb0);                        // k-blocks of this CTA
  const int n_mma = (E + 15) & ~15;                          // UMMA N (multiple of 16 for M=128)
  const int n_blk = (E + 63) / 64;                           // 64-expert TMA boxes
  const uint32_t piece_bytes = n_blk * B_BLK_BYTES;
  // pieces per stage: all three when at least three such stages fit (E <= 128), else one (E <= 256:
  // 4 stages of 48 KB, the hidden tile re-fetched per piece from L2)
  const int pps = (3 * (A_BYTES + 3 * piece_bytes) <= RING_BYTES) ? 3 : 1;
  const int ipk = 3 / pps;                                   // iterations (stages) per k-block
  const int n_iter = n_kb * ipk;
  const uint32_t stage_bytes = A_BYTES + pps * piece_bytes;
  const int n_stages = min(MAX_STAGES, RING_BYTES / static_cast<int>(stage_bytes));
  const bool w4d = (n_mma & 63) == 0;                        // 4-D block view of the pieces (api.cu)
  const uint32_t idesc = umma_idesc_bf16(BM, n_mma, 0, 1);

  if (warp == 0 && lane == 0) {
    if (!ROWS) tma_prefetch_desc(&tm_h);
    tma_prefetch_desc(&tm_w);
    for (int s = 0; s < MAX_STAGES; ++s) { mbar_init(full_bar(s), ROWS ? 1 + 128 : 1); mbar_init(empty_bar(s), 1); }
    mbar_init(done_bar, 1);
    fence_barrier_init();
  }
  if (warp == 2) { tmem_alloc(smem_u32(tmem_slot), 256); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {                              // ---- TMA producer
      int s = 0;
      uint32_t ph = 0;
      for (int it = 0; it < n_iter; ++it) {
        mbar_wait(empty_bar(s), ph ^ 1u);
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
        if (++s == n_stages) { s = 0; ph ^= 1u; }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {                              // ---- MMA issuer
      int s = 0;
      uint32_t ph = 0;
      for (int it = 0; it < n_iter; ++it) {
        mbar_wait(full_bar(s), ph);
        tc_fence_after();
        const uint32_t sa = base + s * stage_bytes, sb = sa + A_BYTES;
        const uint64_t ad = ADESC_HI | ((sa >> 4) & 0x3FFFu);
        for (int pc = 0; pc < pps; ++pc) {        // hidden * hi + hidden * mid + hidden * lo, one accumulator
          const uint64_t bd = BDESC_HI | (((sb + pc * piece_bytes) >> 4) & 0x3FFFu);
          #pragma unroll
          for (int kk = 0; kk < BK / UK; ++kk)
            umma_f16(tmem_base, ad + ((kk * UK * 2) >> 4), bd + ((kk * UK * 128) >> 4), idesc,
                     (it | pc | kk) != 0 ? 1u : 0u);
        }
        umma_commit(empty_bar(s));
        if (++s == n_stages) { s = 0; ph ^= 1u; }
      }
      umma_commit(done_bar);
    }
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
          const int sg = seg_of(seg_start, n_segs, t);
          rowp[j] = static_cast<const uint8_t*>(seg_hidden[sg]) + static_cast<int64_t>(t - __ldg(seg_start + sg)) * d * 2 +
                    chunk * 16;
        }
        dst_off[j] = row * 128 + ((chunk ^ (row & 7)) << 4);   // the 128B swizzle TMA applies
      }
      const uint8_t* dummy = static_cast<const uint8_t*>(seg_hidden[0]);
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
    const int q = warp & 3;                       // TMEM lane quarter of this warp
    const int row = m_tile * BM + q * 32 + lane;
    float* dst = partial + (static_cast<int64_t>(ks) * T + row) * E;
    if (n_kb == 0) {
      if (row < T) for (int e = 0; e < E; ++e) dst[e] = 0.0f;
    } else {
      mbar_wait(done_bar, 0);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16);
      for (int c0 = 0; c0 < n_mma; c0 += 32) {
        uint32_t v[32];
        tmem_ld_32x32(taddr + c0, v);             // columns past n_mma are never used below
        tmem_ld_wait();
        if (row < T) {
          if ((E & 3) == 0) {
            #pragma unroll
            for (int j = 0; j < 32; j += 4)
              if (c0 + j + 4 <= E)
                *reinterpret_cast<float4*>(dst + c0 + j) =
                    make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]),
                                __uint_as_float(v[j + 3]));
          } else {
            #pragma unroll
            for (int j = 0; j < 32; ++j)
              if (c0 + j < E) dst[c0 + j] = __uint_as_float(v[j]);
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, 256); }
}

}  // namespace

cudaError_t router_kernels_init() {
  cudaError_t e = cudaFuncSetAttribute(router_gemm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(router_gemm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
}

cudaError_t launch_split_wr(const float* W_r, int d, int E, void* pieces, cudaStream_t st) {
  const int E_ld = (E + 15) & ~15;
  const int64_t n = static_cast<int64_t>(d) * E_ld;
  split_wr_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, st>>>(W_r, d, E, E_ld,
                                                                          static_cast<__nv_bfloat16*>(pieces));
  return cudaGetLastError();
}

int router_ksplit(int T, int d, int num_sms) {
  const int m_tiles = (T + BM - 1) / BM;
  const int k_blocks = (d + BK - 1) / BK;
  int ks = num_sms / (m_tiles > 0 ? m_tiles : 1);
  if (ks > 8) ks = 8;
  if (ks > k_blocks) ks = k_blocks;
  if (ks < 1) ks = 1;
  return ks;
}

cudaError_t launch_router_gemm(const CUtensorMap& tm_h, const CUtensorMap& tm_w, const CUtensorMap& tm_w1, int T, int d, int E, int ksplit,
                               float* partial, int32_t* zero_buf, int zero_n, cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  dim3 grid((T + BM - 1) / BM, ksplit);
  launch_pdl(router_gemm_kernel<false>, grid, NUM_THREADS, SMEM_BYTES, st, tm_h, tm_w, tm_w1, T, d, E, ksplit, partial,
             zero_buf, zero_n, static_cast<const void* const*>(nullptr), static_cast<const int32_t*>(nullptr), 0);
  return cudaGetLastError();
}

cudaError_t launch_router_gemm_segments(const SegTable& seg, const CUtensorMap& tm_w, const CUtensorMap& tm_w1, int T,
                                        int d, int E, int ksplit, float* partial, int32_t* zero_buf, int zero_n,
                                        cudaStream_t st) {
  if (T == 0) return cudaSuccess;
  dim3 grid((T + BM - 1) / BM, ksplit);
  launch_pdl(router_gemm_kernel<true>, grid, NUM_THREADS, SMEM_BYTES, st, tm_w, tm_w, tm_w1, T, d, E, ksplit, partial,
             zero_buf, zero_n, seg.hidden, seg.start, seg.n);
  return cudaGetLastError();
}

}  // namespace bg
