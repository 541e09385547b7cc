// api.cu -- the C ABI declared in include/bg_moe.h: argument validation, workspace, TMA tensor-map
// encoding and kernel sequencing.  No arithmetic of the layer happens on the host.
#include "../../include/bg_moe.h"
#include "kernels.h"

#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

struct bg_moe_ctx {
  bg_moe_config cfg;
  int num_sms = 0;
  // borrowed parameters
  const float* W_r = nullptr;
  const float* b_r = nullptr;
  const void* W_gate = nullptr;
  const void* W_up = nullptr;
  const void* W_down = nullptr;
  // workspace (one allocation)
  uint8_t* ws = nullptr;
  int64_t ws_bytes = 0;
  float* logits = nullptr;
  void* wr_pieces = nullptr;    // bf16 [3][d][round_up(E,16)]: exact hi/mid/lo split of W_r
  int32_t* topk_idx = nullptr;
  float* topk_w = nullptr;
  int32_t* counts = nullptr;
  int32_t* offsets = nullptr;
  int32_t* tile_counts = nullptr;   // [n_tiles][E] per-128-token-tile expert histograms
  int32_t* tile_base = nullptr;     // [n_tiles][E] first row of tile's entries inside each expert
  int32_t* tile_rank = nullptr;     // [R] stable rank of an entry among its tile's entries of the same expert
  int32_t* row_src = nullptr;
  int32_t* inv_perm = nullptr;
  float* w_perm = nullptr;      // gate weights in expert order (fused path)
  int32_t* tile_counters = nullptr;   // [0..3], [4..7]: hot tickets / cold tickets / clusters finished of the two pair GEMMs; [8]: router tiles done
  bool counters_dirty = false;  // a call failed after launching: re-zero the counters before the next launch
  bool dyn_sched = true;        // dynamic tile feed of the pair GEMMs (bg_moe_set_debug: static = tile t -> cluster t mod 74)
  // segment table of bg_moe_combined_forward_segments (device arrays + pageable host staging)
  int32_t max_segments = 0;
  const void** seg_dev_hidden = nullptr;
  void** seg_dev_out = nullptr;
  int32_t* seg_dev_start = nullptr;
  std::vector<uint8_t> seg_host_img;     // packed host image of the three device arrays
  void* x_perm = nullptr;
  void* H = nullptr;
  void* Y = nullptr;
  // host-pointer entry point: two staging slots and the context's own copy / compute streams
  void* hidden_dev[2] = {nullptr, nullptr};
  void* out_dev[2] = {nullptr, nullptr};
  cudaStream_t st_in = nullptr, st_compute = nullptr, st_out = nullptr;
  cudaEvent_t ev_h2d[2] = {}, ev_compute[2] = {}, ev_d2h[2] = {};
  cudaEvent_t ev_device_call = nullptr;   // recorded after every device-pointer call (orders host calls after them)
  bool device_call_pending = false;       // a device-pointer call was made since the last host call
  bool host_call_pending = false;         // a host call was made since the last device-pointer call
  int host_slot = 0;
  int64_t host_calls = 0;
  // weight tensor maps (encoded in set_weights)
  CUtensorMap tm_wr, tm_wr1;    // W_r pieces; tm_wr1: one-piece box of the 4-D view (E > 128)
  // expert-weight tensor maps: [0] = the resident tensors, [1], [2] = the two halves of the ring (offloaded weights)
  struct WeightMaps {
    CUtensorMap wg, wu, wd;      // [E', K, N] boxes {64, 64, 1}
    CUtensorMap wg4, wu4, wd4;   // 4-D block views (kernels.h GemmLaunch), valid when f % 64 == 0 / d % 64 == 0
  } wm[3];
  // FP8 gate/up (bg_moe_set_precision; readings F1-F4): quantised weights [E, f, d] bytes + per-channel scales,
  // the quantised expert-order rows + per-row scales, and their tensor maps
  int precision = 0;                  // 0 = bf16, 1 = FP8 gate/up, 2 = FP8 gate/up + down
  uint8_t* fp8_buf = nullptr;         // one set-up time allocation
  uint8_t* q_gate = nullptr;
  uint8_t* q_up = nullptr;
  float* sw_gate = nullptr;
  float* sw_up = nullptr;
  uint8_t* xq_perm = nullptr;
  float* sx_perm = nullptr;
  CUtensorMap tm_qg, tm_qu;
  bg::ActMaps am_xq;
  // precision 2 (reading F5): quantised W_down [E, d, f] + scales, quantised H rows + row factors
  uint8_t* q_down = nullptr;
  float* sw_down = nullptr;
  uint8_t* hq = nullptr;
  unsigned* hmax = nullptr;
  float* sh_perm = nullptr;
  float* sc_perm = nullptr;
  CUtensorMap tm_qd;
  bg::ActMaps am_hq;
  // expert-weight ring buffer (bg_moe_set_weights_offloaded; "ring parameter buffer")
  const uint8_t* host_wg = nullptr;   // HOST (pinned) [E,d,f], [E,d,f], [E,f,d] bf16
  const uint8_t* host_wu = nullptr;
  const uint8_t* host_wd = nullptr;
  uint8_t* ring = nullptr;            // device: 2 halves x ring_chunk experts x (W_gate | W_up | W_down)
  int ring_chunk = 0;                 // experts per half (0 = weights are resident)
  size_t ring_bytes = 0;              // size of the `ring` allocation
  cudaStream_t st_ring = nullptr;
  cudaEvent_t ev_ring_ready[2] = {}, ev_ring_free[2] = {};
  bool ring_used[2] = {false, false};
  int64_t ring_h2d_bytes = 0;         // bytes copied host -> ring by the last forward
  // bg_moe_set_ring_skip_empty: this call's expert counts are read back (pinned, event-ordered on st_ring) and only
  // experts that received rows are copied into the ring
  bool ring_skip_empty = false;
  int32_t* counts_host = nullptr;     // pinned [E]
  cudaEvent_t ev_router_done = nullptr, ev_counts = nullptr;
  // activation tensor maps of the workspace x_perm / H (whole capacity: rows past T*k are never stored)
  bg::ActMaps am_x, am_h;
  int sg_max = 0;               // bg_moe_set_debug: overrides the pair kernel's super-group size (tests)
  int router_form = 0;          // bg_moe_set_debug: 0 = by T, 1 = sequential, 2 = cluster
  int64_t launches = 0;
  std::string last_error;
  // optional per-kernel timing of the fused chain
  bool profile = false;
  bool profile_valid = false;
  cudaEvent_t ev[BG_MOE_NUM_STAGES + 1] = {};
};

namespace {

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn == nullptr) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// [rows, K] bf16 row-major, box {64 k, box_rows rows}, 128B swizzle.
bool encode_act_map(CUtensorMap* tm, const void* ptr, int64_t rows, int64_t K, int box_rows = 128) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(rows)};
  cuuint64_t strides[1] = {static_cast<cuuint64_t>(K) * 2};
  cuuint32_t box[2] = {64, static_cast<cuuint32_t>(box_rows)};
  cuuint32_t estr[2] = {1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// The sixteen activation maps of the grouped GEMMs (box rows 8, 16, ..., 128).
bool encode_act_maps(bg::ActMaps* am, const void* ptr, int64_t rows, int64_t K) {
  for (int i = 0; i < 16; ++i)
    if (!encode_act_map(&am->m[i], ptr, rows, K, 8 * (i + 1))) return false;
  return true;
}

// [E, K, N] bf16 viewed as [E, N/64, K, 64] (N % 64 == 0), box {64 n, 64 k, nblk blocks, 1 expert}, 128B swizzle.
bool encode_weight_map_4d(CUtensorMap* tm, const void* ptr, int64_t E, int64_t K, int64_t N, int nblk) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[4] = {64, static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(N / 64), static_cast<cuuint64_t>(E)};
  cuuint64_t strides[3] = {static_cast<cuuint64_t>(N) * 2, 128, static_cast<cuuint64_t>(N) * K * 2};
  cuuint32_t box[4] = {64, 64, static_cast<cuuint32_t>(nblk), 1};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// [E, K, N] bf16 row-major (N contiguous), box {64 n, 64 k, 1 expert}, 128B swizzle.
bool encode_weight_map(CUtensorMap* tm, const void* ptr, int64_t E, int64_t K, int64_t N) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {static_cast<cuuint64_t>(N), static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(E)};
  cuuint64_t strides[2] = {static_cast<cuuint64_t>(N) * 2, static_cast<cuuint64_t>(N) * K * 2};
  cuuint32_t box[3] = {64, 64, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// e4m3 bytes [rows, K] row-major, box {128 k, box_rows rows}, 128B swizzle.
bool encode_act_map_u8(CUtensorMap* tm, const void* ptr, int64_t rows, int64_t K, int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(rows)};
  cuuint64_t strides[1] = {static_cast<cuuint64_t>(K)};
  cuuint32_t box[2] = {128, static_cast<cuuint32_t>(box_rows)};
  cuuint32_t estr[2] = {1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// quantised weights [E, N, K] e4m3 bytes (k contiguous), box {128 k, 64 n, 1 expert}, 128B swizzle.
bool encode_weight_map_u8(CUtensorMap* tm, const void* ptr, int64_t E, int64_t N, int64_t K, int box_rows = 64) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(N), static_cast<cuuint64_t>(E)};
  cuuint64_t strides[2] = {static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(N) * K};
  cuuint32_t box[3] = {128, static_cast<cuuint32_t>(box_rows), 1};
  cuuint32_t estr[3] = {1, 1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline void mark(bg_moe_ctx* ctx, int i, cudaStream_t st) {
  if (ctx->profile) cudaEventRecord(ctx->ev[i], st);
}

int cuda_fail(bg_moe_ctx* ctx, cudaError_t e, const char* where) {
  if (ctx) {
    ctx->last_error = std::string(where) + ": " + cudaGetErrorString(e);
    ctx->counters_dirty = true;     // a chain may have stopped half-way: the ticket / done counters are suspect
  }
  return BG_ERR_CUDA;
}

#define BG_CUDA(ctx, call, where)                          \
  do {                                                     \
    cudaError_t e__ = (call);                              \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, where); \
  } while (0)

#define BG_LAUNCH(ctx, call, where) \
  do {                              \
    BG_CUDA(ctx, call, where);      \
    (ctx)->launches += 1;           \
  } while (0)

struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

int check_T(const bg_moe_ctx* ctx, int32_t T) {
  if (ctx == nullptr) return BG_ERR_INVALID_ARG;
  if (T < 0 || T > ctx->cfg.max_tokens) return BG_ERR_INVALID_ARG;
  return BG_OK;
}

// Start of every device-pointer call that launches kernels on `st`:
//  * counters left non-zero by a call that failed half-way are re-zeroed (stream-ordered);
//  * work the host-pointer entry point still has in flight on the context's own streams is waited for.
int begin_call(bg_moe_ctx* ctx, cudaStream_t st) {
  if (ctx->counters_dirty) {
    BG_CUDA(ctx, cudaMemsetAsync(ctx->tile_counters, 0, 64, st), "memset counters");
    ctx->counters_dirty = false;
  }
  if (ctx->host_call_pending) {
    BG_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_compute[ctx->host_slot ^ 1], 0), "wait for host-path compute");
    ctx->host_call_pending = false;
  }
  return BG_OK;
}
// End of every device-pointer call: remember where the context's work ends on the caller's stream.
int end_call(bg_moe_ctx* ctx, cudaStream_t st, bool internal) {
  if (!internal) {
    BG_CUDA(ctx, cudaEventRecord(ctx->ev_device_call, st), "record device call");
    ctx->device_call_pending = true;
  }
  return BG_OK;
}

// a1-a4 on explicit buffers.
int do_route(bg_moe_ctx* ctx, const void* hidden, int32_t T, const float* logits_in, float* logits_buf,
             int32_t* topk_idx, float* topk_w, int32_t* counts, int32_t* offsets, cudaStream_t st,
             const bg::SegTable* seg = nullptr) {
  const bg_moe_config& c = ctx->cfg;
  if (logits_in == nullptr) {
    bg::RouterLaunch r;
    r.T = T; r.d = c.d; r.E = c.E; r.k = c.k;
    r.b_r = ctx->b_r;
    r.logits_out = logits_buf;
    r.topk_idx = topk_idx; r.topk_w = topk_w;
    r.tile_rank = ctx->tile_rank; r.tile_counts = ctx->tile_counts; r.tile_base = ctx->tile_base;
    r.counts = counts; r.offsets = offsets;
    r.done_counter = ctx->tile_counters + 8;
    r.gemm_counters = ctx->tile_counters;
    r.num_sms = ctx->num_sms;
    r.force_form = ctx->router_form;
    CUtensorMap tm_h;
    if (seg == nullptr && !encode_act_map(&tm_h, hidden, T, c.d)) {
      ctx->last_error = "cuTensorMapEncodeTiled(hidden) failed";
      return BG_ERR_CUDA;
    }
    BG_LAUNCH(ctx, bg::launch_router_fused(seg ? nullptr : &tm_h, ctx->tm_wr, ctx->tm_wr1, r, seg, st), "router_fused");
  } else {
    BG_LAUNCH(ctx, bg::launch_topk_tile(logits_in, T, c.E, c.k, topk_idx, topk_w, ctx->tile_rank, ctx->tile_counts, st),
              "topk_tile");
    BG_LAUNCH(ctx, bg::launch_scan(ctx->tile_counts, bg::route_num_tiles(T), c.E, ctx->tile_base, counts, offsets, st),
              "scan");
  }
  return BG_OK;
}

// offsets: [n_experts + 1] of the experts this launch covers (a slice of the layer's offsets when the weights come
// through the ring); wm: the tensor maps of those experts' weights.
int do_ffn(bg_moe_ctx* ctx, const void* x_perm, const int32_t* offsets, int32_t T, void* y,
           const float* row_scale_perm, cudaStream_t st, int mark_between = -1, int which_maps = 0, int n_experts = -1) {
  const bg_moe_config& c = ctx->cfg;
  const bg_moe_ctx::WeightMaps& wm = ctx->wm[which_maps];
  if (n_experts < 0) n_experts = c.E;
  const int64_t R = static_cast<int64_t>(T) * c.k;
  bg::GemmLaunch g1;
  if (x_perm == ctx->x_perm) {
    g1.tm_act = ctx->am_x;             // workspace maps, encoded once in bg_moe_create
  } else if (!encode_act_maps(&g1.tm_act, x_perm, R, c.d)) {
    ctx->last_error = "cuTensorMapEncodeTiled(x_perm) failed";
    return BG_ERR_CUDA;
  }
  g1.tm_b0 = wm.wg;
  g1.tm_b1 = wm.wu;
  g1.sg_max = ctx->sg_max;
  g1.tile_counter = ctx->dyn_sched ? ctx->tile_counters : nullptr;
  g1.w4d = c.f % 64 == 0;
  g1.tm_b0_4d = g1.w4d ? wm.wg4 : wm.wg;
  g1.tm_b1_4d = g1.w4d ? wm.wu4 : wm.wu;
  g1.offsets = offsets;
  g1.E = n_experts; g1.K = c.d; g1.N = c.f;
  g1.out = ctx->H;
  g1.row_scale_perm = nullptr;
  g1.num_sms = ctx->num_sms;
  const bool fp8 = ctx->precision >= 1 && x_perm == ctx->x_perm && which_maps == 0;
  if (fp8) {
    // FP8 gate/up (fused path): the gather wrote e4m3 rows + scales instead of x_perm
    g1.tm_act = ctx->am_xq;
    g1.tm_b0 = ctx->tm_qg;
    g1.tm_b1 = ctx->tm_qu;
    g1.sx = ctx->sx_perm; g1.sw0 = ctx->sw_gate; g1.sw1 = ctx->sw_up;
    g1.hmax = ctx->precision == 2 ? ctx->hmax : nullptr;
    BG_LAUNCH(ctx, bg::launch_gateup_swiglu_pair_fp8(g1, st), "gateup_swiglu_fp8");
  } else {
    BG_LAUNCH(ctx, bg::launch_gateup_swiglu_pair(g1, st), "gateup_swiglu");
  }
  if (mark_between >= 0) mark(ctx, mark_between, st);
  bg::GemmLaunch g2;
  g2.tm_act = ctx->am_h;
  g2.tm_b0 = wm.wd;
  g2.tm_b1 = wm.wd;
  g2.sg_max = ctx->sg_max;
  g2.tile_counter = ctx->dyn_sched ? ctx->tile_counters + 4 : nullptr;
  g2.w4d = c.d % 64 == 0;
  g2.tm_b0_4d = g2.w4d ? wm.wd4 : wm.wd;
  g2.tm_b1_4d = g2.tm_b0_4d;
  g2.offsets = offsets;
  g2.E = n_experts; g2.K = c.f; g2.N = c.d;
  g2.out = y;
  g2.row_scale_perm = row_scale_perm;
  g2.num_sms = ctx->num_sms;
  if (fp8 && ctx->precision == 2) {
    // FP8 down GEMM (reading F5): quantise H with its per-row scale, then W8A8 with the row factor sh * gate weight
    BG_LAUNCH(ctx, bg::launch_quantize_h(ctx->H, ctx->hmax, row_scale_perm, R, c.f, ctx->hq, ctx->sh_perm, ctx->sc_perm,
                                         ctx->num_sms, st), "quantize_h");
    g2.tm_act = ctx->am_hq;
    g2.tm_b0 = ctx->tm_qd;
    g2.row_scale_perm = ctx->sc_perm;
    g2.sw0 = ctx->sw_down;
    BG_LAUNCH(ctx, bg::launch_down_pair_fp8(g2, st), "down_fp8");
  } else {
    BG_LAUNCH(ctx, bg::launch_down_pair(g2, st), "down");
  }
  return BG_OK;
}

// Expert-weight ring buffer (§5.2, Fig. 7a "the running and prefetching expert
// using the ring buffer"; "fully overlapping parameter transfers with computation").  The expert
// weights live in pinned HOST memory; the device holds two ring halves of `ring_chunk` experts.  Chunk c of the
// experts is copied into half c & 1 on the context's copy stream while the grouped GEMMs of chunk c-1 run out of
// the other half on the caller's stream; a half is handed back to the copy engine when its GEMMs have finished
// ("the buffer slot ownership is released after the module completes execution").  The GEMM kernels are the
// resident path's: they see `ring_chunk` experts whose offsets are the matching slice of the layer's offsets, so
// every row runs through exactly the same arithmetic and the result is bit-identical.  Parameter movement is one
// way, host -> device.  By default every expert is copied (which experts are empty is only known on the device, and
// this path takes no host synchronisation either); with bg_moe_set_ring_skip_empty the call reads its own counts
// back first and copies only the experts that received rows.
int do_ffn_ring(bg_moe_ctx* ctx, int32_t T, cudaStream_t st) {
  const bg_moe_config& c = ctx->cfg;
  const int C = ctx->ring_chunk;
  const size_t gu_bytes = static_cast<size_t>(c.d) * c.f * 2;       // one expert's W_gate (= W_up = W_down) bytes
  const size_t half_bytes = 3 * gu_bytes * C;
  ctx->ring_h2d_bytes = 0;
  const bool skip = ctx->ring_skip_empty;
  if (skip)   // the ONE host synchronisation of this mode: this call's counts have landed in pinned memory
    BG_CUDA(ctx, cudaEventSynchronize(ctx->ev_counts), "wait for this call's expert counts");
  for (int e0 = 0, used = 0; e0 < c.E; e0 += C) {
    const int n = c.E - e0 < C ? c.E - e0 : C;
    if (skip) {                          // a chunk none of whose experts received a row: no copy, no GEMM launch
      bool any = false;
      for (int e = e0; e < e0 + n; ++e) any = any || ctx->counts_host[e] > 0;
      if (!any) continue;
    }
    const int h = used & 1;
    ++used;
    uint8_t* half = ctx->ring + h * half_bytes;
    if (ctx->ring_used[h]) BG_CUDA(ctx, cudaStreamWaitEvent(ctx->st_ring, ctx->ev_ring_free[h], 0), "ring half free");
    // runs of consecutive experts to copy: the whole chunk, or (skip mode) the maximal runs of non-empty experts;
    // an expert keeps its slot (e - e0) in the half either way, so the tensor maps and offsets do not change
    for (int a = 0; a < n;) {
      if (skip && ctx->counts_host[e0 + a] == 0) { ++a; continue; }
      int b = a + 1;
      while (b < n && (!skip || ctx->counts_host[e0 + b] > 0)) ++b;
      const size_t src = (e0 + a) * gu_bytes, dst = a * gu_bytes, len = (b - a) * gu_bytes;
      BG_CUDA(ctx, cudaMemcpyAsync(half + dst, ctx->host_wg + src, len, cudaMemcpyHostToDevice, ctx->st_ring),
              "H2D W_gate chunk");
      BG_CUDA(ctx, cudaMemcpyAsync(half + C * gu_bytes + dst, ctx->host_wu + src, len, cudaMemcpyHostToDevice,
                                   ctx->st_ring), "H2D W_up chunk");
      BG_CUDA(ctx, cudaMemcpyAsync(half + 2 * C * gu_bytes + dst, ctx->host_wd + src, len, cudaMemcpyHostToDevice,
                                   ctx->st_ring), "H2D W_down chunk");
      ctx->ring_h2d_bytes += 3 * static_cast<int64_t>(len);
      a = b;
    }
    BG_CUDA(ctx, cudaEventRecord(ctx->ev_ring_ready[h], ctx->st_ring), "record ring ready");
    BG_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_ring_ready[h], 0), "wait ring ready");
    int rc = do_ffn(ctx, ctx->x_perm, ctx->offsets + e0, T, ctx->Y, ctx->w_perm, st, -1, 1 + h, n);
    if (rc) return rc;
    BG_CUDA(ctx, cudaEventRecord(ctx->ev_ring_free[h], st), "record ring free");
    ctx->ring_used[h] = true;
  }
  return BG_OK;
}

// The fused chain a1-a9; seg != nullptr: token rows are read from / written to the segments' buffers.
int do_forward(bg_moe_ctx* ctx, const void* hidden, int32_t T, void* out, cudaStream_t st, const bg::SegTable* seg) {
  const bg_moe_config& c = ctx->cfg;
  mark(ctx, 0, st);
  int rc = do_route(ctx, hidden, T, nullptr, ctx->logits, ctx->topk_idx, ctx->topk_w, ctx->counts, ctx->offsets, st, seg);
  if (rc) return rc;
  if (ctx->ring_chunk != 0 && ctx->ring_skip_empty) {
    // counts are final once the router kernel has finished: bring them to the host on the ring's copy stream while
    // the gather runs on `st`
    BG_CUDA(ctx, cudaEventRecord(ctx->ev_router_done, st), "record router done");
    BG_CUDA(ctx, cudaStreamWaitEvent(ctx->st_ring, ctx->ev_router_done, 0), "ring stream waits for the router");
    BG_CUDA(ctx, cudaMemcpyAsync(ctx->counts_host, ctx->counts, sizeof(int32_t) * c.E, cudaMemcpyDeviceToHost,
                                 ctx->st_ring), "D2H counts");
    BG_CUDA(ctx, cudaEventRecord(ctx->ev_counts, ctx->st_ring), "record counts on host");
  }
  mark(ctx, 1, st);
  bg::PermLaunch pl = {ctx->topk_idx, ctx->tile_rank, ctx->tile_base, ctx->topk_w, ctx->row_src, ctx->inv_perm,
                       ctx->w_perm};
  if (ctx->precision >= 1)
    BG_LAUNCH(ctx, bg::launch_gather_fp8(hidden, pl, T, c.E, c.k, c.d, ctx->xq_perm, ctx->sx_perm,
                                         ctx->precision == 2 ? ctx->hmax : nullptr, ctx->num_sms, st, seg),
              "gather_fp8");
  else
    BG_LAUNCH(ctx, bg::launch_gather(hidden, pl, T, c.E, c.k, c.d, ctx->x_perm, ctx->num_sms, st, seg), "gather");
  mark(ctx, 2, st);
  if (ctx->ring_chunk == 0) {
    rc = do_ffn(ctx, ctx->x_perm, ctx->offsets, T, ctx->Y, ctx->w_perm, st, /*mark_between=*/3);
    if (rc) return rc;
  } else {
    rc = do_ffn_ring(ctx, T, st);
    if (rc) return rc;
    mark(ctx, 3, st);        // per-kernel profile: the whole streamed FFN is reported as "gateup_swiglu", "down" = 0
  }
  mark(ctx, 4, st);
  BG_LAUNCH(ctx, bg::launch_unpermute(ctx->Y, ctx->inv_perm, nullptr, T, c.k, c.d, out, ctx->num_sms, st, seg),
            "unpermute");
  mark(ctx, 5, st);
  ctx->profile_valid = ctx->profile;
  return BG_OK;
}

// The three expert-weight tensors [n_experts, ...] -> the six tensor maps of a WeightMaps set.
bool encode_weight_maps(bg_moe_ctx* ctx, bg_moe_ctx::WeightMaps* wm, const void* W_gate, const void* W_up,
                        const void* W_down, int n_experts) {
  const bg_moe_config& c = ctx->cfg;
  if (!encode_weight_map(&wm->wg, W_gate, n_experts, c.d, c.f) || !encode_weight_map(&wm->wu, W_up, n_experts, c.d, c.f) ||
      !encode_weight_map(&wm->wd, W_down, n_experts, c.f, c.d)) {
    ctx->last_error = "cuTensorMapEncodeTiled(weights) failed";
    return false;
  }
  // block views for the pair kernel: a7 = 1 block of 64 columns per map, a8 = 2
  if ((c.f % 64 == 0 && (!encode_weight_map_4d(&wm->wg4, W_gate, n_experts, c.d, c.f, 1) ||
                         !encode_weight_map_4d(&wm->wu4, W_up, n_experts, c.d, c.f, 1))) ||
      (c.d % 64 == 0 && !encode_weight_map_4d(&wm->wd4, W_down, n_experts, c.f, c.d, 2))) {
    ctx->last_error = "cuTensorMapEncodeTiled(weight block views) failed";
    return false;
  }
  return true;
}

// Router weights: the exact bf16 hi/mid/lo split of W_r (router_fused.cu) and its tensor maps.
int set_router_weights(bg_moe_ctx* ctx, const float* W_r, cudaStream_t st) {
  const bg_moe_config& c = ctx->cfg;
  {
    DeviceGuard guard(c.device);
    const int64_t E_ld = (c.E + 15) & ~15;
    EncodeTiledFn fn = get_encode_fn();
    CUresult res;
    if (E_ld % 64 == 0) {
      // [3][d][E_ld] viewed as [3][E_ld/64][d][64]: one box {64 e, 64 k, E_ld/64 blocks, 3 pieces} per
      // k-block lands every piece and 64-expert block in the [piece][block][k][64 e] order of the MN-major operand
      cuuint64_t dims[4] = {64, static_cast<cuuint64_t>(c.d), static_cast<cuuint64_t>(E_ld / 64), 3};
      cuuint64_t strides[3] = {static_cast<cuuint64_t>(E_ld) * 2, 128, static_cast<cuuint64_t>(E_ld) * c.d * 2};
      cuuint32_t box[4] = {64, 64, static_cast<cuuint32_t>(E_ld / 64), 3};
      cuuint32_t estr[4] = {1, 1, 1, 1};
      res = fn(&ctx->tm_wr, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, ctx->wr_pieces, dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      box[3] = 1;
      if (res == CUDA_SUCCESS)
        res = fn(&ctx->tm_wr1, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, ctx->wr_pieces, dims, strides, box, estr,
                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    } else {
      cuuint64_t dims[3] = {static_cast<cuuint64_t>(E_ld), static_cast<cuuint64_t>(c.d), 3};
      cuuint64_t strides[2] = {static_cast<cuuint64_t>(E_ld) * 2, static_cast<cuuint64_t>(E_ld) * c.d * 2};
      cuuint32_t box[3] = {64, 64, 1};
      cuuint32_t estr[3] = {1, 1, 1};
      res = fn(&ctx->tm_wr, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, ctx->wr_pieces, dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    if (E_ld % 64 != 0) ctx->tm_wr1 = ctx->tm_wr;
    if (res != CUDA_SUCCESS) {
      ctx->last_error = "cuTensorMapEncodeTiled(W_r pieces) failed";
      return BG_ERR_CUDA;
    }
    int rc = begin_call(ctx, st);      // also orders the split after host-path work that still reads the old pieces
    if (rc) return rc;
    BG_LAUNCH(ctx, bg::launch_split_wr(W_r, c.d, c.E, ctx->wr_pieces, st), "split_wr");
    rc = end_call(ctx, st, false);
    if (rc) return rc;
  }
  return BG_OK;
}

void destroy_ctx(bg_moe_ctx* ctx) {
  for (cudaEvent_t e : ctx->ev)
    if (e) cudaEventDestroy(e);
  for (int i = 0; i < 2; ++i) {
    if (ctx->ev_h2d[i]) cudaEventDestroy(ctx->ev_h2d[i]);
    if (ctx->ev_compute[i]) cudaEventDestroy(ctx->ev_compute[i]);
    if (ctx->ev_d2h[i]) cudaEventDestroy(ctx->ev_d2h[i]);
  }
  if (ctx->ev_device_call) cudaEventDestroy(ctx->ev_device_call);
  for (int i = 0; i < 2; ++i) {
    if (ctx->ev_ring_ready[i]) cudaEventDestroy(ctx->ev_ring_ready[i]);
    if (ctx->ev_ring_free[i]) cudaEventDestroy(ctx->ev_ring_free[i]);
  }
  if (ctx->ev_router_done) cudaEventDestroy(ctx->ev_router_done);
  if (ctx->ev_counts) cudaEventDestroy(ctx->ev_counts);
  if (ctx->counts_host) cudaFreeHost(ctx->counts_host);
  if (ctx->st_ring) cudaStreamDestroy(ctx->st_ring);
  if (ctx->ring) cudaFree(ctx->ring);
  if (ctx->fp8_buf) cudaFree(ctx->fp8_buf);
  if (ctx->st_in) cudaStreamDestroy(ctx->st_in);
  if (ctx->st_compute) cudaStreamDestroy(ctx->st_compute);
  if (ctx->st_out) cudaStreamDestroy(ctx->st_out);
  if (ctx->ws) cudaFree(ctx->ws);
  delete ctx;
}

}  // namespace

extern "C" {

const char* bg_moe_strerror(int status) {
  switch (status) {
    case BG_OK: return "ok";
    case BG_ERR_INVALID_ARG: return "invalid argument";
    case BG_ERR_UNSUPPORTED: return "unsupported configuration or device";
    case BG_ERR_CUDA: return "CUDA error (see bg_moe_last_error)";
    case BG_ERR_NOMEM: return "out of device memory";
    case BG_ERR_NO_WEIGHTS: return "weights not set";
    default: return "unknown status";
  }
}

const char* bg_moe_last_error(const bg_moe_ctx* ctx) { return ctx ? ctx->last_error.c_str() : ""; }
int64_t bg_moe_launch_count(const bg_moe_ctx* ctx) { return ctx ? ctx->launches : 0; }
int64_t bg_moe_workspace_bytes(const bg_moe_ctx* ctx) { return ctx ? ctx->ws_bytes : 0; }

int bg_moe_create(const bg_moe_config* cfg, bg_moe_ctx** out) {
  if (cfg == nullptr || out == nullptr) return BG_ERR_INVALID_ARG;
  const bg_moe_config& c = *cfg;
  if (c.d < 64 || c.f < 64 || c.d % 8 || c.f % 8 || c.E < 1 || c.k < 1 || c.k > c.E || c.max_tokens < 0 ||
      c.device < 0)
    return BG_ERR_INVALID_ARG;
  if (c.E > 256 || c.k > 8 || c.gate_fn != 0) return BG_ERR_UNSUPPORTED;
  if (static_cast<int64_t>(c.max_tokens) * c.k > 0x7fffffffLL) return BG_ERR_INVALID_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || c.device >= ndev) return BG_ERR_UNSUPPORTED;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, c.device) != cudaSuccess) return BG_ERR_CUDA;
  if (prop.major != 10) return BG_ERR_UNSUPPORTED;   // tcgen05 / TMEM: sm_100 only, no fallback
  DeviceGuard guard(c.device);
  if (!guard.ok) return BG_ERR_CUDA;
  if (get_encode_fn() == nullptr) return BG_ERR_CUDA;
  if (bg::router_kernels_init() != cudaSuccess || bg::pair_kernels_init() != cudaSuccess) return BG_ERR_CUDA;

  bg_moe_ctx* ctx = new (std::nothrow) bg_moe_ctx();
  if (!ctx) return BG_ERR_NOMEM;
  ctx->cfg = c;
  ctx->num_sms = prop.multiProcessorCount;
  const int64_t Tm = c.max_tokens > 0 ? c.max_tokens : 1;
  const int64_t Rm = Tm * c.k;
  const bg::WsLayout L = bg::ws_layout(c, Tm, ctx->num_sms);
  ctx->ws_bytes = L.total;
  void* p = nullptr;
  if (cudaMalloc(&p, static_cast<size_t>(L.total)) != cudaSuccess) {
    cudaGetLastError();
    delete ctx;
    return BG_ERR_NOMEM;
  }
  ctx->ws = static_cast<uint8_t*>(p);
  ctx->logits = reinterpret_cast<float*>(ctx->ws + L.logits);
  ctx->wr_pieces = ctx->ws + L.pieces;
  ctx->topk_idx = reinterpret_cast<int32_t*>(ctx->ws + L.idx);
  ctx->topk_w = reinterpret_cast<float*>(ctx->ws + L.w);
  ctx->counts = reinterpret_cast<int32_t*>(ctx->ws + L.counts);
  ctx->offsets = reinterpret_cast<int32_t*>(ctx->ws + L.offsets);
  ctx->tile_counts = reinterpret_cast<int32_t*>(ctx->ws + L.tc);
  ctx->tile_base = reinterpret_cast<int32_t*>(ctx->ws + L.tb);
  ctx->tile_rank = reinterpret_cast<int32_t*>(ctx->ws + L.tr);
  ctx->row_src = reinterpret_cast<int32_t*>(ctx->ws + L.rs);
  ctx->inv_perm = reinterpret_cast<int32_t*>(ctx->ws + L.ip);
  ctx->w_perm = reinterpret_cast<float*>(ctx->ws + L.wp);
  ctx->tile_counters = reinterpret_cast<int32_t*>(ctx->ws + L.tile_counters);
  ctx->max_segments = static_cast<int32_t>(Tm);
  ctx->seg_dev_hidden = reinterpret_cast<const void**>(ctx->ws + L.seg_hidden);
  ctx->seg_dev_out = reinterpret_cast<void**>(ctx->ws + L.seg_out);
  ctx->seg_dev_start = reinterpret_cast<int32_t*>(ctx->ws + L.seg_start);
  ctx->x_perm = ctx->ws + L.x;
  ctx->H = ctx->ws + L.h;
  ctx->Y = ctx->ws + L.y;
  const int64_t stage_bytes = Tm * c.d * 2;
  for (int i = 0; i < 2; ++i) {
    ctx->hidden_dev[i] = ctx->ws + L.hd + i * stage_bytes;
    ctx->out_dev[i] = ctx->ws + L.od + i * stage_bytes;
  }
  bool ok = cudaMemset(ctx->tile_counters, 0, 64) == cudaSuccess;
  ok = ok && encode_act_maps(&ctx->am_x, ctx->x_perm, Rm, c.d) && encode_act_maps(&ctx->am_h, ctx->H, Rm, c.f);
  ok = ok && cudaStreamCreateWithFlags(&ctx->st_in, cudaStreamNonBlocking) == cudaSuccess &&
       cudaStreamCreateWithFlags(&ctx->st_compute, cudaStreamNonBlocking) == cudaSuccess &&
       cudaStreamCreateWithFlags(&ctx->st_out, cudaStreamNonBlocking) == cudaSuccess;
  for (int i = 0; i < 2 && ok; ++i)
    ok = cudaEventCreateWithFlags(&ctx->ev_h2d[i], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&ctx->ev_compute[i], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&ctx->ev_d2h[i], cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&ctx->ev_device_call, cudaEventDisableTiming) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    destroy_ctx(ctx);
    return BG_ERR_CUDA;
  }
  *out = ctx;
  return BG_OK;
}

int bg_moe_destroy(bg_moe_ctx* ctx) {
  if (ctx == nullptr) return BG_OK;
  DeviceGuard guard(ctx->cfg.device);
  // the context's own streams may still hold host-path work that touches the workspace
  if (ctx->st_in) cudaStreamSynchronize(ctx->st_in);
  if (ctx->st_compute) cudaStreamSynchronize(ctx->st_compute);
  if (ctx->st_out) cudaStreamSynchronize(ctx->st_out);
  if (ctx->st_ring) cudaStreamSynchronize(ctx->st_ring);
  destroy_ctx(ctx);
  return BG_OK;
}

int bg_moe_set_debug(bg_moe_ctx* ctx, int32_t static_tile_feed, int32_t supergroup_token_tiles, int32_t router_form) {
  if (ctx == nullptr || supergroup_token_tiles < 0 || router_form < 0 || router_form > 2)
    return BG_ERR_INVALID_ARG;
  ctx->dyn_sched = static_tile_feed == 0;
  ctx->sg_max = supergroup_token_tiles;
  ctx->router_form = router_form;
  return BG_OK;
}

// A failed parameter update must not leave a half-new layer behind (new expert tensor maps with the old router
// pieces, or a freed ring with the old chunk size): after any failure past the argument checks the context holds
// NO weights, and every forward call answers BG_ERR_NO_WEIGHTS until a set_weights call succeeds.
static void drop_weights(bg_moe_ctx* ctx) {
  ctx->W_r = nullptr; ctx->b_r = nullptr;
  ctx->W_gate = ctx->W_up = ctx->W_down = nullptr;
  ctx->host_wg = ctx->host_wu = ctx->host_wd = nullptr;
  ctx->ring_chunk = 0;
  ctx->precision = 0;
}

int bg_moe_set_weights(bg_moe_ctx* ctx, const float* W_r, const float* b_r, const void* W_gate, const void* W_up,
                       const void* W_down, void* stream) {
  if (!ctx || !W_r || !W_gate || !W_up || !W_down) return BG_ERR_INVALID_ARG;
  if (!aligned16(W_r) || !aligned16(W_gate) || !aligned16(W_up) || !aligned16(W_down)) return BG_ERR_INVALID_ARG;
  const bg_moe_config& c = ctx->cfg;
  bg_moe_ctx::WeightMaps maps;                     // encoded aside, committed once nothing can fail any more
  if (!encode_weight_maps(ctx, &maps, W_gate, W_up, W_down, c.E)) return BG_ERR_CUDA;   // context untouched
  int rc = set_router_weights(ctx, W_r, static_cast<cudaStream_t>(stream));
  if (rc) { drop_weights(ctx); return rc; }        // the router pieces may be half written
  ctx->wm[0] = maps;
  ctx->W_r = W_r; ctx->b_r = b_r; ctx->W_gate = W_gate; ctx->W_up = W_up; ctx->W_down = W_down;
  ctx->host_wg = ctx->host_wu = ctx->host_wd = nullptr;
  ctx->ring_chunk = 0;            // resident weights
  ctx->precision = 0;             // new weights: bf16 until bg_moe_set_precision quantises them
  return BG_OK;
}

int bg_moe_set_weights_offloaded(bg_moe_ctx* ctx, const float* W_r, const float* b_r, const void* W_gate_host,
                                 const void* W_up_host, const void* W_down_host, int32_t ring_experts, void* stream) {
  if (!ctx || !W_r || !W_gate_host || !W_up_host || !W_down_host || !aligned16(W_r)) return BG_ERR_INVALID_ARG;
  const bg_moe_config& c = ctx->cfg;
  if (ring_experts < 2 || (ring_experts & 1)) return BG_ERR_INVALID_ARG;
  DeviceGuard guard(c.device);
  const int chunk = ring_experts / 2 < c.E ? ring_experts / 2 : c.E;
  const size_t gu_bytes = static_cast<size_t>(c.d) * c.f * 2;
  const size_t half_bytes = 3 * gu_bytes * chunk;
  if (ctx->ring == nullptr || ctx->ring_bytes != 2 * half_bytes) {
    // set-up time allocation (like the caller's own weight tensors); nothing is allocated per call.  The old ring
    // goes first (both need not fit at once), so a context that was streaming its weights has none from here on
    // until this call succeeds.
    if (ctx->st_ring && cudaStreamSynchronize(ctx->st_ring) != cudaSuccess) {
      ctx->last_error = std::string("ring stream sync: ") + cudaGetErrorString(cudaGetLastError());
      drop_weights(ctx);
      return BG_ERR_CUDA;
    }
    if (ctx->ring) { cudaFree(ctx->ring); ctx->ring = nullptr; ctx->ring_bytes = 0; }
    if (ctx->ring_chunk != 0) drop_weights(ctx);   // streamed weights lose their ring; resident ones are unaffected
    void* p = nullptr;
    if (cudaMalloc(&p, 2 * half_bytes) != cudaSuccess) {
      cudaGetLastError();
      return BG_ERR_NOMEM;
    }
    ctx->ring = static_cast<uint8_t*>(p);
    ctx->ring_bytes = 2 * half_bytes;
    if (ctx->st_ring == nullptr) {
      BG_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->st_ring, cudaStreamNonBlocking), "ring stream");
      for (int i = 0; i < 2; ++i) {
        BG_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_ring_ready[i], cudaEventDisableTiming), "ring event");
        BG_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_ring_free[i], cudaEventDisableTiming), "ring event");
      }
    }
    ctx->ring_used[0] = ctx->ring_used[1] = false;
  }
  bg_moe_ctx::WeightMaps maps[2];
  for (int h = 0; h < 2; ++h) {
    uint8_t* half = ctx->ring + h * half_bytes;
    if (!encode_weight_maps(ctx, &maps[h], half, half + chunk * gu_bytes, half + 2 * chunk * gu_bytes, chunk))
      return BG_ERR_CUDA;                          // nothing committed yet
  }
  int rc = set_router_weights(ctx, W_r, static_cast<cudaStream_t>(stream));
  if (rc) { drop_weights(ctx); return rc; }
  ctx->wm[1] = maps[0]; ctx->wm[2] = maps[1];
  ctx->W_r = W_r; ctx->b_r = b_r;
  ctx->host_wg = static_cast<const uint8_t*>(W_gate_host);
  ctx->host_wu = static_cast<const uint8_t*>(W_up_host);
  ctx->host_wd = static_cast<const uint8_t*>(W_down_host);
  ctx->W_gate = W_gate_host; ctx->W_up = W_up_host; ctx->W_down = W_down_host;   // "weights set" for the entry checks
  ctx->ring_chunk = chunk;
  ctx->precision = 0;             // the streamed path is bf16
  return BG_OK;
}

int bg_moe_set_ring_skip_empty(bg_moe_ctx* ctx, int32_t enable) {
  if (!ctx) return BG_ERR_INVALID_ARG;
  if (enable && ctx->counts_host == nullptr) {      // set-up time: E pinned ints and two events
    DeviceGuard guard(ctx->cfg.device);
    void* p = nullptr;
    if (cudaHostAlloc(&p, sizeof(int32_t) * ctx->cfg.E, cudaHostAllocDefault) != cudaSuccess) {
      cudaGetLastError();
      return BG_ERR_NOMEM;
    }
    ctx->counts_host = static_cast<int32_t*>(p);
    BG_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_router_done, cudaEventDisableTiming), "router-done event");
    BG_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_counts, cudaEventDisableTiming), "counts event");
  }
  ctx->ring_skip_empty = enable != 0;
  return BG_OK;
}

int64_t bg_moe_ring_bytes_per_call(const bg_moe_ctx* ctx) { return ctx ? ctx->ring_h2d_bytes : 0; }

int bg_moe_set_precision(bg_moe_ctx* ctx, int32_t precision, void* stream) {
  if (ctx == nullptr || precision < 0 || precision > 2) return BG_ERR_INVALID_ARG;
  if (precision == 0) { ctx->precision = 0; return BG_OK; }
  const bg_moe_config& c = ctx->cfg;
  if (ctx->W_gate == nullptr || ctx->ring_chunk != 0) return BG_ERR_NO_WEIGHTS;     // needs resident bf16 weights
  if (c.d % 128 != 0 || c.f % 64 != 0) return BG_ERR_UNSUPPORTED;                    // 128-byte k-blocks, 64-feature boxes
  if (precision == 2 && c.f % 128 != 0) return BG_ERR_UNSUPPORTED;                   // the down GEMM's k is f
  DeviceGuard guard(c.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t Tm = c.max_tokens > 0 ? c.max_tokens : 1;
  const int64_t Rm = Tm * c.k;
  if (ctx->fp8_buf == nullptr) {
    // set-up time allocation (like the ring): 3 E d f bytes of codes, scales, and the quantised rows
    auto up = [](int64_t v) { return (v + 1023) / 1024 * 1024; };
    const int64_t wq = up(static_cast<int64_t>(c.E) * c.d * c.f);
    const int64_t swf = up(static_cast<int64_t>(c.E) * c.f * 4), swd = up(static_cast<int64_t>(c.E) * c.d * 4);
    const int64_t xq = up(Rm * c.d), hq = up(Rm * c.f), rv = up(Rm * 4);
    void* p = nullptr;
    if (cudaMalloc(&p, static_cast<size_t>(3 * wq + 2 * swf + swd + xq + hq + 4 * rv)) != cudaSuccess) {
      cudaGetLastError();
      return BG_ERR_NOMEM;
    }
    uint8_t* b = static_cast<uint8_t*>(p);
    ctx->fp8_buf = b;
    ctx->q_gate = b; b += wq;
    ctx->q_up = b; b += wq;
    ctx->q_down = b; b += wq;
    ctx->sw_gate = reinterpret_cast<float*>(b); b += swf;
    ctx->sw_up = reinterpret_cast<float*>(b); b += swf;
    ctx->sw_down = reinterpret_cast<float*>(b); b += swd;
    ctx->xq_perm = b; b += xq;
    ctx->hq = b; b += hq;
    ctx->sx_perm = reinterpret_cast<float*>(b); b += rv;
    ctx->hmax = reinterpret_cast<unsigned*>(b); b += rv;
    ctx->sh_perm = reinterpret_cast<float*>(b); b += rv;
    ctx->sc_perm = reinterpret_cast<float*>(b); b += rv;
    bool ok = encode_weight_map_u8(&ctx->tm_qg, ctx->q_gate, c.E, c.f, c.d) &&
              encode_weight_map_u8(&ctx->tm_qu, ctx->q_up, c.E, c.f, c.d) &&
              (c.f % 128 != 0 || encode_weight_map_u8(&ctx->tm_qd, ctx->q_down, c.E, c.d, c.f, 128));
    for (int i = 0; i < 16 && ok; ++i) ok = encode_act_map_u8(&ctx->am_xq.m[i], ctx->xq_perm, Rm, c.d, 8 * (i + 1));
    for (int i = 0; i < 16 && ok && c.f % 128 == 0; ++i) ok = encode_act_map_u8(&ctx->am_hq.m[i], ctx->hq, Rm, c.f, 8 * (i + 1));
    if (!ok) {
      ctx->last_error = "cuTensorMapEncodeTiled(fp8) failed";
      return BG_ERR_CUDA;
    }
  }
  int rc = begin_call(ctx, st);
  if (rc) return rc;
  BG_LAUNCH(ctx, bg::launch_quantize_weights(ctx->W_gate, c.E, c.d, c.f, ctx->q_gate, ctx->sw_gate, st), "quantize W_gate");
  BG_LAUNCH(ctx, bg::launch_quantize_weights(ctx->W_up, c.E, c.d, c.f, ctx->q_up, ctx->sw_up, st), "quantize W_up");
  if (precision == 2)
    BG_LAUNCH(ctx, bg::launch_quantize_weights(ctx->W_down, c.E, c.f, c.d, ctx->q_down, ctx->sw_down, st), "quantize W_down");
  ctx->precision = precision;
  return end_call(ctx, st, false);
}

int bg_moe_debug_fp8_down_views(bg_moe_ctx* ctx, const void** H, const void** hq, const float** sh_perm,
                                const void** q_down, const float** sw_down) {
  if (!ctx || ctx->fp8_buf == nullptr) return BG_ERR_INVALID_ARG;
  if (H) *H = ctx->H;
  if (hq) *hq = ctx->hq;
  if (sh_perm) *sh_perm = ctx->sh_perm;
  if (q_down) *q_down = ctx->q_down;
  if (sw_down) *sw_down = ctx->sw_down;
  return BG_OK;
}

int bg_moe_debug_ffn_views(bg_moe_ctx* ctx, const void** H, const void** Y) {
  if (!ctx) return BG_ERR_INVALID_ARG;
  if (H) *H = ctx->H;
  if (Y) *Y = ctx->Y;
  return BG_OK;
}

int bg_moe_debug_fp8_views(bg_moe_ctx* ctx, const void** xq_perm, const float** sx_perm, const void** q_gate,
                           const float** sw_gate, const void** q_up, const float** sw_up) {
  if (!ctx || ctx->fp8_buf == nullptr) return BG_ERR_INVALID_ARG;
  if (xq_perm) *xq_perm = ctx->xq_perm;
  if (sx_perm) *sx_perm = ctx->sx_perm;
  if (q_gate) *q_gate = ctx->q_gate;
  if (sw_gate) *sw_gate = ctx->sw_gate;
  if (q_up) *q_up = ctx->q_up;
  if (sw_up) *sw_up = ctx->sw_up;
  return BG_OK;
}

int bg_moe_route(bg_moe_ctx* ctx, const void* hidden, int32_t T, const float* logits_in, float* logits_out,
                 int32_t* topk_idx, float* topk_w, int32_t* counts, int32_t* offsets, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (!counts || !offsets) return BG_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (T == 0) {   // nothing routed: counts and offsets are all zero
    DeviceGuard guard0(ctx->cfg.device);
    if ((rc = begin_call(ctx, st))) return rc;
    BG_LAUNCH(ctx, bg::launch_scan(ctx->tile_counts, 0, ctx->cfg.E, ctx->tile_base, counts, offsets, st), "scan");
    return end_call(ctx, st, false);
  }
  if (!topk_idx || !topk_w) return BG_ERR_INVALID_ARG;
  if (logits_in == nullptr && (hidden == nullptr || !aligned16(hidden))) return BG_ERR_INVALID_ARG;
  if (logits_in == nullptr && ctx->W_r == nullptr) return BG_ERR_NO_WEIGHTS;
  DeviceGuard guard(ctx->cfg.device);
  if ((rc = begin_call(ctx, st))) return rc;
  float* lbuf = logits_out ? logits_out : ctx->logits;
  rc = do_route(ctx, hidden, T, logits_in, lbuf, topk_idx, topk_w, counts, offsets, st);
  if (rc) return rc;
  if (logits_in && logits_out && logits_in != logits_out)
    BG_CUDA(ctx, cudaMemcpyAsync(logits_out, logits_in, sizeof(float) * T * ctx->cfg.E, cudaMemcpyDeviceToDevice, st),
            "copy logits");
  return end_call(ctx, st, false);
}

int bg_moe_permute(bg_moe_ctx* ctx, const void* hidden, int32_t T, const int32_t* topk_idx, const int32_t* offsets,
                   int32_t* row_src, int32_t* inv_perm, void* x_perm, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!topk_idx || !offsets || !row_src || !inv_perm) return BG_ERR_INVALID_ARG;
  if (x_perm && (!hidden || !aligned16(hidden) || !aligned16(x_perm))) return BG_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const bg_moe_config& c = ctx->cfg;
  if ((rc = begin_call(ctx, st))) return rc;
  // the permutation is rebuilt from topk_idx alone (offsets = the exclusive scan of its histogram)
  BG_LAUNCH(ctx, bg::launch_tile_rank(topk_idx, T, c.E, c.k, ctx->tile_rank, ctx->tile_counts, st), "tile_rank");
  BG_LAUNCH(ctx, bg::launch_scan(ctx->tile_counts, bg::route_num_tiles(T), c.E, ctx->tile_base, nullptr, nullptr, st),
            "scan");
  bg::PermLaunch pl = {topk_idx, ctx->tile_rank, ctx->tile_base, nullptr, row_src, inv_perm, nullptr};
  BG_LAUNCH(ctx, bg::launch_gather(hidden, pl, T, c.E, c.k, c.d, x_perm, ctx->num_sms, st), "gather");
  return end_call(ctx, st, false);
}

int bg_moe_expert_ffn(bg_moe_ctx* ctx, const void* x_perm, const int32_t* offsets, int32_t T, void* y_perm,
                      void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!x_perm || !offsets || !y_perm || !aligned16(x_perm) || !aligned16(y_perm)) return BG_ERR_INVALID_ARG;
  if (ctx->W_gate == nullptr || ctx->ring_chunk != 0) return BG_ERR_NO_WEIGHTS;   // needs resident expert weights
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if ((rc = begin_call(ctx, st))) return rc;
  // no router kernel precedes the GEMMs here: zero their ticket counters on the stream
  BG_CUDA(ctx, cudaMemsetAsync(ctx->tile_counters, 0, 32, st), "memset ticket counters");
  // per-kernel profile of the split FFN: "gateup_swiglu" and "down" are timed, the other three stages read 0
  mark(ctx, 0, st); mark(ctx, 1, st); mark(ctx, 2, st);
  rc = do_ffn(ctx, x_perm, offsets, T, y_perm, nullptr, st, /*mark_between=*/3);
  if (rc) return rc;
  mark(ctx, 4, st); mark(ctx, 5, st);
  ctx->profile_valid = ctx->profile;
  return end_call(ctx, st, false);
}

int bg_moe_unpermute(bg_moe_ctx* ctx, const void* y_perm, const int32_t* inv_perm, const float* topk_w, int32_t T,
                     void* out, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!y_perm || !inv_perm || !topk_w || !out || !aligned16(y_perm) || !aligned16(out)) return BG_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if ((rc = begin_call(ctx, st))) return rc;
  BG_LAUNCH(ctx, bg::launch_unpermute(y_perm, inv_perm, topk_w, T, ctx->cfg.k, ctx->cfg.d, out, ctx->num_sms, st),
            "unpermute");
  return end_call(ctx, st, false);
}

int bg_moe_combined_forward(bg_moe_ctx* ctx, const void* hidden, int32_t T, void* out, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!hidden || !out || !aligned16(hidden) || !aligned16(out)) return BG_ERR_INVALID_ARG;
  if (ctx->W_r == nullptr) return BG_ERR_NO_WEIGHTS;
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if ((rc = begin_call(ctx, st))) return rc;
  rc = do_forward(ctx, hidden, T, out, st, nullptr);
  if (rc) return rc;
  return end_call(ctx, st, false);
}

int bg_moe_combined_forward_segments(bg_moe_ctx* ctx, const bg_moe_segment* segments, int32_t n_segments,
                                     void* stream) {
  if (ctx == nullptr || n_segments < 0 || (n_segments > 0 && segments == nullptr)) return BG_ERR_INVALID_ARG;
  if (n_segments > ctx->max_segments) return BG_ERR_INVALID_ARG;
  int64_t T64 = 0;
  for (int i = 0; i < n_segments; ++i) {
    const bg_moe_segment& sg = segments[i];
    if (sg.n_tokens < 0) return BG_ERR_INVALID_ARG;
    if (sg.n_tokens > 0 && (!sg.hidden || !sg.out || !aligned16(sg.hidden) || !aligned16(sg.out)))
      return BG_ERR_INVALID_ARG;
    T64 += sg.n_tokens;
  }
  if (T64 > ctx->cfg.max_tokens) return BG_ERR_INVALID_ARG;
  const int32_t T = static_cast<int32_t>(T64);
  if (T == 0) return BG_OK;
  if (ctx->W_r == nullptr) return BG_ERR_NO_WEIGHTS;
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int rc = begin_call(ctx, st);
  if (rc) return rc;
  // The segment table goes to the device in ONE copy through pageable host staging (cudaMemcpyAsync from
  // pageable memory returns once the bytes are staged, so the vector can be reused by the next call).
  // Device layout (one slab): hidden[max_segments] | out[max_segments] | start[max_segments + 1]; the host
  // image is packed the same way so a single contiguous copy serves the three arrays.
  const int n = n_segments;
  const size_t cap = static_cast<size_t>(ctx->max_segments);
  const size_t img_bytes = 16 * cap + 4 * (cap + 1);
  ctx->seg_host_img.resize(img_bytes);
  const void** h_hidden = reinterpret_cast<const void**>(ctx->seg_host_img.data());
  void** h_out = reinterpret_cast<void**>(ctx->seg_host_img.data() + 8 * cap);
  int32_t* h_start = reinterpret_cast<int32_t*>(ctx->seg_host_img.data() + 16 * cap);
  // an empty segment may carry null pointers (its rows are never looked up); the router uses hidden[0]
  // as the source address of zero-filled copies, so every entry is made a valid address
  const void* first_valid = nullptr;
  for (int i = 0; i < n && first_valid == nullptr; ++i)
    if (segments[i].n_tokens > 0) first_valid = segments[i].hidden;
  int32_t acc = 0;
  for (int i = 0; i < n; ++i) {
    h_hidden[i] = segments[i].n_tokens > 0 ? segments[i].hidden : first_valid;
    h_out[i] = segments[i].out;
    h_start[i] = acc;
    acc += segments[i].n_tokens;
  }
  h_start[n] = acc;
  if (static_cast<size_t>(n) * 4 >= cap) {
    // long tables: one copy of the whole image
    BG_CUDA(ctx, cudaMemcpyAsync(ctx->seg_dev_hidden, ctx->seg_host_img.data(), img_bytes, cudaMemcpyHostToDevice, st),
            "H2D segment table");
  } else {
    // short tables in a large context: three short copies beat one of 20 bytes x max_tokens
    BG_CUDA(ctx, cudaMemcpyAsync(ctx->seg_dev_hidden, h_hidden, sizeof(void*) * n, cudaMemcpyHostToDevice, st),
            "H2D segment table (hidden)");
    BG_CUDA(ctx, cudaMemcpyAsync(ctx->seg_dev_out, h_out, sizeof(void*) * n, cudaMemcpyHostToDevice, st),
            "H2D segment table (out)");
    BG_CUDA(ctx, cudaMemcpyAsync(ctx->seg_dev_start, h_start, sizeof(int32_t) * (n + 1), cudaMemcpyHostToDevice, st),
            "H2D segment table (start)");
  }
  bg::SegTable seg;
  seg.hidden = reinterpret_cast<const void* const*>(ctx->seg_dev_hidden);
  seg.out = reinterpret_cast<void* const*>(ctx->seg_dev_out);
  seg.start = ctx->seg_dev_start;
  seg.n = n;
  rc = do_forward(ctx, nullptr, T, nullptr, st, &seg);
  if (rc) return rc;
  return end_call(ctx, st, false);
}

// Host-pointer entry point, pipelined over the context's own streams (two staging slots):
//   st_in:      H2D of call i           (after the chain of call i-2 has released the slot's input buffer)
//   st_compute: the fused chain of call i (after its H2D; after the D2H of call i-2 has released the output buffer)
//   st_out:     D2H of call i           (after its chain)
// so the upload of call i+1 and the download of call i-1 overlap the GEMMs of call i.  `stream` only WAITS for
// the download: work the caller enqueues on `stream` afterwards (and a synchronize on it) sees out_host complete.
// The host buffers are not stream-ordered objects: hidden_host must hold its data when the call is made.
int bg_moe_combined_forward_host(bg_moe_ctx* ctx, const void* hidden_host, int32_t T, void* out_host, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!hidden_host || !out_host) return BG_ERR_INVALID_ARG;
  if (ctx->W_r == nullptr) return BG_ERR_NO_WEIGHTS;
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int slot = ctx->host_slot;
  const size_t bytes = static_cast<size_t>(T) * ctx->cfg.d * 2;
  if (ctx->counters_dirty) {
    BG_CUDA(ctx, cudaMemsetAsync(ctx->tile_counters, 0, 64, ctx->st_compute), "memset counters");
    ctx->counters_dirty = false;
  }
  // ordered after every earlier device-pointer call on this context (weights, workspace)
  if (ctx->device_call_pending) {
    BG_CUDA(ctx, cudaStreamWaitEvent(ctx->st_compute, ctx->ev_device_call, 0), "order after device calls");
    ctx->device_call_pending = false;
  }
  if (ctx->host_calls >= 2) BG_CUDA(ctx, cudaStreamWaitEvent(ctx->st_in, ctx->ev_compute[slot], 0), "slot input free");
  BG_CUDA(ctx, cudaMemcpyAsync(ctx->hidden_dev[slot], hidden_host, bytes, cudaMemcpyHostToDevice, ctx->st_in), "H2D hidden");
  BG_CUDA(ctx, cudaEventRecord(ctx->ev_h2d[slot], ctx->st_in), "record H2D");
  BG_CUDA(ctx, cudaStreamWaitEvent(ctx->st_compute, ctx->ev_h2d[slot], 0), "wait H2D");
  if (ctx->host_calls >= 2) BG_CUDA(ctx, cudaStreamWaitEvent(ctx->st_compute, ctx->ev_d2h[slot], 0), "slot output free");
  rc = do_forward(ctx, ctx->hidden_dev[slot], T, ctx->out_dev[slot], ctx->st_compute, nullptr);
  if (rc) return rc;
  BG_CUDA(ctx, cudaEventRecord(ctx->ev_compute[slot], ctx->st_compute), "record chain");
  BG_CUDA(ctx, cudaStreamWaitEvent(ctx->st_out, ctx->ev_compute[slot], 0), "wait chain");
  BG_CUDA(ctx, cudaMemcpyAsync(out_host, ctx->out_dev[slot], bytes, cudaMemcpyDeviceToHost, ctx->st_out), "D2H out");
  BG_CUDA(ctx, cudaEventRecord(ctx->ev_d2h[slot], ctx->st_out), "record D2H");
  BG_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_d2h[slot], 0), "caller's stream waits for the result");
  ctx->host_slot ^= 1;
  ctx->host_calls += 1;
  ctx->host_call_pending = true;
  return BG_OK;
}

int bg_moe_host_input_sync(bg_moe_ctx* ctx) {
  if (!ctx) return BG_ERR_INVALID_ARG;
  if (ctx->host_calls == 0) return BG_OK;
  DeviceGuard guard(ctx->cfg.device);
  BG_CUDA(ctx, cudaEventSynchronize(ctx->ev_h2d[ctx->host_slot ^ 1]), "wait for the last upload");
  return BG_OK;
}

int bg_moe_profile_enable(bg_moe_ctx* ctx, int enable) {
  if (!ctx) return BG_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->cfg.device);
  if (enable && ctx->ev[0] == nullptr)
    for (cudaEvent_t& e : ctx->ev) BG_CUDA(ctx, cudaEventCreate(&e), "cudaEventCreate");
  ctx->profile = enable != 0;
  ctx->profile_valid = false;
  return BG_OK;
}

int bg_moe_profile_read(bg_moe_ctx* ctx, float* ms_out) {
  if (!ctx || !ms_out || !ctx->profile_valid) return BG_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->cfg.device);
  BG_CUDA(ctx, cudaEventSynchronize(ctx->ev[BG_MOE_NUM_STAGES]), "cudaEventSynchronize");
  for (int i = 0; i < BG_MOE_NUM_STAGES; ++i)
    BG_CUDA(ctx, cudaEventElapsedTime(ms_out + i, ctx->ev[i], ctx->ev[i + 1]), "cudaEventElapsedTime");
  return BG_OK;
}

int bg_moe_debug_views(bg_moe_ctx* ctx, const float** logits, const int32_t** topk_idx, const float** topk_w,
                       const int32_t** counts, const int32_t** offsets, const int32_t** row_src,
                       const int32_t** inv_perm) {
  if (!ctx) return BG_ERR_INVALID_ARG;
  if (logits) *logits = ctx->logits;
  if (topk_idx) *topk_idx = ctx->topk_idx;
  if (topk_w) *topk_w = ctx->topk_w;
  if (counts) *counts = ctx->counts;
  if (offsets) *offsets = ctx->offsets;
  if (row_src) *row_src = ctx->row_src;
  if (inv_perm) *inv_perm = ctx->inv_perm;
  return BG_OK;
}

}  // extern "C"
