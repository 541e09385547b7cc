// api.cu -- the C ABI declared in include/bg_moe.h: argument validation, workspace, TMA tensor-map
// encoding and kernel sequencing.  No arithmetic of the layer happens on the host.
#include "../../include/bg_moe.h"
#include "kernels.h"

#include <cstdio>
#include <cstdlib>
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
  float* partial = nullptr;     // router split-K partials [ksplit][T][E]
  void* wr_pieces = nullptr;    // bf16 [3][d][round_up(E,16)]: exact hi/mid/lo split of W_r
  int32_t* topk_idx = nullptr;
  float* topk_w = nullptr;
  int32_t* counts = nullptr;
  int32_t* offsets = nullptr;
  int32_t* block_counts = nullptr;
  int32_t* block_base = nullptr;
  int32_t* row_src = nullptr;
  int32_t* inv_perm = nullptr;
  float* w_perm = nullptr;      // gate weights in expert order (fused path)
  int32_t* tile_counters = nullptr;   // [4]: ticket / finished counters of the two pair GEMMs (self re-arming)
  bool dyn_sched = true;        // dynamic tile feed of the pair GEMMs (BG_MOE_SCHED=static: tile t -> cluster t mod 74)
  // segment table of bg_moe_combined_forward_segments (device arrays + pageable host staging)
  int32_t max_segments = 0;
  const void** seg_dev_hidden = nullptr;
  void** seg_dev_out = nullptr;
  int32_t* seg_dev_start = nullptr;
  std::vector<const void*> seg_host_ptrs;
  std::vector<int32_t> seg_host_start;
  void* x_perm = nullptr;
  void* H = nullptr;
  void* Y = nullptr;
  void* hidden_dev = nullptr;   // staging for the host-pointer entry point
  void* out_dev = nullptr;
  // weight tensor maps (encoded in set_weights)
  CUtensorMap tm_wg, tm_wu, tm_wd, tm_wr, tm_wr1;   // tm_wr1: one-piece box of the 4-D W_r view (E > 128)
  CUtensorMap tm_wg4, tm_wu4, tm_wd4;   // 4-D block views (kernels.h GemmLaunch), valid when f % 64 == 0 / d % 64 == 0
  // activation tensor maps of the workspace x_perm / H (whole capacity: rows past T*k are never stored)
  bg::ActMaps am_x, am_h;
  int sg_max = 0;               // BG_MOE_SG_TOKEN_TILES=n overrides the pair kernel's super-group size (tests)
  bool pair_gemm = true;        // CTA-pair grouped GEMM (BG_MOE_GEMM=tile selects the 1-CTA 128x256 kernel)
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

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline void mark(bg_moe_ctx* ctx, int i, cudaStream_t st) {
  if (ctx->profile) cudaEventRecord(ctx->ev[i], st);
}

int cuda_fail(bg_moe_ctx* ctx, cudaError_t e, const char* where) {
  if (ctx) ctx->last_error = std::string(where) + ": " + cudaGetErrorString(e);
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

// a1-a4 on explicit buffers.
int do_route(bg_moe_ctx* ctx, const void* hidden, int32_t T, const float* logits_in, float* logits_buf,
             int32_t* topk_idx, float* topk_w, int32_t* counts, int32_t* offsets, cudaStream_t st,
             const bg::SegTable* seg = nullptr) {
  const bg_moe_config& c = ctx->cfg;
  if (logits_in == nullptr) {
    const int ks = bg::router_ksplit(T, c.d, ctx->num_sms);
    if (seg != nullptr) {
      mark(ctx, 0, st);
      BG_LAUNCH(ctx, bg::launch_router_gemm_segments(*seg, ctx->tm_wr, ctx->tm_wr1, T, c.d, c.E, ks, ctx->partial,
                                                     ctx->block_counts, bg::route_num_blocks(T, c.k) * c.E, st),
                "router_gemm_segments");
    } else {
      CUtensorMap tm_h;
      if (!encode_act_map(&tm_h, hidden, T, c.d)) { ctx->last_error = "cuTensorMapEncodeTiled(hidden) failed"; return BG_ERR_CUDA; }
      mark(ctx, 0, st);
      BG_LAUNCH(ctx, bg::launch_router_gemm(tm_h, ctx->tm_wr, ctx->tm_wr1, T, c.d, c.E, ks, ctx->partial, ctx->block_counts,
                                            bg::route_num_blocks(T, c.k) * c.E, st), "router_gemm");
    }
    mark(ctx, 1, st);
    BG_LAUNCH(ctx, bg::launch_topk_hist(ctx->partial, ks, ctx->b_r, logits_buf, T, c.E, c.k, topk_idx, topk_w,
                                        ctx->block_counts, st), "topk_hist");
  } else {
    BG_CUDA(ctx, cudaMemsetAsync(ctx->block_counts, 0, sizeof(int32_t) * bg::route_num_blocks(T, c.k) * c.E, st),
            "memset block_counts");
    BG_LAUNCH(ctx, bg::launch_topk_hist(logits_in, 1, nullptr, nullptr, T, c.E, c.k, topk_idx, topk_w,
                                        ctx->block_counts, st), "topk_hist");
  }
  mark(ctx, 2, st);
  BG_LAUNCH(ctx, bg::launch_scan(ctx->block_counts, bg::route_num_blocks(T, c.k), c.E, ctx->block_base, counts,
                                 offsets, st), "scan");
  return BG_OK;
}

int do_ffn(bg_moe_ctx* ctx, const void* x_perm, const int32_t* offsets, int32_t T, void* y,
           const float* row_scale, const int32_t* row_src, cudaStream_t st, int mark_between = -1) {
  const bg_moe_config& c = ctx->cfg;
  const int64_t R = static_cast<int64_t>(T) * c.k;
  bg::GemmLaunch g1;
  if (x_perm == ctx->x_perm) {
    g1.tm_act = ctx->am_x;             // workspace maps, encoded once in bg_moe_create
  } else if (!encode_act_maps(&g1.tm_act, x_perm, R, c.d)) {
    ctx->last_error = "cuTensorMapEncodeTiled(x_perm) failed";
    return BG_ERR_CUDA;
  }
  g1.tm_b0 = ctx->tm_wg;
  g1.tm_b1 = ctx->tm_wu;
  g1.sg_max = ctx->sg_max;
  g1.tile_counter = ctx->dyn_sched ? ctx->tile_counters : nullptr;
  g1.w4d = c.f % 64 == 0;
  g1.tm_b0_4d = g1.w4d ? ctx->tm_wg4 : ctx->tm_wg;
  g1.tm_b1_4d = g1.w4d ? ctx->tm_wu4 : ctx->tm_wu;
  g1.offsets = offsets;
  g1.E = c.E; g1.K = c.d; g1.N = c.f;
  g1.out = ctx->H;
  g1.row_scale = nullptr; g1.row_src = nullptr; g1.row_scale_perm = nullptr;
  g1.num_sms = ctx->num_sms;
  BG_LAUNCH(ctx, ctx->pair_gemm ? bg::launch_gateup_swiglu_pair(g1, st) : bg::launch_gateup_swiglu(g1, st),
            "gateup_swiglu");
  if (mark_between >= 0) mark(ctx, mark_between, st);
  bg::GemmLaunch g2;
  g2.tm_act = ctx->am_h;
  g2.tm_b0 = ctx->tm_wd;
  g2.tm_b1 = ctx->tm_wd;
  g2.sg_max = ctx->sg_max;
  g2.tile_counter = ctx->dyn_sched ? ctx->tile_counters + 2 : nullptr;
  g2.w4d = c.d % 64 == 0;
  g2.tm_b0_4d = g2.w4d ? ctx->tm_wd4 : ctx->tm_wd;
  g2.tm_b1_4d = g2.tm_b0_4d;
  g2.offsets = offsets;
  g2.E = c.E; g2.K = c.f; g2.N = c.d;
  g2.out = y;
  g2.row_scale = row_scale; g2.row_src = row_src;
  g2.row_scale_perm = row_scale ? ctx->w_perm : nullptr;
  g2.num_sms = ctx->num_sms;
  BG_LAUNCH(ctx, ctx->pair_gemm ? bg::launch_down_pair(g2, st) : bg::launch_down(g2, st), "down");
  return BG_OK;
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
  if (bg::gemm_kernels_init() != cudaSuccess || bg::router_kernels_init() != cudaSuccess ||
      bg::pair_kernels_init() != cudaSuccess)
    return BG_ERR_CUDA;

  bg_moe_ctx* ctx = new (std::nothrow) bg_moe_ctx();
  if (!ctx) return BG_ERR_NOMEM;
  ctx->cfg = c;
  ctx->num_sms = prop.multiProcessorCount;
  const int64_t Tm = c.max_tokens > 0 ? c.max_tokens : 1;
  const int64_t Rm = Tm * c.k;
  const bg::WsLayout L = bg::ws_layout(c, Tm, ctx->num_sms);
  const int64_t off = L.total;
  const int64_t o_logits = L.logits, o_idx = L.idx, o_w = L.w, o_part = L.part, o_pieces = L.pieces;
  const int64_t o_counts = L.counts, o_offsets = L.offsets, o_bc = L.bc, o_bb = L.bb;
  const int64_t o_rs = L.rs, o_ip = L.ip, o_wp = L.wp, o_x = L.x, o_h = L.h, o_y = L.y, o_hd = L.hd, o_od = L.od;
  ctx->ws_bytes = off;
  void* p = nullptr;
  if (cudaMalloc(&p, static_cast<size_t>(off)) != cudaSuccess) {
    cudaGetLastError();
    delete ctx;
    return BG_ERR_NOMEM;
  }
  ctx->ws = static_cast<uint8_t*>(p);
  ctx->logits = reinterpret_cast<float*>(ctx->ws + o_logits);
  ctx->partial = reinterpret_cast<float*>(ctx->ws + o_part);
  ctx->wr_pieces = ctx->ws + o_pieces;
  ctx->topk_idx = reinterpret_cast<int32_t*>(ctx->ws + o_idx);
  ctx->topk_w = reinterpret_cast<float*>(ctx->ws + o_w);
  ctx->counts = reinterpret_cast<int32_t*>(ctx->ws + o_counts);
  ctx->offsets = reinterpret_cast<int32_t*>(ctx->ws + o_offsets);
  ctx->block_counts = reinterpret_cast<int32_t*>(ctx->ws + o_bc);
  ctx->block_base = reinterpret_cast<int32_t*>(ctx->ws + o_bb);
  ctx->row_src = reinterpret_cast<int32_t*>(ctx->ws + o_rs);
  ctx->inv_perm = reinterpret_cast<int32_t*>(ctx->ws + o_ip);
  ctx->w_perm = reinterpret_cast<float*>(ctx->ws + o_wp);
  ctx->tile_counters = reinterpret_cast<int32_t*>(ctx->ws + L.tile_counters);
  if (cudaMemset(ctx->tile_counters, 0, 16) != cudaSuccess) {
    cudaFree(ctx->ws);
    delete ctx;
    return BG_ERR_CUDA;
  }
  ctx->max_segments = static_cast<int32_t>(Tm);
  ctx->seg_dev_hidden = reinterpret_cast<const void**>(ctx->ws + L.seg_hidden);
  ctx->seg_dev_out = reinterpret_cast<void**>(ctx->ws + L.seg_out);
  ctx->seg_dev_start = reinterpret_cast<int32_t*>(ctx->ws + L.seg_start);
  ctx->x_perm = ctx->ws + o_x;
  ctx->H = ctx->ws + o_h;
  ctx->Y = ctx->ws + o_y;
  ctx->hidden_dev = ctx->ws + o_hd;
  ctx->out_dev = ctx->ws + o_od;
  if (!encode_act_maps(&ctx->am_x, ctx->x_perm, Rm, c.d) || !encode_act_maps(&ctx->am_h, ctx->H, Rm, c.f)) {
    cudaFree(ctx->ws);
    delete ctx;
    return BG_ERR_CUDA;
  }
  {
    const char* g = std::getenv("BG_MOE_GEMM");
    if (g != nullptr && std::strcmp(g, "tile") == 0) ctx->pair_gemm = false;
    const char* sc = std::getenv("BG_MOE_SCHED");
    if (sc != nullptr && std::strcmp(sc, "static") == 0) ctx->dyn_sched = false;
    const char* sg = std::getenv("BG_MOE_SG_TOKEN_TILES");
    if (sg != nullptr && std::atoi(sg) > 0) ctx->sg_max = std::atoi(sg);
  }
  *out = ctx;
  return BG_OK;
}

int bg_moe_destroy(bg_moe_ctx* ctx) {
  if (ctx == nullptr) return BG_OK;
  DeviceGuard guard(ctx->cfg.device);
  for (cudaEvent_t e : ctx->ev)
    if (e) cudaEventDestroy(e);
  if (ctx->ws) cudaFree(ctx->ws);
  delete ctx;
  return BG_OK;
}

int bg_moe_set_weights(bg_moe_ctx* ctx, const float* W_r, const float* b_r, const void* W_gate, const void* W_up,
                       const void* W_down) {
  if (!ctx || !W_r || !W_gate || !W_up || !W_down) return BG_ERR_INVALID_ARG;
  if (!aligned16(W_r) || !aligned16(W_gate) || !aligned16(W_up) || !aligned16(W_down)) return BG_ERR_INVALID_ARG;
  const bg_moe_config& c = ctx->cfg;
  if (!encode_weight_map(&ctx->tm_wg, W_gate, c.E, c.d, c.f) || !encode_weight_map(&ctx->tm_wu, W_up, c.E, c.d, c.f) ||
      !encode_weight_map(&ctx->tm_wd, W_down, c.E, c.f, c.d)) {
    ctx->last_error = "cuTensorMapEncodeTiled(weights) failed";
    return BG_ERR_CUDA;
  }
  {
    // block views: pair kernel a7 = 1 block per map, a8 = 2; tile kernel a7 = 2, a8 = 4
    const int nb_gu = ctx->pair_gemm ? 1 : 2, nb_d = ctx->pair_gemm ? 2 : 4;
    if ((c.f % 64 == 0 && (!encode_weight_map_4d(&ctx->tm_wg4, W_gate, c.E, c.d, c.f, nb_gu) ||
                           !encode_weight_map_4d(&ctx->tm_wu4, W_up, c.E, c.d, c.f, nb_gu))) ||
        (c.d % 64 == 0 && !encode_weight_map_4d(&ctx->tm_wd4, W_down, c.E, c.f, c.d, nb_d))) {
      ctx->last_error = "cuTensorMapEncodeTiled(weight block views) failed";
      return BG_ERR_CUDA;
    }
  }
  // exact bf16 hi/mid/lo split of W_r for the tensor-core router (router_gemm.cu); [3][d][E_ld]
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
    BG_LAUNCH(ctx, bg::launch_split_wr(W_r, c.d, c.E, ctx->wr_pieces, nullptr), "split_wr");
    BG_CUDA(ctx, cudaStreamSynchronize(nullptr), "split_wr sync");   // set_weights is the one synchronous call
  }
  ctx->W_r = W_r; ctx->b_r = b_r; ctx->W_gate = W_gate; ctx->W_up = W_up; ctx->W_down = W_down;
  return BG_OK;
}

int bg_moe_route(bg_moe_ctx* ctx, const void* hidden, int32_t T, const float* logits_in, float* logits_out,
                 int32_t* topk_idx, float* topk_w, int32_t* counts, int32_t* offsets, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (!counts || !offsets) return BG_ERR_INVALID_ARG;
  if (T == 0) {   // nothing routed: counts and offsets are all zero
    DeviceGuard guard0(ctx->cfg.device);
    BG_LAUNCH(ctx, bg::launch_scan(ctx->block_counts, 0, ctx->cfg.E, ctx->block_base, counts, offsets,
                                   static_cast<cudaStream_t>(stream)), "scan");
    return BG_OK;
  }
  if (!topk_idx || !topk_w) return BG_ERR_INVALID_ARG;
  if (logits_in == nullptr && (hidden == nullptr || !aligned16(hidden))) return BG_ERR_INVALID_ARG;
  if (logits_in == nullptr && ctx->W_r == nullptr) return BG_ERR_NO_WEIGHTS;
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  float* lbuf = logits_out ? logits_out : ctx->logits;
  rc = do_route(ctx, hidden, T, logits_in, lbuf, topk_idx, topk_w, counts, offsets, st);
  if (rc) return rc;
  if (logits_in && logits_out && logits_in != logits_out && T > 0)
    BG_CUDA(ctx, cudaMemcpyAsync(logits_out, logits_in, sizeof(float) * T * ctx->cfg.E, cudaMemcpyDeviceToDevice, st),
            "copy logits");
  return BG_OK;
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
  BG_LAUNCH(ctx, bg::launch_block_hist(topk_idx, T, c.E, c.k, ctx->block_counts, st), "block_hist");
  BG_LAUNCH(ctx, bg::launch_scan(ctx->block_counts, bg::route_num_blocks(T, c.k), c.E, ctx->block_base, nullptr,
                                 nullptr, st), "scan");
  BG_LAUNCH(ctx, bg::launch_rank(topk_idx, ctx->block_base, T, c.E, c.k, row_src, inv_perm, nullptr, nullptr, st), "rank");
  if (x_perm) BG_LAUNCH(ctx, bg::launch_gather(hidden, inv_perm, T, c.k, c.d, x_perm, ctx->num_sms, st), "gather");
  return BG_OK;
}

int bg_moe_expert_ffn(bg_moe_ctx* ctx, const void* x_perm, const int32_t* offsets, int32_t T, void* y_perm,
                      void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!x_perm || !offsets || !y_perm || !aligned16(x_perm) || !aligned16(y_perm)) return BG_ERR_INVALID_ARG;
  if (ctx->W_gate == nullptr) return BG_ERR_NO_WEIGHTS;
  DeviceGuard guard(ctx->cfg.device);
  return do_ffn(ctx, x_perm, offsets, T, y_perm, nullptr, nullptr, static_cast<cudaStream_t>(stream));
}

int bg_moe_unpermute(bg_moe_ctx* ctx, const void* y_perm, const int32_t* inv_perm, const float* topk_w, int32_t T,
                     void* out, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!y_perm || !inv_perm || !topk_w || !out || !aligned16(y_perm) || !aligned16(out)) return BG_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->cfg.device);
  BG_LAUNCH(ctx, bg::launch_unpermute(y_perm, inv_perm, topk_w, T, ctx->cfg.k, ctx->cfg.d, out, ctx->num_sms,
                                      static_cast<cudaStream_t>(stream)), "unpermute");
  return BG_OK;
}

// The fused chain a1-a9; seg != nullptr: token rows are read from / written to the segments' buffers.
static int do_forward(bg_moe_ctx* ctx, const void* hidden, int32_t T, void* out, cudaStream_t st,
                      const bg::SegTable* seg) {
  const bg_moe_config& c = ctx->cfg;
  int rc = do_route(ctx, hidden, T, nullptr, ctx->logits, ctx->topk_idx, ctx->topk_w, ctx->counts, ctx->offsets, st, seg);
  if (rc) return rc;
  mark(ctx, 3, st);
  BG_LAUNCH(ctx, bg::launch_rank(ctx->topk_idx, ctx->block_base, T, c.E, c.k, ctx->row_src, ctx->inv_perm, ctx->topk_w,
                                 ctx->w_perm, st), "rank");
  mark(ctx, 4, st);
  BG_LAUNCH(ctx, bg::launch_gather(hidden, ctx->inv_perm, T, c.k, c.d, ctx->x_perm, ctx->num_sms, st, seg), "gather");
  mark(ctx, 5, st);
  rc = do_ffn(ctx, ctx->x_perm, ctx->offsets, T, ctx->Y, ctx->topk_w, ctx->row_src, st, /*mark_between=*/6);
  if (rc) return rc;
  mark(ctx, 7, st);
  BG_LAUNCH(ctx, bg::launch_unpermute(ctx->Y, ctx->inv_perm, nullptr, T, c.k, c.d, out, ctx->num_sms, st, seg),
            "unpermute");
  mark(ctx, 8, st);
  ctx->profile_valid = ctx->profile;
  return BG_OK;
}

int bg_moe_combined_forward(bg_moe_ctx* ctx, const void* hidden, int32_t T, void* out, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!hidden || !out || !aligned16(hidden) || !aligned16(out)) return BG_ERR_INVALID_ARG;
  if (ctx->W_r == nullptr) return BG_ERR_NO_WEIGHTS;
  DeviceGuard guard(ctx->cfg.device);
  return do_forward(ctx, hidden, T, out, static_cast<cudaStream_t>(stream), nullptr);
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
  // The segment table goes to the device through pageable host staging: cudaMemcpyAsync from pageable
  // memory returns once the bytes are staged, so the vectors can be reused by the next call.
  const int n = n_segments;
  ctx->seg_host_ptrs.resize(2 * static_cast<size_t>(n));
  ctx->seg_host_start.resize(static_cast<size_t>(n) + 1);
  // an empty segment may carry null pointers (its rows are never looked up); the router uses hidden[0]
  // as the source address of zero-filled copies, so every entry is made a valid address
  const void* first_valid = nullptr;
  for (int i = 0; i < n && first_valid == nullptr; ++i)
    if (segments[i].n_tokens > 0) first_valid = segments[i].hidden;
  int32_t acc = 0;
  for (int i = 0; i < n; ++i) {
    ctx->seg_host_ptrs[i] = segments[i].n_tokens > 0 ? segments[i].hidden : first_valid;
    ctx->seg_host_ptrs[n + i] = segments[i].out;
    ctx->seg_host_start[i] = acc;
    acc += segments[i].n_tokens;
  }
  ctx->seg_host_start[n] = acc;
  BG_CUDA(ctx, cudaMemcpyAsync(ctx->seg_dev_hidden, ctx->seg_host_ptrs.data(), sizeof(void*) * n, cudaMemcpyHostToDevice, st),
          "H2D segment table (hidden)");
  BG_CUDA(ctx, cudaMemcpyAsync(ctx->seg_dev_out, ctx->seg_host_ptrs.data() + n, sizeof(void*) * n, cudaMemcpyHostToDevice, st),
          "H2D segment table (out)");
  BG_CUDA(ctx, cudaMemcpyAsync(ctx->seg_dev_start, ctx->seg_host_start.data(), sizeof(int32_t) * (n + 1),
                               cudaMemcpyHostToDevice, st), "H2D segment table (start)");
  bg::SegTable seg;
  seg.hidden = reinterpret_cast<const void* const*>(ctx->seg_dev_hidden);
  seg.out = reinterpret_cast<void* const*>(ctx->seg_dev_out);
  seg.start = ctx->seg_dev_start;
  seg.n = n;
  return do_forward(ctx, nullptr, T, nullptr, st, &seg);
}

int bg_moe_combined_forward_host(bg_moe_ctx* ctx, const void* hidden_host, int32_t T, void* out_host, void* stream) {
  int rc = check_T(ctx, T);
  if (rc) return rc;
  if (T == 0) return BG_OK;
  if (!hidden_host || !out_host) return BG_ERR_INVALID_ARG;
  DeviceGuard guard(ctx->cfg.device);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t bytes = static_cast<size_t>(T) * ctx->cfg.d * 2;
  BG_CUDA(ctx, cudaMemcpyAsync(ctx->hidden_dev, hidden_host, bytes, cudaMemcpyHostToDevice, st), "H2D hidden");
  rc = bg_moe_combined_forward(ctx, ctx->hidden_dev, T, ctx->out_dev, stream);
  if (rc) return rc;
  BG_CUDA(ctx, cudaMemcpyAsync(out_host, ctx->out_dev, bytes, cudaMemcpyDeviceToHost, st), "D2H out");
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
