/* bg_moe.h -- C ABI of the B200-native combined MoE layer (the hot path behind BatchGen's
 * `combine` primitive).
 *
 * What the library computes.  The paper's runtime yields sequence coroutines at the MoE module
 * boundary and COMBINEs them -- a concatenation of their hidden-state tensors (PAPER.md:192-194,
 * §4.2) -- so that each expert receives a larger batch; what then runs is
 *     h_out <- MoE(h_combined, l)            (Algorithm 1 line 8; prose PAPER.md:263)
 * The paper does not spell out the MoE arithmetic; BASELINE.json `north_star` fixes it (restated
 * in DESIGN.md §1): fp32 router -> top-k (ties to the lower expert index, softmax-renormalised
 * gates) -> per-expert histogram -> exclusive scan -> stable permutation into expert-contiguous
 * rows -> grouped SwiGLU expert FFN (gate/up GEMM, SiLU.mul, down GEMM) -> gate-weighted
 * un-permute that sums each token's top-k results in slot order.
 *
 * Conventions (all entry points):
 *  - Every data pointer is a DEVICE pointer owned by the caller (e.g. a torch tensor), 16-byte
 *    aligned, valid until the work enqueued on `stream` has completed.  The only HOST-pointer
 *    entry point is bg_moe_combined_forward_host (named so).  The library owns only its context
 *    and workspace.  Inputs are never modified; outputs are fully overwritten.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Every call
 *    is asynchronous on that stream: no host synchronisation, no allocation after bg_moe_create.
 *  - All tensors are row-major (last index contiguous).  bf16 tensors are passed as void*.
 *    T = combined tokens, d = hidden, E = experts, k = top-k, f = expert intermediate, R = T*k.
 *  - Indices are int32 (R <= 2^31-1); byte offsets are computed in 64 bits.
 *  - Return value: BG_OK (0) or a negative bg_moe_status.  Nothing aborts or throws across the
 *    ABI.  T == 0 is BG_OK and a no-op.  A context is not thread-safe: one call at a time, and the
 *    calls made on one context must be STREAM-ORDERED with respect to each other (same stream, or
 *    streams the caller orders with events): they share the context's workspace and tile counters.
 *  - Supported ranges: 1 <= E <= 256, 1 <= k <= min(E, 8), d and f multiples of 8 (d >= 64,
 *    f >= 64), 0 <= T <= max_tokens.  Device must be sm_100 (B200).  There is no CPU fallback.
 */
#ifndef BG_MOE_H_
#define BG_MOE_H_

#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bg_moe_ctx bg_moe_ctx;

typedef enum {
  BG_OK = 0,
  BG_ERR_INVALID_ARG = -1,  /* NULL, T<0, T>max_tokens, k<1, k>E, misaligned pointer, d/f not /8 */
  BG_ERR_UNSUPPORTED = -2,  /* E>256, k>8, gate_fn != 0, device is not sm_100 */
  BG_ERR_CUDA = -3,         /* a CUDA call failed; bg_moe_last_error(ctx) has the string */
  BG_ERR_NOMEM = -4,        /* workspace allocation failed */
  BG_ERR_NO_WEIGHTS = -5    /* bg_moe_set_weights has not been called */
} bg_moe_status;

typedef struct {
  int32_t d;          /* hidden size */
  int32_t f;          /* expert intermediate size */
  int32_t E;          /* number of routed experts */
  int32_t k;          /* experts per token */
  int32_t max_tokens; /* workspace is sized for T <= max_tokens */
  int32_t gate_fn;    /* 0 = softmax over the k selected logits (the only one defined) */
  int32_t device;     /* CUDA device ordinal */
} bg_moe_config;

/* Allocates the context and its device workspace (logits, routing tables, x_perm, H, Y).
 * *out is set only on BG_OK. */
int bg_moe_create(const bg_moe_config* cfg, bg_moe_ctx** out);
int bg_moe_destroy(bg_moe_ctx* ctx);

/* Borrows (does not copy) the layer's parameters.  W_r fp32 [d,E]; b_r fp32 [E] or NULL (reading
 * S7: added to the logits in fp32, used for selection and gates); W_gate, W_up bf16 [E,d,f];
 * W_down bf16 [E,f,d].  Consumed in these layouts as given (reading S14). */
/* Asynchronous on `stream` like every other call: the only device work is the exact bf16 three-way
 * split of W_r (read on `stream`, so a W_r produced on that stream is ordered before it). */
int bg_moe_set_weights(bg_moe_ctx* ctx, const float* W_r, const float* b_r, const void* W_gate,
                       const void* W_up, const void* W_down, void* stream);

/* Expert-weight ring buffer.  The paper keeps model parameters in host memory -- "a single
 * source of truth ... Parameter movement is unidirectional: host memory serves as the source for GPU
 * prefetching" -- and streams the experts of a module through a GPU-side "ring parameter buffer" whose slot
 * ownership "is released after the module completes execution" (§5.2, Fig. 7a), "fully
 * overlapping parameter transfers with computation" (§6.5).
 *   W_r, b_r                      DEVICE, as in bg_moe_set_weights (the router stays resident: 4 d E bytes)
 *   W_gate_host, W_up_host, W_down_host   HOST pointers (pinned memory, or the copies are not asynchronous), the
 *                                 same layouts as the resident tensors; borrowed, must outlive the calls
 *   ring_experts                  even, >= 2: the device ring holds this many experts' weights in two halves
 *                                 (6 d f ring_experts bytes, allocated here, at set-up time)
 * Afterwards bg_moe_combined_forward (and the _segments / _host forms) runs the expert FFN chunk by chunk:
 * ring_experts/2 experts are copied into one half on a stream the context owns while the grouped GEMMs of the
 * previous chunk run out of the other half.  Same kernels, same per-row arithmetic: results are bit-identical to
 * the resident path.  By default every expert is copied (which experts are empty is known only on the device; no
 * host synchronisation is taken) -- see bg_moe_set_ring_skip_empty.  The split calls (bg_moe_expert_ffn) need
 * resident weights. */
int bg_moe_set_weights_offloaded(bg_moe_ctx* ctx, const float* W_r, const float* b_r, const void* W_gate_host,
                                 const void* W_up_host, const void* W_down_host, int32_t ring_experts,
                                 void* stream);
/* Skip the experts nobody was routed to (the ring holds "the running and prefetching expert";
 * offloaded experts are streamed only when they run).  With enable != 0 a fused call on offloaded
 * weights reads its own per-expert counts back into pinned memory (copied on the ring's stream as soon as the
 * router kernel has finished, while the gather runs) and copies into the ring only the experts that received at
 * least one row; chunks with no such expert are skipped altogether.  Same kernels, same rows: the result stays
 * bit-identical to the resident path.  Cost: ONE host synchronisation per call -- the calling thread blocks until
 * this call's router has finished (and so until everything queued before it on `stream` has) -- which is why it is
 * opt-in; it pays when routing is skewed (BASELINE config C4: ~60 of 256 experts are empty at T = 8192) and the
 * step is bound by the PCIe copy anyway.  Set-up time allocation: E pinned ints.  No effect on resident weights. */
int bg_moe_set_ring_skip_empty(bg_moe_ctx* ctx, int32_t enable);
/* Host -> device bytes the ring copied during the last fused call (0 with resident weights). */
int64_t bg_moe_ring_bytes_per_call(const bg_moe_ctx* ctx);

/* FP8 expert GEMM.  The paper's MoE GEMMs run in FP8 ("FP8 MoE GEMMs",
 * PAPER.md:442 FP8 DeepSeek-R1 / Kimi-K2 weights, PAPER.md:476-478 FP8 decoding) with no recipe given; readings F1-F4
 * of DESIGN.md §2: OCP e4m3, round-to-nearest-even, saturating; activations one fp32 scale per token row
 * (max|x| / 448), weights one fp32 scale per expert and output channel; the gate/up GEMM runs W8A8 on
 * tcgen05 kind::f8f6f4 with fp32 accumulation and the scales applied in its epilogue before the SwiGLU; H and the
 * down GEMM stay bf16 (precision 1).  Precision 2 (reading F5) runs the down GEMM W8A8 as well: the gate/up epilogue
 * keeps the row maximum of |H| (integer max on float bits: order-independent), a quantising pass turns the bf16 H
 * into e4m3 rows with one scale per row, W_down is quantised per expert and output channel.
 *   precision 0: bf16 (default);  1: FP8 gate/up;  2: FP8 gate/up and down.
 * Switching to 1 / 2 quantises the resident bf16 weights on `stream` into library-owned buffers ([E, f, d] / [E, d, f]
 * e4m3 bytes + per-channel scales; 3 E d f bytes, allocated at the first switch) -- call it again after
 * bg_moe_set_weights.  It applies to the fused calls (bg_moe_combined_forward and its _segments / _host forms); the
 * split calls and the offloaded-weights path stay bf16.  BG_ERR_UNSUPPORTED unless d % 128 == 0 and f % 64 == 0
 * (precision 2: f % 128 == 0). */
int bg_moe_set_precision(bg_moe_ctx* ctx, int32_t precision, void* stream);
/* Device pointers to the FP8 artefacts of the last fused call / last quantisation (any out-pointer may be NULL):
 * xq_perm e4m3 [T*k, d] and sx_perm fp32 [T*k] in expert order; q_gate / q_up e4m3 [E, f, d]; sw_gate / sw_up fp32 [E, f]. */
int bg_moe_debug_fp8_views(bg_moe_ctx* ctx, const void** xq_perm, const float** sx_perm, const void** q_gate,
                           const float** sw_gate, const void** q_up, const float** sw_up);
/* Precision 2: H bf16 [T*k, f] (workspace), its codes hq e4m3 [T*k, f] and scales sh_perm fp32 [T*k] of the last fused
 * call; q_down e4m3 [E, d, f], sw_down fp32 [E, d]. */
int bg_moe_debug_fp8_down_views(bg_moe_ctx* ctx, const void** H, const void** hq, const float** sh_perm,
                                const void** q_down, const float** sw_down);

/* Debug / test switches of the grouped-GEMM tile scheduler; production never calls this.
 *   static_tile_feed != 0     tile t -> cluster (t mod #clusters) instead of the dynamic ticket feed
 *   supergroup_token_tiles    > 0: token tiles per super-group (forces the super-group order on small
 *                             shapes); 0: sized from K so that a super-group's tokens fit ~48 MB of L2
 *   router_form               0: the router picks its form from T; 1: sequential form (one CTA per 128-token
 *                             tile) wherever it exists; 2: cluster form.  Both forms give the same bits. */
int bg_moe_set_debug(bg_moe_ctx* ctx, int32_t static_tile_feed, int32_t supergroup_token_tiles,
                     int32_t router_form);

/* Steps a1-a4: router logits, top-k + gates, histogram, exclusive scan.
 *   hidden     bf16 [T,d]
 *   logits_in  NULL, or fp32 [T,E]: use these logits instead of computing a1
 *   logits_out NULL, or fp32 [T,E]: receives the logits used
 *   topk_idx   int32 [T,k]  slot s = s-th largest under (logit desc, expert index asc)
 *   topk_w     fp32 [T,k]   softmax over the k selected logits
 *   counts     int32 [E];  offsets int32 [E+1], offsets[E] = T*k */
int bg_moe_route(bg_moe_ctx* ctx, const void* hidden, int32_t T, const float* logits_in,
                 float* logits_out, int32_t* topk_idx, float* topk_w, int32_t* counts,
                 int32_t* offsets, void* stream);

/* Steps a2-a4 from given logits WITHOUT any allocation and without a context: the same results as
 * bg_moe_route(ctx, NULL, T, logits, NULL, ...) -- same selection order, same gate arithmetic, same
 * counts / offsets.
 *
 * Why it exists.  bg_moe_create cudaMallocs a workspace, and some users of this library cannot do
 * that: a serving runtime that has already given all of HBM to pools it manages itself (the paper's
 * runtime fills the device with KV cache and its ring parameter buffer, so a
 * library-side cudaMalloc fails or eats memory its planner counted on), and code on a
 * latency-critical path where cudaMalloc / cudaFree are banned because they serialise with all work
 * in flight on the device.  This call allocates nothing -- no cudaMalloc, no cudaFree, no
 * allocating library routine, on any call -- because the only global memory it needs beyond its
 * arguments (per-tile expert histograms and a tile ticket) is a fixed array inside the library image.
 *
 * The price, all of it a consequence of that array:
 *  - Limit: T <= BG_MOE_NOALLOC_MAX_TOKENS and E <= 256 (k <= 8).  A larger T is refused with
 *    BG_ERR_INVALID_ARG and a message saying so in bg_moe_noalloc_last_error(); nothing is launched.
 *  - Footprint: 131,328 bytes of device memory on EVERY GPU that loads the library, held until the
 *    process exits whether or not this call is ever made.
 *  - One array per GPU, shared by all calls, threads and streams.  Two calls whose kernels can be on
 *    the same GPU at the same time (different streams without an event between them) RACE on it and
 *    produce garbage counts; calls on one stream, or ordered by events, are fine.  The array keeps
 *    the previous call's contents; the call clears the one word that has to start at zero itself.
 *  - The call works on the CURRENT device: `stream` and every pointer must belong to it.  The first
 *    call on each device looks up that device's copy of the array (cudaGetSymbolAddress, which may
 *    make the runtime load the library's kernels onto the device); make that first call during
 *    set-up, before any stream capture is begun.  Later calls only enqueue a 256-byte memset and
 *    one kernel on `stream`.
 *
 *   logits    DEVICE fp32 [T,E] (row-major), read only
 *   topk_idx  DEVICE int32 [T,k]; topk_w DEVICE fp32 [T,k]   (may be NULL only when T == 0)
 *   counts    DEVICE int32 [E];   offsets DEVICE int32 [E+1], offsets[E] = T*k
 * T == 0 writes zero counts / offsets.  All buffers are the caller's; the call is asynchronous on
 * `stream` and never synchronises.  Returns BG_OK, BG_ERR_INVALID_ARG, BG_ERR_UNSUPPORTED (E > 256,
 * k > 8, device not sm_100) or BG_ERR_CUDA. */
#define BG_MOE_NOALLOC_MAX_TOKENS 16384
int bg_moe_route_logits_noalloc(const float* logits, int32_t T, int32_t E, int32_t k,
                                int32_t* topk_idx, float* topk_w, int32_t* counts, int32_t* offsets,
                                void* stream);
/* Why the calling thread's last bg_moe_route_logits_noalloc failed ("" after a success).  The
 * string is thread-local and owned by the library. */
const char* bg_moe_noalloc_last_error(void);

/* Steps a5-a6: stable counting sort of flat index i = t*k+s by expert, and the row gather.
 *   topk_idx int32 [T,k], every entry in [0,E).  Any list is sorted correctly: a token may name the
 *            same expert in several slots (each entry gets its own row, lower slot first).
 *   offsets  int32 [E+1]: must be the exclusive scan of topk_idx's histogram (what bg_moe_route
 *            returned for these indices).  The permutation is rebuilt from topk_idx alone; offsets is
 *            not read, and a table that disagrees with topk_idx does not change the result.
 *   row_src  int32 [T*k]: row_src[r] = i;   inv_perm int32 [T*k]: inv_perm[i] = r
 *   x_perm   bf16 [T*k,d]: x_perm[r,:] = hidden[row_src[r]/k,:]   (may be NULL: skip the gather) */
int bg_moe_permute(bg_moe_ctx* ctx, const void* hidden, int32_t T, const int32_t* topk_idx,
                   const int32_t* offsets, int32_t* row_src, int32_t* inv_perm, void* x_perm,
                   void* stream);

/* Steps a7-a8, un-fused form: y_perm[r,:] = (silu(x W_gate[e]) . (x W_up[e])) W_down[e] for the
 * rows r in [offsets[e], offsets[e+1]); bf16 in, fp32 accumulate, H rounded to bf16 between the
 * two GEMMs, y_perm bf16 [T*k,d] in expert order, NOT gate-weighted. */
int bg_moe_expert_ffn(bg_moe_ctx* ctx, const void* x_perm, const int32_t* offsets, int32_t T,
                      void* y_perm, void* stream);

/* Step a9, un-fused form: out[t,:] = sum_{s<k} topk_w[t,s] * y_perm[inv_perm[t*k+s],:], summed in
 * slot order in fp32, rounded once (RNE) to bf16.  No floating-point atomics. */
int bg_moe_unpermute(bg_moe_ctx* ctx, const void* y_perm, const int32_t* inv_perm,
                     const float* topk_w, int32_t T, void* out, void* stream);

/* The fused chain a1-a9 on the context's workspace: hidden bf16 [T,d] -> out bf16 [T,d].
 * Same math as the split calls except that the down-GEMM epilogue applies the gate weight (in
 * fp32, before the bf16 rounding of Y) and the final reduce only sums. */
int bg_moe_combined_forward(bg_moe_ctx* ctx, const void* hidden, int32_t T, void* out, void* stream);

/* Zero-copy COMBINE (Algorithm 1 l.7; Table 2 "COMBINE without offloading: 0 (GPU
 * resident)"): the combined batch given as the list of the yielded coroutines' own buffers instead of
 * one concatenated tensor.  Segment s holds n_tokens rows of bf16 [n_tokens, d] at `hidden` (device,
 * 16-byte aligned) and receives its rows of the result at `out`; the combined token order is the list
 * order (token t of the batch = row t - sum_{s'<s} n_tokens_{s'} of segment s).  `segments` is a HOST
 * array, copied to the device on `stream`; 0 <= n_segments <= max_tokens, sum of n_tokens <= max_tokens;
 * empty segments are allowed.  The result is bit-identical to bg_moe_combined_forward on the
 * concatenation: the router, the gather and the un-permute address rows through the segment table,
 * every other kernel is the same. */
typedef struct {
  const void* hidden;   /* device, bf16 [n_tokens, d] */
  void* out;            /* device, bf16 [n_tokens, d] */
  int32_t n_tokens;
} bg_moe_segment;
int bg_moe_combined_forward_segments(bg_moe_ctx* ctx, const bg_moe_segment* segments,
                                     int32_t n_segments, void* stream);

/* Same, but `hidden_host` and `out_host` are HOST pointers (pinned memory, or the copies are not
 * asynchronous): hidden host->device, the fused chain, out device->host.  The three run on streams the
 * context owns, over two staging slots, so that consecutive calls overlap the upload of call i+1 and the
 * download of call i-1 with the GEMMs of call i.
 * Ordering and lifetime of the two host buffers:
 *  - The upload does NOT run on `stream` and does not wait for it (if it did, call i+1's upload would
 *    queue behind call i's download and nothing would overlap).  hidden_host must therefore hold its
 *    data when the call is made -- work still pending on `stream` that fills it (a D2H copy, a host
 *    function) is NOT ordered before the upload; finish it first.
 *  - hidden_host is read asynchronously after the call returns: keep it alive and unmodified until the
 *    upload has finished.  bg_moe_host_input_sync(ctx) blocks the calling thread until the upload of the
 *    most recent host call is done (it does not wait for the GEMMs); a synchronize on `stream` after the
 *    call implies it too.  A caller cycling through >= 2 input buffers needs neither.
 *  - The call is ordered after every earlier call on the context; `stream` is made to wait for the
 *    download, so work enqueued on `stream` afterwards -- or a synchronize on it -- sees out_host
 *    complete.  out_host must stay alive until then. */
int bg_moe_combined_forward_host(bg_moe_ctx* ctx, const void* hidden_host, int32_t T,
                                 void* out_host, void* stream);
/* Blocks until the host->device upload of the most recent bg_moe_combined_forward_host call has
 * finished, i.e. until that call's hidden_host may be overwritten or freed.  BG_OK at once if no
 * host call has been made. */
int bg_moe_host_input_sync(bg_moe_ctx* ctx);

/* Device pointers into the workspace holding the routing artefacts of the LAST fused call
 * (valid until the next call on this context).  Any out-pointer may be NULL. */
int bg_moe_debug_views(bg_moe_ctx* ctx, const float** logits, const int32_t** topk_idx,
                       const float** topk_w, const int32_t** counts, const int32_t** offsets,
                       const int32_t** row_src, const int32_t** inv_perm);

/* The two intermediates of the expert FFN of the LAST fused call, in expert order (row r = the r-th row of
 * row_src): H bf16 [T*k, f] = silu(x W_gate) . (x W_up), and Y bf16 [T*k, d] = the down GEMM's output,
 * already multiplied by the row's gate weight in the fused chain.  Workspace pointers, valid until the next
 * call on this context; either out-pointer may be NULL.  For tests that check one expert's rows. */
int bg_moe_debug_ffn_views(bg_moe_ctx* ctx, const void** H, const void** Y);

/* Per-kernel timing of the fused chain.  While enabled, bg_moe_combined_forward records a CUDA
 * event on `stream` before and after each of its BG_MOE_NUM_STAGES kernels (in launch order:
 * fused router (logits, top-k, histogram, scan, tile ranks), gather (+ permutation), gate/up
 * GEMM+SwiGLU, down GEMM, un-permute reduce); bg_moe_expert_ffn records its two GEMMs in the same
 * slots (the other three read 0).
 * bg_moe_profile_read waits for the last recorded call and writes that call's per-kernel
 * durations in milliseconds to ms_out[BG_MOE_NUM_STAGES] (HOST pointer). */
#define BG_MOE_NUM_STAGES 5
int bg_moe_profile_enable(bg_moe_ctx* ctx, int enable);
int bg_moe_profile_read(bg_moe_ctx* ctx, float* ms_out);

/* Number of kernels this library has launched through `ctx` since creation. */
int64_t bg_moe_launch_count(const bg_moe_ctx* ctx);
/* Bytes of device workspace owned by `ctx`. */
int64_t bg_moe_workspace_bytes(const bg_moe_ctx* ctx);

/* ---- Module-level roofline fit and B_moe choice (host only; no GPU work, no context needed) -------
 * The paper plans the MoE batch statically: "a module-level roofline model enables static planning
 * for batch accumulation ... we can select the largest feasible module batch size that remains
 * within memory constraints" (§5.1); the model is fitted to profiled runtimes of the
 * module "over multiple batch sizes" (§5.4).  Here the module is this library's fused
 * chain, the profile is bench.py's combine-size sweep, and memory is the context's workspace.
 *
 * Model: t(T) = max(t_floor_ms, t0_ms + ms_per_token * T) -- flat while the expert weights bound
 * the step (small combined batches), linear once the tensor cores do.  Utilisation of a batch of T
 * tokens = its token rate relative to the asymptotic rate: u(T) = ms_per_token * T / t(T). */
typedef struct {
  double t_floor_ms;    /* weight-bound floor */
  double t0_ms;         /* intercept of the compute-bound line */
  double ms_per_token;  /* slope of the compute-bound line (> 0) */
  double ridge_tokens;  /* where the two meet: (t_floor_ms - t0_ms) / ms_per_token */
  double rms_rel_err;   /* root mean square of (model - measured) / measured over the fitted points */
} bg_moe_fit;

/* Least-squares fit of the model to n >= 3 measured points (tokens strictly increasing, ms > 0; HOST
 * pointers): every split "first j points flat, the rest on a line" (1 <= j <= n-2) is tried, the flat
 * level is the mean of its points and the line the ordinary least-squares line of its points; the
 * split with the smallest sum of squared relative errors of max(flat, line) wins (lowest j on ties).
 * BG_ERR_INVALID_ARG if no split has a positive slope. */
int bg_moe_fit_roofline(const int32_t* tokens, const double* ms, int32_t n, bg_moe_fit* out);

/* Bytes of device workspace a context with this config and max_tokens = tokens would allocate
 * (what bg_moe_create allocates on a 148-SM B200; cfg->max_tokens and cfg->device are ignored). */
int bg_moe_workspace_bytes_for(const bg_moe_config* cfg, int32_t tokens, int64_t* bytes_out);

/* B_moe: *tokens_out = the SMALLEST multiple of `granularity` (>= 1) whose model utilisation reaches
 * target_util (0 < target_util < 1), capped at the LARGEST multiple of `granularity` whose workspace
 * fits in memory_budget_bytes; *reached_out (may be NULL) = 1 if the target was reached under the
 * cap, 0 if the cap bound it.  BG_ERR_NOMEM if not even `granularity` tokens fit. */
int bg_moe_choose_tokens(const bg_moe_config* cfg, const bg_moe_fit* fit, double target_util,
                         int64_t memory_budget_bytes, int32_t granularity, int32_t* tokens_out,
                         int32_t* reached_out);

const char* bg_moe_strerror(int status);
/* Text of the last CUDA error seen by `ctx` ("" if none).  Owned by the context. */
const char* bg_moe_last_error(const bg_moe_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* BG_MOE_H_ */
