/* dlm.h -- C ABI of the B200-native denoising-step library (libdlm.so).
 *
 * One confidence-thresholded denoising step of a masked diffusion language model under approximate
 * (block-wise, prefix + suffix) KV caching: the GPU work a TeDiServe model instance performs for each
 * scheduler command.  Citations are to /root/reference/PAPER.md as P:<line>.
 *
 *   - the executor command carries "the request prompt and output length (if not already present), the set
 *     of tokens unmasked in the previous denoising step, and the selected confidence threshold" and
 *     the reply carries "the newly unmasked tokens and confidence statistics";
 *   - "cache steps compute only the tokens inside the current cache block, while recompute steps process
 *     all tokens in the sequence"; here recompute step = dlm_refresh_step, cache step = dlm_cached_step;
 *   - every step ends by unmasking "tokens whose confidence exceeds a predefined threshold. If no predicted
 *     tokens have confidence exceeding the threshold, the token with the highest confidence is unmasked";
 *   - "one-time latency profiling step to measure the per-denoising-step latency for each batch size"
 *     = dlm_profile_step_costs.
 *
 * Conventions.  All functions return 0 (DLM_OK) or a negative DLM_E_* code; dlm_last_error() gives the text.
 * Nothing is partially applied on error.  Calls are synchronous (results are in the caller's HOST buffers at
 * return) and a ctx must be used from one thread at a time.  The library owns every device allocation; the
 * caller owns every host buffer it passes.  Unless stated otherwise pointers are HOST pointers.
 * There is no CPU fallback: without a CUDA device every compute entry point returns DLM_E_CUDA.
 */
#ifndef DLM_H_
#define DLM_H_

#include <stddef.h>
#include <stdint.h>

#ifndef DLM_API
#define DLM_API __attribute__((visibility("default")))
#endif

#ifdef __cplusplus
extern "C" {
#endif

#define DLM_OK          0
#define DLM_E_ARG      (-1)   /* bad argument (null pointer, length, G % B != 0, unknown request ...) */
#define DLM_E_CAPACITY (-2)   /* request table, page pool, token budget or caller's result buffer too small */
#define DLM_E_STATE    (-3)   /* cached step without a valid cache, step on a removed request ...       */
#define DLM_E_CUDA     (-4)   /* CUDA error or no device                                                */

#define DLM_DTYPE_F32   0
#define DLM_DTYPE_BF16  1
#define DLM_DTYPE_BF16_PRECISE 2   /* precise mode (SURVEY 8(c) protocol P-D): the bf16 model's weight VALUES (Definition W rounded
                                      to bf16) held in fp32, activations, K/V store and every product in fp32 on the plain CUDA
                                      kernels.  No activation is rounded to bf16, so committed tokens match the fp64 oracle
                                      outside the 1e-3 band; slow (SIMT), for parity runs.  Chosen at init because it changes
                                      the storage type of the weights and of the K/V pages (it is SURVEY's DLM_OPT_PRECISE). */

typedef struct dlm_ctx dlm_ctx;          /* opaque; owns all device memory */

/* Model shape ("arch") and capacities.  Weights are [out, in] row-major; no biases; RMSNorm gains are 1. */
typedef struct {
  int32_t n_layers, d_model, n_heads, n_kv_heads, head_dim, d_ffn, vocab, mask_id;
  int32_t weight_dtype;          /* DLM_DTYPE_F32: fp32 weights, all-fp32 arithmetic (config 1);
                                    DLM_DTYPE_BF16: bf16 weights, tcgen05 GEMMs, fp32 accumulate/residual;
                                    DLM_DTYPE_BF16_PRECISE: bf16 weight values, all-fp32 arithmetic        */
  float   logit_scale, rms_eps, rope_theta, init_std;
  int32_t max_requests;          /* request slots (cf. maxNumSeqPerBatch)                       */
  int32_t max_seq;               /* longest prompt + generation per request                             */
  int32_t max_block;             /* largest denoising block length B (<= 64)                            */
  int32_t kv_page_tokens;        /* tokens per K/V page (64)                                            */
  int32_t max_batch_tokens;      /* most tokens one step may compute (sum of S_r in a refresh batch)    */
  int64_t kv_pool_tokens;        /* total tokens the paged K/V store can hold (0 => max_requests*max_seq) */
} dlm_arch;

/* Optional memory / stream provider: lets the Python harness hand out torch-owned device memory and a torch
 * stream ("PyTorch only for device memory and streams").  NULL callbacks => cudaMalloc / cudaFree; NULL stream
 * => a stream the library creates. alloc returns a DEVICE pointer (256-byte aligned) or NULL. */
typedef struct {
  void* (*alloc)(size_t bytes, void* user);
  void  (*free)(void* dev_ptr, void* user);
  void*  user;
  void*  cuda_stream;            /* cudaStream_t */
} dlm_mem;

#define DLM_DRY_RUN 1u           /* compute and report, mutate nothing but the K/V store */

/* One batch of requests for one step. */
typedef struct {
  int32_t        n;              /* number of requests                                                  */
  const int32_t* req;            /* [n] request handles from dlm_request_add, distinct                  */
  const float*   threshold;      /* [n] or NULL => each request's stored threshold                      */
  uint32_t       flags;          /* DLM_DRY_RUN                                                         */
} dlm_batch;

/* Step result, caller-owned host buffers.  Commits are packed request by request in batch order, positions
 * ascending inside a request; pos is the absolute index in prompt||generation. */
typedef struct {
  int32_t* n_committed;          /* [n] out: commits of request i                                       */
  int32_t* pos;                  /* [capacity] out                                                      */
  int32_t* tok;                  /* [capacity] out                                                      */
  float*   conf;                 /* [capacity] out: softmax probability of the committed token          */
  int32_t  capacity;             /* in: entries available in pos/tok/conf (n*max_block always suffices) */
  int32_t  total;                /* out: sum of n_committed                                             */
  int32_t* n_masked_left;        /* [n] out, may be NULL: MASK positions left in the request            */
  float*   lse;                  /* [n*max_block] out, may be NULL: log-sum-exp of each block row       */
  float*   row_conf;             /* [n*max_block] out, may be NULL: confidence of each block row        */
  int32_t* row_tok;              /* [n*max_block] out, may be NULL: predicted token of each block row   */
  float*   features;             /* [n*DLM_N_FEATURES] out, may be NULL: the Step Predictor's features of each request after
                                    this step ("confidence statistics", App. A), in the paper's order:
                                    confidence_threshold, output_length, full_progress, full_unmask_progress, block_progress,
                                    block_unmask_progress, output_{min, q25, median, avg, q75}_confidence.  An output token's
                                    confidence is the one its position last had while masked (frozen at commit, 0 before any
                                    step evaluated it); quartiles by linear interpolation; computed on the device.            */
} dlm_result;
#define DLM_N_FEATURES 11

#define DLM_KIND_REFRESH 0
#define DLM_KIND_CACHED  1
/* One row of the per-step cost table (the paper's latencyProfile[tp][batch], tp = 1,
 * split by step kind as Algorithms 4/5 use it, with the K/V length added). */
typedef struct { int32_t kind, n_requests, n_tokens, kv_tokens; float usec; } dlm_cost_row;

/* dlm_init: build a model instance; weights are generated ON THE DEVICE from `seed` by the counter-based
 * definition W in DESIGN.md (the paper gives no weights; BASELINE.json: "random-init ~N(0,0.02) from seed"). */
DLM_API int  dlm_init(const dlm_arch* arch, uint64_t seed, dlm_ctx** out);
DLM_API int  dlm_init_ex(const dlm_arch* arch, uint64_t seed, const dlm_mem* mem, dlm_ctx** out);
DLM_API void dlm_destroy(dlm_ctx* ctx);

/* Register a request: prompt ids [prompt_len] (host), generation of gen_len positions initialised to [MASK]
 * ("starting from a fully corrupted sequence containing only [MASK] tokens") in blocks of block_len
 * (P:109).  gen_len % block_len must be 0 (P:380 outputs are rounded up to the block size).  *out_req is the
 * handle.  dlm_request_set_tokens overwrites prompt||generation ([S] ids, host): it constructs mid-flight state
 * (the constructed phases of configs 3/5) and applies tokens decided elsewhere (a command carries "the set
 * of tokens unmasked in the previous denoising step").  keep_cache = 0 invalidates the request's K/V cache;
 * keep_cache = 1 leaves the K/V store and its validity untouched (the approximate cache tolerates stale K/V by
 * design) unless the current block changes, which always invalidates. */
DLM_API int  dlm_request_add(dlm_ctx*, const int32_t* prompt, int32_t prompt_len, int32_t gen_len,
                     int32_t block_len, float threshold, int32_t* out_req);
DLM_API int  dlm_request_set_tokens(dlm_ctx*, int32_t req, const int32_t* tokens, int32_t n, int32_t keep_cache);
DLM_API int  dlm_request_remove(dlm_ctx*, int32_t req);
DLM_API int  dlm_request_tokens(dlm_ctx*, int32_t req, int32_t* out, int32_t cap);     /* returns S or error    */
DLM_API int  dlm_request_info(dlm_ctx*, int32_t req, int32_t* cur_block, int32_t* cache_valid, int32_t* n_masked);

/* Migration ("a request may be migrated to another instance only at recompute steps",
 * P:365 the executor command carries the request's tokens).  dlm_request_export serialises what a request is apart
 * from its K/V cache -- prompt||generation ids, block length, threshold, completed-step count and the per-position
 * confidence state of the Step Predictor features -- into a caller-owned HOST blob and returns the blob size in
 * bytes (nothing is written when cap_bytes is smaller; call with blob = NULL to size it).  Layout, little-endian:
 * int32 {magic 0x524D4C44 "DLMR", version 1, prompt_len, gen_len, block_len, steps_done, cache_valid_at_export,
 * reserved}, float threshold, int32 reserved, int32 tokens[S], float conf_state[S].  dlm_request_import registers
 * the blob as a new request of ctx (which may be another context, on another GPU, of the same arch): the cache is
 * INVALID, so the next step must be dlm_refresh_step, which recomputes every K/V.  Exported at a block's first step
 * (cache invalid there anyway) the imported request continues bit-identically; exported mid-block it continues with
 * a fresh cache instead of the approximate one (legal, G19, but not the same trajectory).  Errors: DLM_E_ARG for a
 * malformed blob or ids outside the vocabulary, DLM_E_CAPACITY as dlm_request_add; nothing is applied on error. */
DLM_API int64_t dlm_request_export(dlm_ctx*, int32_t req, void* blob, int64_t cap_bytes);
DLM_API int  dlm_request_import(dlm_ctx*, const void* blob, int64_t bytes, int32_t* out_req);

/* Recompute step: all S_r positions of every request in the batch pass through the model,
 * every layer's K (post-RoPE) and V are written to the request's pages, then the current block (the
 * lowest-index block holding a MASK) is unmasked with the batch's / stored threshold.  Legal at any time;
 * required at a block's first step.  A finished request commits 0. */
DLM_API int  dlm_refresh_step(dlm_ctx*, const dlm_batch*, dlm_result*);

/* Cache step: only the current block's B_r positions are computed; they attend, without any
 * mask, to their own fresh K/V plus the cached K/V of every other position.  per_request_threshold
 * ([n], may be NULL) overrides batch->threshold, which overrides the stored value (the threshold may
 * change at every step).  DLM_E_STATE if a request's cache is not valid (new request, block just completed). */
DLM_API int  dlm_cached_step(dlm_ctx*, const dlm_batch*, const float* per_request_threshold, dlm_result*);

/* Mixed step (P:616-618 batches are sized by their total token count, whatever the kinds):
 * ONE ragged launch in which every request of the batch takes the step kind that is due -- a recompute step if
 * its cache is not valid (new request, block just completed), a cache step otherwise.  Results per request are
 * those of dlm_refresh_step / dlm_cached_step on that request alone (requests are independent, G17); the weights
 * are streamed once for the whole batch instead of once per kind.  Thresholds as in dlm_cached_step. */
DLM_API int  dlm_mixed_step(dlm_ctx*, const dlm_batch*, const float* per_request_threshold, dlm_result*);

/* One-time latency profiling: times synthetic refresh and cached steps over a grid of (requests,
 * tokens, K/V length) with CUDA events and fills rows[0..*n_rows).  Uses scratch requests; needs free slots. */
DLM_API int  dlm_profile_step_costs(dlm_ctx*, dlm_cost_row* rows, int32_t cap, int32_t* n_rows);
/* The same with the denoising block length B (<= max_block; dlm_profile_step_costs uses min(32, max_block)) and the number of
 * timed repeats per row (at least 10 are always taken; a row is their MEDIAN, after two untimed runs).  Rows:
 *   DLM_KIND_CACHED   n in {1,2,4,8,16,32,64} requests x per-request K/V length in {512,1024,2048,4608}: n_tokens = n*B
 *                     (the paper's index cacheBlockSize x numReqs; K/V length added), caches built untimed;
 *   DLM_KIND_REFRESH  total tokens 128, 256, ... 32768 (LP[tp][numTokens]) as one request while it fits max_seq,
 *                     then as several requests of the largest power of two <= max_seq (kv_tokens = tokens per request).
 * Combinations that exceed max_requests, max_seq, max_batch_tokens or the free K/V pages are skipped. */
DLM_API int  dlm_profile_step_costs_ex(dlm_ctx*, int32_t block_len, int32_t repeats, dlm_cost_row* rows, int32_t cap, int32_t* n_rows);

/* Options. */
#define DLM_OPT_SIMPLE_KERNELS 1   /* 1: run the bf16 model through the plain SIMT kernels (on-device debugging
                                      reference; same rounding points as the tcgen05 path; not a CPU fallback) */
#define DLM_OPT_DEBUG_DUMP     2   /* 1: keep every stage tensor of the next steps for dlm_debug_tensor      */
#define DLM_OPT_CUDA_GRAPH     3   /* 1 (default): replay steps of a batch shape seen before from a captured CUDA graph */
#define DLM_OPT_FLASH_ATTENTION 4  /* 0: use the plain attention kernel in the bf16 path (debugging)          */
#define DLM_OPT_KERNEL_TIMING  5   /* 1: bracket every kernel launch of the next steps with CUDA events (dlm_kernel_times) */
#define DLM_OPT_PDL            6   /* 1 (default): programmatic dependent launch between the kernels of a step           */
#define DLM_OPT_SKINNY_GEMM    7   /* 1 (default): weight-streaming split-K GEMM for steps of <= 128 tokens; 0: tile GEMM */
#define DLM_OPT_TC_ATTENTION   9   /* 1 (default): tcgen05/TMEM attention kernel when a step has enough (request, head) work; 0: mma.sync kernel */
#define DLM_OPT_FUSE_ROPE     10   /* 1 (default): above 128 tokens RoPE + K/V page write run in the QKV GEMM's epilogue; 0: separate kernel */
#define DLM_OPT_PAIR_GEMM      8   /* 1 (default): persistent CTA-pair (cta_group::2) GEMM above 128 tokens; 0: single-CTA tile GEMM */
#define DLM_OPT_TRACE         11   /* 1: every kernel of the next steps stamps %globaltimer into its own record (dlm_step_trace); works
                                      under CUDA-graph replay and programmatic dependent launch, costs ~3 atomics per CTA      */
#define DLM_OPT_TCT_MIN_ITEMS 12   /* fewest (request, KV head, query tile) work items for which a step takes the tcgen05 attention
                                      kernels (default 64); below it the mma.sync kernel runs.  1 = always tcgen05 (A/B timing)         */
#define DLM_OPT_LAYER_KERNEL  13   /* default 0 (measured slower than the per-stage kernels).  1: steps of <= 64 tokens whose
                                      requests each compute <= 64 stacked query rows (the
                                      batch-1 cache step) run ALL layers in one persistent launch (layer_mega_kernel: weight
                                      stream never stops, stream-K work split, in-kernel phase counter); 0: one kernel per stage */
#define DLM_OPT_LAYER_KERNEL_PHASE_TS 14 /* 1: that kernel records a timestamp per phase in CTA 0 (tuning aid, dlm_layer_kernel_phases) */
DLM_API int  dlm_set_option(dlm_ctx*, int32_t key, int32_t value);
/* Phase end times of the last whole-stack launch taken with DLM_OPT_LAYER_KERNEL_PHASE_TS, microseconds since its first phase
 * ended, 7 per layer (fold+norm, QKV + RoPE, attention, O, fold+norm, gate/up + SwiGLU, down) + the final fold.  Returns the count. */
DLM_API int  dlm_layer_kernel_phases(dlm_ctx*, float* usec, int32_t cap);

/* Which kernel families the LAST step launched (bit set), so that a caller -- and the parity tests -- can see when a step
 * left the tcgen05 / TMA kernels: DLM_PATH_ATTN_PLAIN or DLM_PATH_GEMM_PLAIN on a bf16 model means the SIMT debugging
 * kernels ran (head_dim != 128 or page_tokens != 64 for attention; DLM_OPT_SIMPLE_KERNELS), which is ~100x slower. */
#define DLM_PATH_GEMM_SKINNY  0x001u   /* weight-streaming split-K tcgen05 GEMM (<= 128 tokens)          */
#define DLM_PATH_GEMM_PAIR    0x002u   /* persistent CTA-pair tcgen05 GEMM                               */
#define DLM_PATH_GEMM_TC      0x004u   /* single-CTA tcgen05 GEMM (LM head <= 128 rows, fallbacks)        */
#define DLM_PATH_GEMM_PLAIN   0x008u   /* SIMT GEMM (fp32 models, DLM_OPT_SIMPLE_KERNELS)                 */
#define DLM_PATH_ATTN_TC      0x010u   /* row-major tcgen05 attention                                    */
#define DLM_PATH_ATTN_TCT     0x020u   /* transposed-score tcgen05 attention                             */
#define DLM_PATH_ATTN_FLASH   0x040u   /* mma.sync attention                                             */
#define DLM_PATH_ATTN_PLAIN   0x080u   /* SIMT attention                                                 */
#define DLM_PATH_ROPE_FUSED   0x100u   /* RoPE + K/V page write in the QKV GEMM's epilogue                */
#define DLM_PATH_GRAPH_REPLAY 0x200u   /* the step was one CUDA-graph launch                             */
#define DLM_PATH_LAYER_KERNEL 0x400u   /* all layers in one persistent launch (DLM_OPT_LAYER_KERNEL)     */
DLM_API uint32_t dlm_last_step_kernels(dlm_ctx*);

/* Timeline of the LAST step taken with DLM_OPT_TRACE = 1, one row per kernel launch in launch order: microseconds since the
 * step's first kernel began -- begin: first CTA entered the kernel; wait: griddepcontrol.wait first returned in it, i.e. the
 * kernel before it in the stream had completed (= begin without programmatic dependent launch); end: last CTA left.
 * The time a launch holds the step's critical path is wait(next launch) - wait(this launch); these sum to the step's
 * duration, which overlapping CUDA-event pairs cannot give.  kernel = DLM_K_* class. */
typedef struct { int32_t kernel, slot; float begin_us, wait_us, end_us; } dlm_trace_row;
DLM_API int  dlm_step_trace(dlm_ctx*, dlm_trace_row* rows, int32_t cap, int32_t* n_rows);

/* Per-kernel-class device time accumulated over the steps run with DLM_OPT_KERNEL_TIMING = 1 (CUDA events on
 * the library's stream around each launch; the measurement behind bench.py's roofline object, P:123 profiling).
 * rows[0..*n_rows) lists the classes that launched; reset != 0 clears the accumulators afterwards. */
#define DLM_K_EMBED          0   /* a1 */
#define DLM_K_RMSNORM        1   /* a2 / a7 / a10 */
#define DLM_K_GEMM_QKV       2   /* a3 */
#define DLM_K_ROPE_KV        3   /* a4 */
#define DLM_K_ATTENTION      4   /* a5 (split-KV merge included) */
#define DLM_K_GEMM_O         5   /* a6 */
#define DLM_K_GEMM_GATEUP    6   /* a8 */
#define DLM_K_GEMM_DOWN      7   /* a9 */
#define DLM_K_LMHEAD         8   /* a11 */
#define DLM_K_COMBINE_UNMASK 9   /* a12 + a13 */
#define DLM_K_LAYERS         10  /* a2 .. a9 of every layer in one persistent launch (cached steps of <= 64 tokens) */
#define DLM_K_COUNT          11
typedef struct { int32_t kernel, launches; float usec; } dlm_kernel_time;
DLM_API int  dlm_kernel_times(dlm_ctx*, dlm_kernel_time* rows, int32_t cap, int32_t* n_rows, int32_t reset);

/* Stage tensors of the LAST step (needs DLM_OPT_DEBUG_DUMP), as float32 on the host, for the rows the step
 * computed for `req` (refresh: S rows, cached: B rows), row-major [rows, width].  Returns the number of
 * floats written or an error.  Stages follow the rounding points of the bf16 path. */
#define DLM_T_X_IN    0   /* residual stream entering the layer        [rows, d]      fp32 */
#define DLM_T_NORM1   1   /* RMSNorm(x) fed to the QKV GEMM            [rows, d]           */
#define DLM_T_Q       2   /* Q after RoPE                              [rows, H*d_h]       */
#define DLM_T_K       3   /* K after RoPE, as written to the store     [rows, H_kv*d_h]    (read back from the pages; needs no dump) */
#define DLM_T_V       4   /* V as written to the store                 [rows, H_kv*d_h]    (read back from the pages; needs no dump) */
#define DLM_T_ATTN    5   /* attention output                          [rows, H*d_h]       */
#define DLM_T_X_MID   6   /* residual after O-proj                     [rows, d]      fp32 */
#define DLM_T_NORM2   7   /* RMSNorm(x_mid) fed to gate/up             [rows, d]           */
#define DLM_T_ACT     8   /* silu(gate)*up                             [rows, F]           */
#define DLM_T_X_OUT   9   /* residual leaving the layer                [rows, d]      fp32 */
#define DLM_T_FINAL_NORM 10 /* layer ignored: RMSNorm of the block rows fed to the LM head [B, d] */
#define DLM_T_KCACHE  11  /* the request's stored K for ALL S positions [S, H_kv*d_h]      */
#define DLM_T_VCACHE  12  /* the request's stored V for ALL S positions [S, H_kv*d_h]      */
DLM_API int64_t dlm_debug_tensor(dlm_ctx*, int32_t req, int32_t layer, int32_t which, float* out, int64_t cap_floats);

/* Counters: kernels launched for this context since dlm_init returned (bench.py's gpu_launches). */
DLM_API int64_t dlm_launch_count(dlm_ctx*);
/* Device time of the last step in microseconds (CUDA events on the library's stream). */
DLM_API float dlm_last_step_usec(dlm_ctx*);

DLM_API const char* dlm_last_error(dlm_ctx*);     /* ctx may be NULL: error of the last failed dlm_init        */

#ifdef __cplusplus
}
#endif
#endif /* DLM_H_ */
