/* dlm_ops.h -- kernel-level entry points of libdlm.so, for kernel parity tests and micro-benchmarks.
 * All pointers are DEVICE pointers unless stated; `stream` is a cudaStream_t (NULL = default stream);
 * calls are asynchronous on that stream.  Return 0 or a negative DLM_E_* code (see dlm.h);
 * dlm_last_error(NULL) gives the text.
 */
#ifndef DLM_OPS_H_
#define DLM_OPS_H_

#include <stdint.h>

#ifndef DLM_API
#define DLM_API __attribute__((visibility("default")))
#endif

#ifdef __cplusplus
extern "C" {
#endif

#define DLM_EPI_F32    0   /* out fp32  [M, N]                      = A . W^T                              */
#define DLM_EPI_BF16   1   /* out bf16  [M, N]                      = bf16(A . W^T)                         */
#define DLM_EPI_RESID  2   /* out fp32  [M, N]                     += A . W^T   (residual stream, a6 / a9)  */
#define DLM_EPI_SWIGLU 3   /* out bf16  [M, N]: W is [2N, K] (gate rows then up rows); silu(A.Wg^T)*(A.Wu^T) (a8) */

/* tcgen05/TMEM GEMM fed by TMA (rows a3/a6/a8/a9 of DESIGN.md): A bf16 [M, K] row-major, W bf16 [N(or 2N), K]
 * row-major ([out, in]), fp32 accumulation.  bn = MMA N of the CTA tile (0 = pick automatically; otherwise a
 * multiple of 32 in [32, 256], multiple of 64 for SwiGLU).  K % 8 == 0 (16-byte rows for TMA). */
DLM_API int dlm_op_gemm_bf16(const void* A, const void* W, void* out, int32_t M, int32_t N, int32_t K, int32_t epilogue,
                     int32_t bn, void* stream);

/* Same contraction and epilogues on the persistent CTA-pair kernel the engine uses for M > 128 tokens (refresh
 * steps, large cached batches): clusters of two CTAs, tcgen05.mma.cta_group::2 on 256 x bn tiles, accumulator
 * double-buffered in tensor memory.  bn = 0 picks the tile width; otherwise a multiple of 32 in [64, 256]
 * (multiple of 64 for SwiGLU).  splits (DLM_EPI_F32 only): 1 = no split-K; n > 1 = n K ranges, each writing an fp32
 * slice, summed in slice order; 0 = the split the engine would choose.  Returns the number of K splits used
 * (>= 1) or a DLM_E_* code; with splits != 1 the call synchronises the stream. */
DLM_API int dlm_op_gemm_pair_bf16(const void* A, const void* W, void* out, int32_t M, int32_t N, int32_t K, int32_t epilogue,
                          int32_t bn, int32_t splits, void* stream);

/* The tile plan dlm_op_gemm_pair_bf16 / the engine take for a shape with bn = 0 (no split-K): *bn = width of the column blocks,
 * and when the launch mixes two widths (gate/up projections of <= 1024 rows: the pairs' last tiles are narrower so that the
 * last wave is full) *bn2 = the narrow width and *n_wide = how many leading column blocks are *bn wide; else *bn2 = 0. */
DLM_API int dlm_op_gemm_pair_plan(int32_t M, int32_t N, int32_t K, int32_t epilogue, int32_t* bn, int32_t* bn2, int32_t* n_wide);

/* Weight-streaming split-K tcgen05 GEMM for T <= 128 tokens (the cached step's a3/a6/a8/a9): swap-AB (weights on
 * the MMA's M side, tokens on N), every K split writes an fp32 slice and the slices are summed in a fixed order.
 * epilogue DLM_EPI_F32: out fp32 [T, N] = X . W^T; DLM_EPI_SWIGLU: out bf16 [T, N], W = [2N, K] (gate rows, up rows).
 * splits = 0 picks the split the engine would use; returns the number of K splits used (>= 1) or a DLM_E_* code. */
DLM_API int dlm_op_gemm_skinny_bf16(const void* X, const void* W, void* out, int32_t T, int32_t N, int32_t K, int32_t epilogue,
                            int32_t splits, void* stream);

/* Same contraction on the plain SIMT kernel (debugging reference of the engine; fp32 out only). */
DLM_API int dlm_op_gemm_plain_bf16(const void* A, const void* W, float* out, int32_t M, int32_t N, int32_t K, void* stream);

/* Fused LM head (a11 + a12): hidden bf16 [R, K] x W_lm bf16 [V, K] -> per row token = argmax_v z (lowest id on
 * ties), conf = softmax(z)[token], lse = log sum exp z, z = scale * logits, z[mask_id] = -inf.
 * Full logits are never written.  scratch: device buffer of dlm_op_lmhead_scratch_bytes(R, V) bytes. */
DLM_API int64_t dlm_op_lmhead_scratch_bytes(int32_t R, int32_t V);
DLM_API int dlm_op_lmhead_bf16(const void* hidden, const void* W_lm, int32_t R, int32_t V, int32_t K, float scale,
                       int32_t mask_id, int32_t* tok, float* conf, float* lse, void* scratch, void* stream);

/* Fused LM head + threshold unmask (a11..a13, config 5 micro-benchmark): n requests x B rows each (R = n*B);
 * tokens_io int32 [n, B] holds each block's current ids (mask_id = still masked) and is updated in place;
 * n_committed int32 [n]; commits (pos in block, tok, conf) packed per request with stride B. */
DLM_API int dlm_op_lmhead_unmask_bf16(const void* hidden, const void* W_lm, int32_t n, int32_t B, int32_t V, int32_t K,
                              float scale, int32_t mask_id, const float* tau, int32_t* tokens_io,
                              int32_t* n_committed, int32_t* pos, int32_t* tok, float* conf, void* scratch,
                              void* stream);

/* dlm_op_lmhead_bf16 for callers that must not allocate device memory and have none to spare for scratch.
 *
 * Who this is for: code that runs where cudaMalloc is off the table -- a serving loop whose whole HBM budget was handed
 * to a pool at start-up (K/V pages, weights) and must not grow, a latency-critical section that cannot afford the
 * device-wide synchronisation cudaMalloc / cudaFree imply, a plug-in that is only ever given input and output buffers by
 * its host program.  dlm_op_lmhead_bf16 asks such a caller for a scratch buffer (the split-vocabulary partials: one
 * (max, sum, argmax) record per row and 128-column vocabulary tile); this entry point keeps that scratch inside the
 * library instead, in one file-scope device array of DLM_LMHEAD_STATIC_SCRATCH_BYTES bytes that every GPU which loads
 * libdlm.so holds from module load until the process exits.  The caller passes inputs and outputs only.
 *
 * Same operation, same kernels, same results as dlm_op_lmhead_bf16 (tok = argmax_v z, lowest id on ties;
 * conf = softmax(z)[tok]; lse = log sum exp z; z = scale * hidden . W_lm^T, z[mask_id] = -inf).
 * hidden bf16 [R, K], W_lm bf16 [V, K], tok int32 [R], conf / lse fp32 [R]: device pointers, caller-owned.
 *
 * Limits: 1 <= R <= DLM_LMHEAD_STATIC_MAX_ROWS and dlm_op_lmhead_static_bytes(R, V) <= DLM_LMHEAD_STATIC_SCRATCH_BYTES
 * (128 rows x 152 064 columns needs 2.4 MB); anything larger returns DLM_E_CAPACITY with the numbers in
 * dlm_last_error(NULL) and launches nothing.  K % 8 == 0 as for the other GEMMs.
 *
 * The call performs no cudaMalloc / cudaFree / cudaMallocAsync and calls no library routine that does; it only
 * enqueues kernels on `stream` and returns without synchronising.  The first call on each device looks up the array's
 * device address (cudaGetSymbolAddress, with that device current) and sets the GEMM kernel's shared-memory attribute;
 * make that first call during start-up, outside any stream capture.  Later calls on that device reuse the address.
 *
 * All calls on a device share the one array and it keeps whatever the previous call left: each call rewrites every word
 * it later reads (partials, row metadata, the zeroed token / threshold rows), so calls that follow one another on one
 * stream are independent, but two calls whose kernels may overlap on the GPU (different streams, no event between them)
 * race on it and give garbage.  Serialise them, or use dlm_op_lmhead_bf16 with a scratch buffer per stream. */
#define DLM_LMHEAD_STATIC_MAX_ROWS      128
#define DLM_LMHEAD_STATIC_SCRATCH_BYTES (4 << 20)
DLM_API int64_t dlm_op_lmhead_static_bytes(int32_t R, int32_t V);   /* bytes of the array a call with these sizes uses */
DLM_API int dlm_op_lmhead_static_bf16(const void* hidden, const void* W_lm, int32_t R, int32_t V, int32_t K, float scale,
                              int32_t mask_id, int32_t* tok, float* conf, float* lse, void* stream);

/* Non-causal block attention over a contiguous (unpaged) K/V, bf16 (a5): q [Tq, H, d_h], k/v [S, H_kv, d_h]
 * -> out [Tq, H, d_h]; softmax_j(q.k_j/sqrt(d_h)) v_j over all j.  flash = 0: plain kernel; 1: mma.sync
 * online-softmax kernel; 2: tcgen05/TMEM kernel with the K/V split the engine would pick (the transposed-score variant when Tq * H / H_kv <= 64); 2 + s: the same
 * with s K/V splits; 102 / 102 + s: the row-major tcgen05 kernel even when the transposed one fits. */
DLM_API int dlm_op_attention_bf16(const void* q, const void* k, const void* v, void* out, int32_t Tq, int32_t S,
                          int32_t H, int32_t H_kv, int32_t d_h, int32_t flash, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DLM_OPS_H_ */
