/* dlm_sched.h -- host-side consumers of the per-step cost table: the paper's control-plane
 * formulas that read dlm_profile_step_costs' rows (the latency profile LP of P:123 / P:154 for one instance, TP 1).
 * Pure host arithmetic, no device work; all pointers are HOST pointers owned by the caller.  Garbled lines of the
 * algorithms are read as DESIGN.md G18 states.  Functions returning double give NaN on bad arguments (no rows of the
 * wanted kind, NULL pointers, non-positive sizes).
 */
#ifndef DLM_SCHED_H_
#define DLM_SCHED_H_

#include <stdint.h>

#include "dlm.h"

#ifdef __cplusplus
extern "C" {
#endif

/* LP lookup in microseconds: rows of `kind` (DLM_KIND_REFRESH / DLM_KIND_CACHED) whose per-request K/V length is
 * nearest to kv_tokens (ties: the shorter), piecewise-linear in the token count, clamped at both ends. */
DLM_API double dlm_lp_lookup(const dlm_cost_row* rows, int32_t n_rows, int32_t kind, double tokens, int32_t kv_tokens);

/* Alg. 4 ReqLoad: (pred_steps_left - recomp_steps_left) * cache_block + recomp_steps_left * num_tokens. */
DLM_API double dlm_req_load(double pred_steps_left, int32_t recomp_steps_left, int32_t num_tokens, int32_t cache_block);

/* Alg. 4 ClusterCapacity for one instance: tokens processed inside the SLO window,
 * tput = (L (B-1) + num_token_per_req) / (LP_cached[L] (B-1) + LP_refresh[num_token_per_req]), L = B * max_seq_per_batch. */
DLM_API double dlm_instance_capacity(const dlm_cost_row* rows, int32_t n_rows, int32_t cache_block, int32_t max_seq_per_batch,
                                     int32_t num_token_per_req, int32_t kv_tokens, double slo_sec);

/* Alg. 5 PredictedTimeLeft in seconds: LP_cached[B * num_reqs] * (pred_steps_left - recomp_steps_left)
 * + recomp_steps_left * LP_refresh[num_tokens]. */
DLM_API double dlm_time_left(const dlm_cost_row* rows, int32_t n_rows, double pred_steps_left, int32_t recomp_steps_left,
                             int32_t cache_block, int32_t num_reqs, int32_t num_tokens, int32_t kv_tokens);

/* Alg. 1 UpdateConfThreshold with Alg. 5 as PredictedTimeLeft: thresholds allowed_desc[0..n) in
 * descending order, pred_steps_left[i] the Step Predictor's estimate under allowed_desc[i].  Returns the index of the
 * first threshold whose predicted time left is <= slo_left_sec, n - 1 if none fits, DLM_E_ARG on bad arguments. */
DLM_API int32_t dlm_pick_threshold(const float* allowed_desc, const double* pred_steps_left, int32_t n, double slo_left_sec,
                                   const dlm_cost_row* rows, int32_t n_rows, int32_t recomp_steps_left, int32_t cache_block,
                                   int32_t num_reqs, int32_t num_tokens, int32_t kv_tokens);

#ifdef __cplusplus
}
#endif
#endif /* DLM_SCHED_H_ */
