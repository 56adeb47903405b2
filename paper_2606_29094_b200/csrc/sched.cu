// Host-side consumers of the cost table (include/dlm_sched.h).  Plain host code in libdlm.so.
#include <math.h>

#include <algorithm>
#include <vector>

#include "../../include/dlm_sched.h"

static double nan_() { return nan(""); }

extern "C" double dlm_lp_lookup(const dlm_cost_row* rows, int32_t n_rows, int32_t kind, double tokens, int32_t kv_tokens) {
  if (!rows || n_rows <= 0) return nan_();
  long long best_kv = -1;
  for (int i = 0; i < n_rows; ++i) {
    if (rows[i].kind != kind) continue;
    const long long k = rows[i].kv_tokens, d = llabs(k - kv_tokens), bd = llabs(best_kv - kv_tokens);
    if (best_kv < 0 || d < bd || (d == bd && k < best_kv)) best_kv = k;
  }
  if (best_kv < 0) return nan_();
  std::vector<std::pair<double, double>> pts;
  for (int i = 0; i < n_rows; ++i)
    if (rows[i].kind == kind && rows[i].kv_tokens == best_kv) pts.push_back({(double)rows[i].n_tokens, (double)rows[i].usec});
  std::sort(pts.begin(), pts.end());
  if (tokens <= pts.front().first) return pts.front().second;
  if (tokens >= pts.back().first) return pts.back().second;
  for (size_t i = 0; i + 1 < pts.size(); ++i)
    if (tokens >= pts[i].first && tokens <= pts[i + 1].first)
      return pts[i].second + (pts[i + 1].second - pts[i].second) * (tokens - pts[i].first) / (pts[i + 1].first - pts[i].first);
  return nan_();
}

extern "C" double dlm_req_load(double pred_steps_left, int32_t recomp_steps_left, int32_t num_tokens, int32_t cache_block) {
  return (pred_steps_left - recomp_steps_left) * cache_block + (double)recomp_steps_left * num_tokens;
}

extern "C" double dlm_instance_capacity(const dlm_cost_row* rows, int32_t n_rows, int32_t cache_block, int32_t max_seq_per_batch,
                                        int32_t num_token_per_req, int32_t kv_tokens, double slo_sec) {
  if (cache_block <= 0 || max_seq_per_batch <= 0 || num_token_per_req <= 0) return nan_();
  const double load = (double)cache_block * max_seq_per_batch;
  const double cache_lat = dlm_lp_lookup(rows, n_rows, DLM_KIND_CACHED, load, kv_tokens) * 1e-6;
  const double recomp_lat = dlm_lp_lookup(rows, n_rows, DLM_KIND_REFRESH, num_token_per_req, kv_tokens) * 1e-6;
  const double tput = (load * (cache_block - 1) + num_token_per_req) / (cache_lat * (cache_block - 1) + recomp_lat);
  return tput * slo_sec;
}

extern "C" double dlm_time_left(const dlm_cost_row* rows, int32_t n_rows, double pred_steps_left, int32_t recomp_steps_left,
                                int32_t cache_block, int32_t num_reqs, int32_t num_tokens, int32_t kv_tokens) {
  if (cache_block <= 0 || num_reqs <= 0 || num_tokens <= 0) return nan_();
  const double cache_lat = dlm_lp_lookup(rows, n_rows, DLM_KIND_CACHED, (double)cache_block * num_reqs, kv_tokens) * 1e-6;
  const double recomp_lat = dlm_lp_lookup(rows, n_rows, DLM_KIND_REFRESH, num_tokens, kv_tokens) * 1e-6;
  return cache_lat * (pred_steps_left - recomp_steps_left) + recomp_steps_left * recomp_lat;
}

extern "C" int32_t dlm_pick_threshold(const float* allowed_desc, const double* pred_steps_left, int32_t n, double slo_left_sec,
                                      const dlm_cost_row* rows, int32_t n_rows, int32_t recomp_steps_left, int32_t cache_block,
                                      int32_t num_reqs, int32_t num_tokens, int32_t kv_tokens) {
  if (!allowed_desc || !pred_steps_left || n <= 0 || !rows || n_rows <= 0) return DLM_E_ARG;
  for (int i = 0; i < n; ++i) {
    const double t = dlm_time_left(rows, n_rows, pred_steps_left[i], recomp_steps_left, cache_block, num_reqs, num_tokens, kv_tokens);
    if (t != t) return DLM_E_ARG;
    if (t <= slo_left_sec) return i;
  }
  return n - 1;
}
