// Host side of libdlm.so: context, request table, paged K/V bookkeeping, the ragged step planner and the
// extern "C" boundary declared in include/dlm.h and include/dlm_ops.h.  Every step of the path runs in the
// CUDA kernels of this directory; there is no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <string>
#include <tuple>
#include <vector>

#include "../../include/dlm.h"
#include "../../include/dlm_ops.h"
#include "attn_flash.cuh"
#include "attn_tc.cuh"
#include "attn_tct.cuh"
#include "common.cuh"
#include "gemm_skinny.cuh"
#include "gemm_pair.cuh"
#include "gemm_tc.cuh"
#include "kernels_basic.cuh"
#include "layer_mega.cuh"

namespace dlm {
thread_local long long g_launches = 0;
thread_local int g_num_sms = 148;
thread_local int g_dev = 0;
static thread_local std::string g_init_error;

static void set_err(std::string* dst, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  *dst = buf;
}

// One launch path for every kernel of a step: a plain launch, or a programmatic dependent launch (PDL) whose
// prologue (and, for the GEMMs, weight prefetch) overlaps the tail of the previous kernel in the stream.
// launch_k_attr: the same with an optional cooperative launch (all CTAs co-resident, or the launch fails instead of hanging).
template <typename... KArgs, typename... Args>
static cudaError_t launch_k_attr(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, bool coop, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[2];
  int na = 0;
  if (pdl) {
    at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  if (coop) {
    at[na].id = cudaLaunchAttributeCooperative;
    at[na].val.cooperative = 1;
    ++na;
  }
  if (na) { cfg.attrs = at; cfg.numAttrs = na; }
  g_launches++;
  if constexpr (sizeof...(Args) + 1 == sizeof...(KArgs))       // caller left out the trailing TraceSlot: tracing off for this launch
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)..., TraceSlot{nullptr});
  else
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

template <typename... KArgs, typename... Args>
static cudaError_t launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  if (pdl) {
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
  }
  g_launches++;
  if constexpr (sizeof...(Args) + 1 == sizeof...(KArgs))       // caller left out the trailing TraceSlot: tracing off for this launch
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)..., TraceSlot{nullptr});
  else
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

#define CU_TRY(ctx_err, expr)                                                                         \
  do {                                                                                                \
    cudaError_t e__ = (expr);                                                                         \
    if (e__ != cudaSuccess) {                                                                         \
      set_err(ctx_err, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__);   \
      return DLM_E_CUDA;                                                                              \
    }                                                                                                 \
  } while (0)

// ------------------------------------------------------------------------------------------------
// TMA tensor maps (driver entry point fetched through the runtime, so libcuda is not a link dependency)
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess) fn = (EncodeTiledFn)p;
  }
  return fn;
}
// bf16 row-major [rows, cols] matrix, box = box_rows x 64 columns, 128-byte swizzle, OOB reads give zeros.
static bool make_tmap_bf16(CUtensorMap* m, const void* ptr, long long rows, long long cols, int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)cols * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// Tiled weight storage (ptx_sm100.cuh tma_load_w_tiled): [K/64][rows/128][128 rows][64 columns] bf16, rows and K padded with
// zeros to multiples of 128 / 64.  A GEMM CTA streams one 128-row tile after the other along K, i.e. one contiguous region of
// HBM instead of 128 row segments of 128 bytes per box (measured: +5.7 % on the whole C2 cached step).
static bool make_tmap_w_tiled(CUtensorMap* m, const void* ptr, long long rows_pad, long long k_pad, int box_rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn || rows_pad % 128 || k_pad % 64 || (box_rows != 32 && box_rows != 64 && box_rows != 128)) return false;
  const cuuint64_t kb = (cuuint64_t)k_pad / 64;
  const cuuint64_t rb = (cuuint64_t)rows_pad / 128;
  cuuint64_t dims[4] = {64, 128, rb, kb};
  cuuint64_t strides[3] = {128, 16384, rb * 16384};
  cuuint32_t box[4] = {64, (cuuint32_t)box_rows, 1, 1};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(ptr), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}
static inline long long pad_to(long long v, long long m) { return (v + m - 1) / m * m; }

// fp32 output [splits][rows][ldc] of which `cols` columns are valid: box 32 columns x 32 rows x 1 slice, 128-byte swizzle
// (the layout of the epilogue's coalescing stage).  TMA clips rows >= rows and columns >= cols, so ragged tiles need no code.
static bool make_tmap_f32_out(CUtensorMap* m, const void* ptr, long long rows, long long cols, long long ldc, long long splits, long long split_stride) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {(cuuint64_t)cols, (cuuint64_t)rows, (cuuint64_t)splits};
  cuuint64_t strides[2] = {(cuuint64_t)ldc * 4, (cuuint64_t)split_stride * 4};
  cuuint32_t box[3] = {32, 32, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

struct TmapCache {
  std::map<std::tuple<const void*, long long, long long, long long, long long>, CUtensorMap> mo;
  const CUtensorMap* get_f32_out(const void* ptr, long long rows, long long cols, long long ldc, long long splits) {
    auto key = std::make_tuple(ptr, rows, cols, ldc, splits);
    auto it = mo.find(key);
    if (it != mo.end()) return &it->second;
    CUtensorMap t;
    if (!make_tmap_f32_out(&t, ptr, rows, cols, ldc, splits, rows * ldc)) return nullptr;
    return &mo.emplace(key, t).first->second;
  }
  std::map<std::tuple<const void*, long long, long long, int>, CUtensorMap> m;
  const CUtensorMap* get(const void* ptr, long long rows, long long cols, int box_rows) {
    auto key = std::make_tuple(ptr, rows, cols, box_rows);
    auto it = m.find(key);
    if (it != m.end()) return &it->second;
    CUtensorMap t;
    if (!make_tmap_bf16(&t, ptr, rows, cols, box_rows)) return nullptr;
    return &m.emplace(key, t).first->second;
  }
  // Weights of which the engine keeps a second, tiled copy (make_tmap_w_tiled), registered at init: row-major pointer ->
  // twin.  The weight-streaming launchers (T <= 128 tokens) ask twin(W) and read the tiled copy; the dlm_op_* entry points
  // never register anything, their caller-owned weights are row-major only.
  struct Twin { const void* ptr; long long rows_pad, k_pad; };
  std::map<const void*, Twin> tiled;
  const Twin* twin(const void* rowmajor) const { auto it = tiled.find(rowmajor); return it == tiled.end() ? nullptr : &it->second; }
  const CUtensorMap* get_w(const Twin& tw, int box_rows) {
    auto key = std::make_tuple(tw.ptr, tw.rows_pad, tw.k_pad, -box_rows);
    auto it = m.find(key);
    if (it != m.end()) return &it->second;
    CUtensorMap t;
    if (!make_tmap_w_tiled(&t, tw.ptr, tw.rows_pad, tw.k_pad, box_rows)) return nullptr;
    return &m.emplace(key, t).first->second;
  }
};

// ------------------------------------------------------------------------------------------------
// tcgen05 GEMM launcher
// ------------------------------------------------------------------------------------------------
static int pick_bn(int M, int N, int epi) {
  // N = output features (SwiGLU: F, each tile covers bn/2).  Aim for one resident wave of equal tiles:
  // the largest tile that still yields >= ~0.8 * SMs CTAs; when even the smallest cannot, take the smallest.
  const int m_tiles = (M + 127) / 128;
  if (epi == EPI_LMHEAD) return 128;
  static const int cand_std[] = {256, 192, 128, 96, 64, 32};
  static const int cand_glu[] = {256, 192, 128, 64};
  const int* cand = epi == EPI_SWIGLU ? cand_glu : cand_std;
  const int nc = epi == EPI_SWIGLU ? 4 : 6;
  for (int i = 0; i < nc; ++i) {
    int per = epi == EPI_SWIGLU ? cand[i] / 2 : cand[i];
    long long tiles = (long long)m_tiles * ((N + per - 1) / per);
    if (tiles >= (long long)(g_num_sms * 4) / 5) return cand[i];
  }
  return cand[nc - 1];
}

template <int EPI>
static cudaError_t launch_gemm_tc_t(const CUtensorMap* ma, const CUtensorMap* mb, const GemmTcParams& p, int n_tiles_x,
                                    cudaStream_t st, bool pdl) {
  static bool configured[kMaxDevices] = {};     // one-time per device (a process may hold contexts on several GPUs)
  const int smem = gemm_tc_smem_bytes(p.bn, p.stages);
  if (!configured[g_dev]) {
    cudaError_t e = cudaFuncSetAttribute(gemm_tc_kernel<EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    configured[g_dev] = true;
  }
  dim3 grid(n_tiles_x, (p.M + 127) / 128);
  return launch_k(gemm_tc_kernel<EPI>, grid, dim3(kGemmThreads), (size_t)smem, st, pdl, *ma, *mb, p);
}

// A: bf16 [a_rows_cap, K] buffer (M valid rows); W: bf16 [w_rows, K].
static int gemm_tc(TmapCache& tc, std::string* err, const void* A, long long a_rows_cap, const void* W, long long w_rows,
                   int M, int N, int K, int epi, int bn, GemmTcParams p, cudaStream_t st, bool pdl = false) {
  if (M <= 0) return DLM_OK;
  if (K % 8) { set_err(err, "gemm_tc: K=%d must be a multiple of 8", K); return DLM_E_ARG; }
  if (epi != EPI_LMHEAD && p.ldc % 8) { set_err(err, "gemm_tc: output row pitch %lld must be a multiple of 8 elements", p.ldc); return DLM_E_ARG; }
  if (bn <= 0) bn = pick_bn(M, N, epi);
  if (bn % 32 || bn < 32 || bn > 256 || (epi == EPI_SWIGLU && bn % 64)) { set_err(err, "gemm_tc: bad bn=%d", bn); return DLM_E_ARG; }
  p.M = M; p.N = N; p.K = K; p.bn = bn;
  p.a_box_rows = M <= 32 ? 32 : (M <= 64 ? 64 : 128);
  const int num_kb = (K + kBK - 1) / kBK;
  p.stages = std::max(2, std::min(std::min(num_kb, 12), (200 * 1024) / gemm_tc_stage_bytes(bn)));
  p.w_policy = DLM_L2_EVICT_FIRST;
  const int per = epi == EPI_SWIGLU ? bn / 2 : bn;
  const int n_tiles_x = (N + per - 1) / per;
  if (epi == EPI_LMHEAD && n_tiles_x != p.n_tiles) { set_err(err, "gemm_tc: lm-head tile count mismatch"); return DLM_E_ARG; }
  const CUtensorMap* ma = tc.get(A, a_rows_cap, K, p.a_box_rows);
  const CUtensorMap* mb = tc.get(W, w_rows, K, per);
  if (!ma || !mb) { set_err(err, "cuTensorMapEncodeTiled failed (A=%p rows=%lld K=%d, W=%p rows=%lld box=%d)", A, a_rows_cap, K, W, w_rows, per); return DLM_E_CUDA; }
  cudaError_t e;
  switch (epi) {
    case EPI_F32: e = launch_gemm_tc_t<EPI_F32>(ma, mb, p, n_tiles_x, st, pdl); break;
    case EPI_BF16: e = launch_gemm_tc_t<EPI_BF16>(ma, mb, p, n_tiles_x, st, pdl); break;
    case EPI_RESID: e = launch_gemm_tc_t<EPI_RESID>(ma, mb, p, n_tiles_x, st, pdl); break;
    case EPI_SWIGLU: e = launch_gemm_tc_t<EPI_SWIGLU>(ma, mb, p, n_tiles_x, st, pdl); break;
    case EPI_LMHEAD: e = launch_gemm_tc_t<EPI_LMHEAD>(ma, mb, p, n_tiles_x, st, pdl); break;
    default: set_err(err, "gemm_tc: bad epilogue %d", epi); return DLM_E_ARG;
  }
  if (e != cudaSuccess) { set_err(err, "gemm_tc launch failed: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
  return DLM_OK;
}

// ------------------------------------------------------------------------------------------------
// CTA-pair persistent tcgen05 GEMM launcher (M > 128)
// ------------------------------------------------------------------------------------------------
// Tile width and K split.  Measured on B200: with both operands in shared memory one 256 x bn x 16 UMMA takes
// ~128 cycles for every bn <= 256 (the A-operand read paces it), so a work unit costs its K blocks whatever its
// width.  Cost of a launch ~ waves x (K blocks per unit + fixed per-unit cost); ties go to fewer splits, then to the
// wider tile (fewer operand bytes per flop).  Split-K (fp32 slices, summed by the consumer in a fixed order) is what
// fills the 74 CTA pairs when M x N alone gives fewer than ~74 tiles (O / down projections at 512 tokens).
static void plan_pair(int M, int N, int K, int epi, int max_splits, int* bn_out, int* splits_out) {
  const int m_tiles = (M + 255) / 256;
  const int pairs = std::max(1, g_num_sms / 2);
  const int num_kb = (K + kBK - 1) / kBK;
  static const int cand_std[] = {256, 224, 192, 160, 128, 96, 64};
  static const int cand_glu[] = {256, 192, 128, 64};
  static const int cand_lm[] = {256};
  static const int cand_rope[] = {256, 128};          // whole 128-wide heads per tile
  const int* cand = epi == EPI_SWIGLU ? cand_glu : (epi == EPI_LMHEAD ? cand_lm : (epi == EPI_ROPE ? cand_rope : cand_std));
  const int nc = epi == EPI_SWIGLU ? 4 : (epi == EPI_LMHEAD ? 1 : (epi == EPI_ROPE ? 2 : 7));
  // Cost of a unit in 1/256 K-block units of a 256-wide tile.  Measured with two K blocks per ring stage (4096 x 12288 x 4096,
  // whole kernel): bn 256 / 192 / 128 -> 1.00 / 0.78 / 0.61 of the 256-wide tile per tile, i.e. ~0.22 + 0.78 bn / 256 (the MMA
  // time is bn / 2 cycles, the stage hand-off is not free); the fixed part (ramp, exposed epilogue) shrinks with the tile too.
  auto kb_cost = [](int bn) { return 56 + (200 * bn) / 256; };
  long long best = -1;
  *bn_out = cand[0]; *splits_out = 1;
  for (int sp = 1; sp <= std::max(1, max_splits); ++sp) {
    const int kb_per = (num_kb + sp - 1) / sp;
    if (sp > 1 && ((sp - 1) * kb_per >= num_kb || kb_per < 8)) continue;
    for (int i = 0; i < nc; ++i) {
      const int per = epi == EPI_SWIGLU ? cand[i] / 2 : cand[i];
      const long long units = (long long)m_tiles * ((N + per - 1) / per) * sp;
      const long long waves = (units + pairs - 1) / pairs;
      const long long cost = waves * ((long long)kb_per * kb_cost(cand[i]) + 8LL * (128 + cand[i] / 2));
      if (best < 0 || cost < best) { best = cost; *bn_out = cand[i]; *splits_out = sp; }
    }
  }
}

// Mixed tile widths for launches with few row tiles (<= 16: one panel, column blocks dealt round-robin in order): the first
// n_a column blocks are bn1 wide, the rest bn2 < bn1, so that the pairs' last tiles are narrower, cheaper ones instead of a
// partly filled wave of wide tiles (512 tokens: 192 gate/up tiles of 256 on 74 pairs = 3 waves for 2.6 waves of work; measured
// gate/up at 512 tokens 2590 -> 2468 us per C2 refresh step, 3006 -> 2611 us per C4 cached step).  Exact
// makespan of the round-robin dealing under plan_pair's cost model; taken only when it beats the best uniform width by > 3 %.
static bool plan_pair_mixed(int M, int N, int K, int epi, int bn_uniform, int* bn1_out, int* bn2_out, int* n_a_out, int* n_b_out) {
  const int m_tiles = (M + 255) / 256, pairs = std::max(1, g_num_sms / 2), num_kb = (K + kBK - 1) / kBK;
  // gate/up only: for the fused-RoPE QKV epilogue the 256-wide first tiles measured slower than three waves of 128-wide ones
  // (C2 refresh: QKV 1485 -> 1534 us per step), its long epilogue is cheaper in small pieces
  // and only up to 1024 rows: with more row tiles the tail wave is a small share (< 3 % by this model at 9 row tiles), and the
  // search below is host time on the launch path of steps that are not replayed from a graph (memoised per shape)
  if (m_tiles > 4 || epi != EPI_SWIGLU) return false;
  struct Plan { bool ok; int b1, b2, na, nb; };
  static thread_local std::map<std::tuple<int, int, int, int, int>, Plan> memo;
  const auto key = std::make_tuple(M, N, K, bn_uniform, g_num_sms);
  auto hit = memo.find(key);
  if (hit != memo.end()) {
    if (hit->second.ok) { *bn1_out = hit->second.b1; *bn2_out = hit->second.b2; *n_a_out = hit->second.na; *n_b_out = hit->second.nb; }
    return hit->second.ok;
  }
  auto per = [&](int bn) { return epi == EPI_SWIGLU ? bn / 2 : bn; };
  auto cost = [&](int bn) { return (long long)num_kb * (56 + (200 * bn) / 256) + 8LL * (128 + bn / 2); };
  auto makespan = [&](int n_a, int bn1, int n_b, int bn2) {
    std::vector<long long> load(pairs, 0);
    const int tiles = m_tiles * (n_a + n_b);
    for (int t = 0; t < tiles; ++t) load[t % pairs] += cost(t / m_tiles < n_a ? bn1 : bn2);
    return *std::max_element(load.begin(), load.end());
  };
  const long long uni = makespan((N + per(bn_uniform) - 1) / per(bn_uniform), bn_uniform, 0, bn_uniform);
  static const int w_glu[][2] = {{256, 192}, {256, 128}, {192, 128}, {256, 64}, {192, 64}, {128, 64}};
  const int (*w)[2] = w_glu;
  const int nw = 6;
  long long best = uni;
  for (int i = 0; i < nw; ++i) {
    const int p1 = per(w[i][0]), p2 = per(w[i][1]);
    for (int n_a = 1; n_a * p1 < N; ++n_a) {
      const int n_b = (N - n_a * p1 + p2 - 1) / p2;
      const long long c = makespan(n_a, w[i][0], n_b, w[i][1]);
      if (c < best) { best = c; *bn1_out = w[i][0]; *bn2_out = w[i][1]; *n_a_out = n_a; *n_b_out = n_b; }
    }
  }
  const bool ok = best * 100 < uni * 97;
  memo[key] = Plan{ok, *bn1_out, *bn2_out, *n_a_out, *n_b_out};
  return ok;
}

template <int EPI>
static cudaError_t launch_gemm_pair_t(const CUtensorMap* ma, const CUtensorMap* mb, const CUtensorMap* mc, const GemmPairParams& p, cudaStream_t st, bool pdl) {
  static bool configured[kMaxDevices] = {};
  if (!configured[g_dev]) {
    cudaError_t e = cudaFuncSetAttribute(gemm_pair_kernel<EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    configured[g_dev] = true;
  }
  const int pairs = std::max(1, std::min(g_num_sms / 2, p.m_tiles * p.n_tiles_n * p.splits));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2 * pairs); cfg.blockDim = dim3(kPairThreads);
  cfg.dynamicSmemBytes = (size_t)gemm_pair_smem_bytes(p.bn, p.stages); cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 2 : 1;
  g_launches++;
  return cudaLaunchKernelEx(&cfg, gemm_pair_kernel<EPI>, *ma, *mb, *mc, p);
}

// A: bf16 [a_rows_cap, K] buffer (M valid rows); W: bf16 [w_rows, K].  max_splits > 1 (EPI_F32 only) allows split-K:
// p.out_f32 then receives *splits_out slices [split][M][ldc] which the consumer sums.
static int gemm_pair(TmapCache& tc, std::string* err, const void* A, long long a_rows_cap, const void* W, long long w_rows,
                     int M, int N, int K, int epi, int bn, GemmPairParams p, cudaStream_t st, bool pdl = false,
                     int max_splits = 1, int* splits_out = nullptr) {
  if (splits_out) *splits_out = M > 0 ? 1 : 0;
  if (M <= 0) return DLM_OK;
  if (K % 8) { set_err(err, "gemm_pair: K=%d must be a multiple of 8", K); return DLM_E_ARG; }
  if (epi != EPI_LMHEAD && epi != EPI_ROPE && p.ldc % 8) { set_err(err, "gemm_pair: output row pitch %lld must be a multiple of 8 elements", p.ldc); return DLM_E_ARG; }
  if (epi != EPI_F32) max_splits = 1;
  int splits = 1;
  if (epi == EPI_ROPE && bn != 128 && bn != 256) bn = 0;         // whole 128-wide heads per tile: 256 or 128, planned
  const bool auto_bn = bn <= 0;
  if (bn <= 0) plan_pair(M, N, K, epi, max_splits, &bn, &splits);
  else if (max_splits < 0) splits = -max_splits;                 // test hook: forced split count
  if (bn % 32 || bn < 64 || bn > 256 || (epi == EPI_SWIGLU && bn % 64)) { set_err(err, "gemm_pair: bad bn=%d", bn); return DLM_E_ARG; }
  p.M = M; p.N = N; p.K = K; p.bn = bn;
  const int num_kb = (K + kBK - 1) / kBK;
  splits = std::max(1, std::min(splits, num_kb));
  p.kb_per_split = (num_kb + splits - 1) / splits;
  p.splits = (num_kb + p.kb_per_split - 1) / p.kb_per_split;
  p.split_stride = (long long)M * p.ldc;
  if (splits_out) *splits_out = p.splits;
  p.stages = std::max(2, std::min(std::min((num_kb + kPairKbPerStage - 1) / kPairKbPerStage, 12), (224 * 1024 - kPairEpiStageBytes) / gemm_pair_stage_bytes(bn)));
  const int per = epi == EPI_SWIGLU ? bn / 2 : bn;
  p.m_tiles = (M + 255) / 256;
  p.n_tiles_n = (N + per - 1) / per;
  p.panel = std::min(p.m_tiles, 16);
  p.bn2 = 0; p.n_tiles_a = p.n_tiles_n;
  if (auto_bn && p.splits == 1 && getenv("DLM_NO_MIXED_TILES") == nullptr) {
    int b1 = bn, b2 = 0, na = 0, nb = 0;
    if (plan_pair_mixed(M, N, K, epi, bn, &b1, &b2, &na, &nb)) {
      bn = b1; p.bn = b1; p.bn2 = b2; p.n_tiles_a = na; p.n_tiles_n = na + nb;
      p.stages = std::max(2, std::min(std::min((num_kb + kPairKbPerStage - 1) / kPairKbPerStage, 12), (224 * 1024 - kPairEpiStageBytes) / gemm_pair_stage_bytes(bn)));
    }
  }
  p.w_policy = DLM_L2_EVICT_NORMAL;
  p.a_policy = DLM_L2_EVICT_NORMAL;
  if (epi == EPI_LMHEAD && p.n_tiles_n != p.n_tiles) { set_err(err, "gemm_pair: lm-head tile count mismatch"); return DLM_E_ARG; }
  const CUtensorMap* ma = tc.get(A, a_rows_cap, K, 128);
  const CUtensorMap* mb = tc.get(W, w_rows, K, bn / 2);
  // fp32 outputs leave through TMA (store / reduce-add) from the epilogue's shared-memory stage
  const CUtensorMap* mc = ma;
  if (epi == EPI_F32 || epi == EPI_RESID) {
    mc = tc.get_f32_out(p.out_f32, M, N, p.ldc, p.splits);
    if (!mc) { set_err(err, "cuTensorMapEncodeTiled failed (gemm_pair output %p)", (void*)p.out_f32); return DLM_E_CUDA; }
  }
  if (!ma || !mb) { set_err(err, "cuTensorMapEncodeTiled failed (gemm_pair A=%p rows=%lld K=%d, W=%p rows=%lld box=%d)", A, a_rows_cap, K, W, w_rows, bn / 2); return DLM_E_CUDA; }
  cudaError_t e;
  switch (epi) {
    case EPI_F32: e = launch_gemm_pair_t<EPI_F32>(ma, mb, mc, p, st, pdl); break;
    case EPI_BF16: e = launch_gemm_pair_t<EPI_BF16>(ma, mb, mc, p, st, pdl); break;
    case EPI_RESID: e = launch_gemm_pair_t<EPI_RESID>(ma, mb, mc, p, st, pdl); break;
    case EPI_SWIGLU: e = launch_gemm_pair_t<EPI_SWIGLU>(ma, mb, mc, p, st, pdl); break;
    case EPI_LMHEAD: e = launch_gemm_pair_t<EPI_LMHEAD>(ma, mb, mc, p, st, pdl); break;
    case EPI_ROPE: e = launch_gemm_pair_t<EPI_ROPE>(ma, mb, mc, p, st, pdl); break;
    default: set_err(err, "gemm_pair: bad epilogue %d", epi); return DLM_E_ARG;
  }
  if (e != cudaSuccess) { set_err(err, "gemm_pair launch failed: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
  return DLM_OK;
}

// ------------------------------------------------------------------------------------------------
// tcgen05 attention launcher.  *done = false when the shape is not supported or too small to fill the GPU with
// 128-row tiles (the caller then takes the mma.sync kernel).
// ------------------------------------------------------------------------------------------------
static int attn_tc_launch(TmapCache& tc, bf16* out, const bf16* q, const bf16* kv_store, int n_layers_total, const int* page_table,
                          const BatchDesc& bd, const KvGeom& g, int layer, int n_heads, float scale, float** ws, size_t* ws_bytes,
                          cudaStream_t st, bool pdl, std::string* err, bool* done, int force = 0, const TraceSlot* tr = nullptr,
                          unsigned* paths = nullptr, int min_items = 64) {
  *done = false;
  static const TraceSlot no_trace[3] = {{nullptr}, {nullptr}, {nullptr}};
  if (!tr) tr = no_trace;                      // tr[0..2]: records of up to three launches (DLM_OPT_TRACE)
  unsigned path_dummy = 0;
  if (!paths) paths = &path_dummy;
  if (g.head_dim != 128 || g.page_tokens != 64 || bd.T <= 0) return 0;
  const int r = n_heads / g.n_kv_heads;
  const int q_tiles = (bd.max_q_len * r + kTaTile - 1) / kTaTile;
  const bool ragged = bd.qt_off != nullptr && bd.max_q_len * r > kTtNQ;      // row-major kernel over the requests' own query tiles
  const long long items = ragged ? (long long)bd.qt_total * g.n_kv_heads : (long long)bd.n * g.n_kv_heads * q_tiles;
  const int kv_tiles = (bd.max_kv_len + kTaTile - 1) / kTaTile;
  const bool no_transposed = force >= 100;      // test hook: 100 + f = attn_tc_kernel even when the transposed kernel fits
  if (no_transposed) force -= 100;
  if (!force && items < min_items) return 0;       // too few (request, head, query tile) items to fill the SMs with one CTA each
  const long long rows = (long long)n_layers_total * g.n_pages * 2 * g.n_kv_heads * g.page_tokens;
  if (rows >= (1LL << 31)) return 0;
  int splits = 1;
  {
    long long best = -1;
    for (int s = 1; s <= std::min(8, kv_tiles); ++s) {
      const long long waves = (items * s + g_num_sms - 1) / g_num_sms;
      const long long cost = waves * ((kv_tiles + s - 1) / s + 3);      // + per-item ramp, epilogue and combine share (measured: ~3 tiles)
      if (best < 0 || cost < best) { best = cost; splits = s; }
    }
    if (force > 1) splits = std::min(force - 1, kv_tiles);
  }
  // stacked rows <= 64 (cached steps of MHA models): the transposed-score kernel shares the exponentials over all four
  // sub-partitions; force: 0 engine choice, 1 = forced with the split the engine would pick, 1 + s = forced with s splits
  const bool fits_t = bd.max_q_len * r <= kTtNQ;
  const bool transposed = fits_t && !no_transposed;
  // mixed step: the cached requests (<= 64 stacked rows) go to the transposed-score kernel, the refreshing ones to the
  // row-major kernel; each launch skips the other's requests (row_filter), no K/V split
  const bool two_kernels = !force && !fits_t && bd.min_q_len > 0 && bd.min_q_len * r <= kTtNQ;
  if (two_kernels) splits = 1;
  const CUtensorMap* mkv = tc.get(kv_store, rows, 128, 64);
  if (!mkv) { set_err(err, "cuTensorMapEncodeTiled failed (attention K/V store %p, %lld rows)", (const void*)kv_store, rows); return DLM_E_CUDA; }
  static bool configured[kMaxDevices] = {};
  if (!configured[g_dev]) {
    cudaError_t e = cudaFuncSetAttribute(attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTaSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(attn_tct_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTtSmem);
    if (e != cudaSuccess) { set_err(err, "attn_tc: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
    configured[g_dev] = true;
  }
  TaParams p;
  p.out = out; p.q = q; p.page_table = page_table; p.b = bd; p.g = g; p.layer = layer; p.n_heads = n_heads;
  p.splits = splits; p.q_tiles_max = q_tiles; p.n_items = (int)(items * splits);
  p.scale_log2 = scale * 1.4426950408889634f; p.ws_o = nullptr; p.ws_ml = nullptr;
  p.kv_policy = q_tiles == 1 ? DLM_L2_EVICT_FIRST : DLM_L2_EVICT_NORMAL;
  p.row_filter = 0; p.req_lo = 0; p.req_n = bd.n; p.ragged_q = 0; p.tr = TraceSlot{nullptr};
  const long long TH = (long long)bd.T * n_heads;
  while (splits > 1 && (size_t)splits * TH * (128 + 2) * 4 > *ws_bytes) --splits;     // fixed workspace (see attn_flash_launch)
  p.splits = splits; p.n_items = (int)(items * splits);
  if (splits > 1) {
    p.ws_o = *ws;
    p.ws_ml = *ws + (size_t)splits * TH * 128;
  }
  if (two_kernels) {
    TaParams pt = p;
    // `order` lists the n_big requests of the row-major kernel first: each launch walks its own requests only
    pt.row_filter = 1; pt.q_tiles_max = 1; pt.req_lo = bd.n_big; pt.n_items = (bd.n - bd.n_big) * g.n_kv_heads; pt.kv_policy = DLM_L2_EVICT_FIRST;
    pt.req_n = bd.n - bd.n_big;
    p.row_filter = 2; p.req_n = bd.n_big; p.ragged_q = 1; p.n_items = bd.qt_big * g.n_kv_heads;
    if (pt.n_items <= 0 || p.n_items <= 0) { set_err(err, "attn_tc: inconsistent mixed batch (%d of %d requests above 64 rows)", bd.n_big, bd.n); return DLM_E_ARG; }
    pt.tr = tr[0]; p.tr = tr[1];
    cudaError_t e2 = launch_k(attn_tct_kernel, dim3((unsigned)std::min(g_num_sms, pt.n_items)), dim3(kTaThreads), (size_t)kTtSmem, st, pdl, *mkv, pt);
    if (e2 == cudaSuccess)
      e2 = launch_k(attn_tc_kernel, dim3((unsigned)std::min<long long>(g_num_sms, p.n_items)), dim3(kTaThreads), (size_t)kTaSmem, st, pdl, *mkv, p);
    if (e2 != cudaSuccess) { set_err(err, "attn_tc launch: %s", cudaGetErrorString(e2)); return DLM_E_CUDA; }
    *paths |= DLM_PATH_ATTN_TC | DLM_PATH_ATTN_TCT;
    *done = true;
    return 0;
  }
  if (ragged && !transposed) p.ragged_q = 1;
  p.tr = tr[0];
  *paths |= transposed ? DLM_PATH_ATTN_TCT : DLM_PATH_ATTN_TC;
  const dim3 grid((unsigned)std::min<long long>(g_num_sms, p.n_items));
  cudaError_t e = transposed ? launch_k(attn_tct_kernel, grid, dim3(kTaThreads), (size_t)kTtSmem, st, pdl, *mkv, p)
                             : launch_k(attn_tc_kernel, grid, dim3(kTaThreads), (size_t)kTaSmem, st, pdl, *mkv, p);
  if (splits > 1 && e == cudaSuccess)
    e = launch_k(attn_combine_kernel, dim3((unsigned)TH), dim3(kFaDh), 0, st, pdl, out, (const float*)p.ws_o, (const float*)p.ws_ml, TH, splits, tr[1]);
  if (e != cudaSuccess) { set_err(err, "attn_tc launch: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
  *done = true;
  return 0;
}

// ------------------------------------------------------------------------------------------------
// weight-streaming GEMM launcher (T <= 128 tokens): picks the K split so ~2 CTAs per SM stream concurrently
// ------------------------------------------------------------------------------------------------
constexpr int kSkMaxSplits = 16;
constexpr int kSkMaxTokens = 128;

static void skinny_plan(int T, int N, int K, int epi, int force_splits, SkinnyParams* p, int* n_tiles) {
  const int per = epi == SK_SWIGLU ? 64 : 128;
  *n_tiles = (N + per - 1) / per;
  const int num_kb = (K + 63) / 64;
  int s = force_splits > 0 ? force_splits : (2 * g_num_sms) / *n_tiles;
  if (epi == SK_SWIGLU) s = 1;                                  // silu(g)*u needs complete sums
  s = std::max(1, std::min(std::min(s, kSkMaxSplits), std::max(1, num_kb / 4)));
  p->kb_per_split = (num_kb + s - 1) / s;
  p->splits = (num_kb + p->kb_per_split - 1) / p->kb_per_split;
  p->T = T; p->N = N; p->K = K;
  p->tpad = (T + 31) / 32 * 32;
  const int budget = 100 * 1024 - (epi == SK_SWIGLU ? 32 * 65 * 4 : 0);      // two CTAs per SM; 84 / 72 / 56 KB rings measured 1 / 3 / 14 % slower
  p->stages = std::max(2, std::min(std::min(p->kb_per_split, 8), budget / skinny_stage_bytes(p->tpad)));
  p->w_policy = DLM_L2_EVICT_FIRST;
}

// X: bf16 [x_rows_cap, K] (T valid rows); W: bf16 [w_rows, K].  SK_PARTIAL: p.out_f32 receives p.splits slices
// [split][T][ldc]; *splits_out tells the consumer how many to sum.
static int gemm_skinny(TmapCache& tc, std::string* err, const void* X, long long x_rows_cap, const void* W, long long w_rows,
                       int T, int N, int K, int epi, int force_splits, SkinnyParams p, int* splits_out, cudaStream_t st, bool pdl) {
  if (T <= 0) { if (splits_out) *splits_out = 0; return DLM_OK; }
  if (T > kSkMaxTokens || K % 8 || p.ldc <= 0) { set_err(err, "gemm_skinny: bad shape T=%d K=%d", T, K); return DLM_E_ARG; }
  int n_tiles = 0;
  skinny_plan(T, N, K, epi, force_splits, &p, &n_tiles);
  const TmapCache::Twin* tw = tc.twin(W);
  p.w_box = tw ? (epi == SK_SWIGLU ? 64 : 128) : 0;
  if (tw) p.up_row0 = (int)pad_to(p.up_row0, 128);
  const CUtensorMap* mw = tw ? tc.get_w(*tw, p.w_box) : tc.get(W, w_rows, K, epi == SK_SWIGLU ? 64 : 128);
  const CUtensorMap* mx = tc.get(X, x_rows_cap, K, p.tpad);
  if (!mw || !mx) { set_err(err, "cuTensorMapEncodeTiled failed (gemm_skinny X=%p W=%p)", X, W); return DLM_E_CUDA; }
  const int smem = skinny_smem_bytes(p.tpad, p.stages, epi);
  static bool configured[kMaxDevices][2] = {};
  cudaError_t e = cudaSuccess;
  if (!configured[g_dev][epi]) {
    e = epi == SK_SWIGLU ? cudaFuncSetAttribute(gemm_skinny_kernel<SK_SWIGLU>, cudaFuncAttributeMaxDynamicSharedMemorySize, 113 * 1024)
                         : cudaFuncSetAttribute(gemm_skinny_kernel<SK_PARTIAL>, cudaFuncAttributeMaxDynamicSharedMemorySize, 113 * 1024);
    if (e != cudaSuccess) { set_err(err, "gemm_skinny: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
    configured[g_dev][epi] = true;
  }
  dim3 grid(n_tiles, p.splits);
  e = epi == SK_SWIGLU ? launch_k(gemm_skinny_kernel<SK_SWIGLU>, grid, dim3(kSkThreads), (size_t)smem, st, pdl, *mw, *mx, p)
                       : launch_k(gemm_skinny_kernel<SK_PARTIAL>, grid, dim3(kSkThreads), (size_t)smem, st, pdl, *mw, *mx, p);
  if (e != cudaSuccess) { set_err(err, "gemm_skinny launch failed: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
  if (splits_out) *splits_out = p.splits;
  return DLM_OK;
}

template <typename TA, typename TW>
static void gemm_plain(float* C, const TA* A, const TW* W, int M, int N, int K, cudaStream_t st, bool pdl = false) {
  if (M <= 0) return;
  dim3 grid((N + 63) / 64, (M + 63) / 64);
  launch_k(gemm_plain_kernel<TA, TW>, grid, dim3(256), 0, st, pdl, C, A, W, M, N, K, K, K, N);
}

// Test op: contiguous q/k/v -> repack into a private paged store (64-token pages, identity page table) -> attention.
__global__ void repack_kv_kernel(bf16* __restrict__ store, const bf16* __restrict__ k, const bf16* __restrict__ v, int S, KvGeom g) {
  int j = blockIdx.x;
  int page = j / g.page_tokens, off = j % g.page_tokens;
  int n = g.n_kv_heads * g.head_dim;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    int h = i / g.head_dim, e = i % g.head_dim;
    store[g.offset(0, page, 0, h, off) + e] = k[(long long)j * n + i];
    store[g.offset(0, page, 1, h, off) + e] = v[(long long)j * n + i];
  }
}

static int attn_op_contiguous(const void* q, const void* k, const void* v, void* out, int Tq, int S, int H, int Hkv, int dh, int flash,
                              cudaStream_t st, std::string* err) {
  if (!q || !k || !v || !out || Tq <= 0 || S <= 0 || H <= 0 || Hkv <= 0 || H % Hkv || dh <= 0 || dh > 256) { set_err(err, "dlm_op_attention_bf16: bad arguments"); return DLM_E_ARG; }
  KvGeom g;
  g.n_kv_heads = Hkv; g.head_dim = dh; g.page_tokens = 64; g.max_pages_per_req = (S + 63) / 64; g.n_pages = g.max_pages_per_req;
  bf16* store = nullptr;
  int* meta = nullptr;
  const size_t store_bytes = (size_t)g.n_pages * g.page_elems() * 2;
  if (cudaMalloc(&store, store_bytes) != cudaSuccess || cudaMalloc(&meta, (size_t)(g.n_pages + 16 + Tq) * 4) != cudaSuccess) { set_err(err, "dlm_op_attention_bf16: allocation failed"); return DLM_E_CAPACITY; }
  cudaMemsetAsync(store, 0xFF, store_bytes, st);      // NaN pattern in the unused page tail: must not leak into results
  std::vector<int> h(g.n_pages + 16 + Tq, 0);
  for (int i = 0; i < g.n_pages; ++i) h[i] = i;
  int* hd = h.data() + g.n_pages;   // slot, q_off, q_len, q_pos0, kv_len
  hd[0] = 0; hd[1] = 0; hd[2] = Tq; hd[3] = 0; hd[4] = S;
  cudaMemcpyAsync(meta, h.data(), h.size() * 4, cudaMemcpyHostToDevice, st);
  repack_kv_kernel<<<S, 128, 0, st>>>(store, (const bf16*)k, (const bf16*)v, S, g);
  DLM_LAUNCH_CHECK();
  BatchDesc bd = {};
  bd.n = 1; bd.T = Tq; bd.max_q_len = Tq; bd.max_kv_len = S; bd.min_q_len = Tq;
  int* md = meta + g.n_pages;
  bd.slot = md; bd.q_off = md + 1; bd.q_len = md + 2; bd.q_pos0 = md + 3; bd.kv_len = md + 4; bd.tok_bi = md + 16;
  bd.order = md + 5;                                  // one request: [0]
  const float scale = 1.f / sqrtf((float)dh);
  int rc = DLM_OK;
  bool done = false;
  float* ws = nullptr;
  size_t wsb = (size_t)32 * Tq * H * (128 + 2) * 4;
  if (flash && cudaMalloc(&ws, wsb) != cudaSuccess) { cudaFree(store); cudaFree(meta); set_err(err, "dlm_op_attention_bf16: allocation failed"); return DLM_E_CAPACITY; }
  if (flash >= 2) {
    static TmapCache op_maps;
    op_maps.m.clear();
    rc = attn_tc_launch(op_maps, (bf16*)out, (const bf16*)q, store, 1, meta, bd, g, 0, H, scale, &ws, &wsb, st, false, err, &done, flash >= 102 ? 100 + (flash - 101) : flash - 1);
    if (!rc && !done) { set_err(err, "dlm_op_attention_bf16: tcgen05 kernel does not support d_h=%d", dh); rc = DLM_E_ARG; }
  } else if (flash) {
    rc = attn_flash_launch((bf16*)out, (const bf16*)q, store, meta, bd, g, 0, H, scale, &ws, &wsb, g_num_sms, st, false, err, &done);
    if (!rc && !done) { set_err(err, "dlm_op_attention_bf16: flash kernel does not support d_h=%d", dh); rc = DLM_E_ARG; }
  } else {
    attention_plain_kernel<bf16><<<dim3(Tq, H), 128, (size_t)S * 4, st>>>((bf16*)out, (const bf16*)q, store, meta, bd, g, 0, H, scale);
    DLM_LAUNCH_CHECK();
  }
  cudaError_t e = cudaStreamSynchronize(st);
  cudaFree(store); cudaFree(meta); if (ws) cudaFree(ws);
  if (!rc && e != cudaSuccess) { set_err(err, "dlm_op_attention_bf16: %s", cudaGetErrorString(e)); rc = DLM_E_CUDA; }
  return rc;
}

}  // namespace dlm

using namespace dlm;

// ------------------------------------------------------------------------------------------------
// Context
// ------------------------------------------------------------------------------------------------
struct Req {
  bool used = false;
  int P = 0, G = 0, B = 0, S = 0;
  float tau = 0.9f;
  int cur_block = 0;          // lowest-index block holding a MASK; == G/B when finished
  bool cache_valid = false;
  int n_masked = 0;           // whole request
  int n_masked_block = 0;     // current block
  int steps_done = 0;         // completed (non-dry) denoising steps (Step Predictor feature full_progress)
  std::vector<int> pages;
};

struct LayerW { void *wqkv, *wo, *wgu, *wd; };

struct HostBatch {
  int n = 0, T = 0, R = 0, max_q = 0, max_kv = 0, min_q = 1 << 30, n_big = 0, qt_big = 0, qt_total = 0;
  std::vector<int> slot, q_off, q_len, q_pos0, kv_len, blk_lo, blk_len, row_off, gen_lo, gen_len, tok_bi, order, qt_off;
  std::vector<float> tau;
  std::vector<char> refresh;     // per request: whole sequence recomputed this step
};

// Per-kernel-class device timing (DLM_OPT_KERNEL_TIMING): an event pair around every launch, resolved after the
// step's synchronize.  Feeds bench.py's roofline object and the ncu cross-check; off by default.
struct KProf {
  bool on = false;
  std::vector<cudaEvent_t> ev;
  std::vector<int> cls;
  size_t used = 0;
  double usec[DLM_K_COUNT] = {};
  long long launches[DLM_K_COUNT] = {};
  void begin(int k, cudaStream_t st) {
    if (ev.size() < used + 2) { ev.resize(used + 2); cudaEventCreate(&ev[used]); cudaEventCreate(&ev[used + 1]); }
    cudaEventRecord(ev[used], st);
    cls.push_back(k);
  }
  void end(cudaStream_t st) { cudaEventRecord(ev[used + 1], st); used += 2; }
  void collect() {      // after the stream has been synchronised
    for (size_t i = 0; i < cls.size(); ++i) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, ev[2 * i], ev[2 * i + 1]) == cudaSuccess) { usec[cls[i]] += 1000.0 * ms; launches[cls[i]]++; }
    }
    cls.clear(); used = 0;
  }
  void reset() { for (int i = 0; i < DLM_K_COUNT; ++i) { usec[i] = 0; launches[i] = 0; } }
  ~KProf() { for (auto e : ev) cudaEventDestroy(e); }
};

typedef std::tuple<int, int, int, int, int, int, int, int, int, int, int> GraphKey;   // kind, dry, n, T, R, max_q, max_kv, options, n_big, qt_big, qt_total
struct GraphEntry { int seen = 0; cudaGraphExec_t exec = nullptr; long long launches = 0; unsigned paths = 0; unsigned long long used = 0; std::vector<int> trace_cls; };
constexpr size_t kMaxGraphs = 64;          // captured step graphs kept per context (least recently used evicted)
constexpr int kMaxTraceSlots = 2048;       // launches of one step that DLM_OPT_TRACE can record

struct dlm_ctx {
  dlm_arch a;
  uint64_t seed;
  dlm_mem mem;
  int device = 0;              // the CUDA device the context lives on; every entry point binds the calling thread to it
  int num_sms = 148;
  long long launches = 0;      // kernels launched for this context (dlm_launch_count)
  bool own_stream = false;
  cudaStream_t st = nullptr;
  std::string err;
  std::vector<void*> allocs;
  size_t esize = 4;            // bytes per weight / activation element
  bool bf16_model = false;
  bool w_tiled = false;        // projection / LM-head weights in tiled storage (bf16 models)

  // weights
  void *E = nullptr, *Wlm = nullptr;
  std::vector<LayerW> L;
  float *rope_cos = nullptr, *rope_sin = nullptr;
  // request state
  int* tokens = nullptr;       // [max_requests, max_seq]
  float* conf_state = nullptr; // [max_requests, max_seq] per position: confidence last seen while masked (NEXT-1)
  bool want_feat = false;      // this step's caller asked for the Step Predictor features
  int* page_table = nullptr;   // [max_requests, max_pages_per_req]
  void* kv_store = nullptr;
  KvGeom kg;
  std::vector<Req> reqs;
  std::vector<int> free_pages;
  // activations
  int Tmax = 0, Rmax = 0, n_tiles = 0;
  float *x = nullptr, *qkv = nullptr, *tmp = nullptr, *logits = nullptr;
  void *u = nullptr, *q = nullptr, *attn = nullptr, *act = nullptr, *hf = nullptr;
  RowPartial* part = nullptr;
  int* row_src = nullptr;
  // descriptors / results
  int* desc_dev = nullptr; int* desc_host = nullptr; size_t desc_cap_ints = 0;
  char* out_dev = nullptr; char* out_host = nullptr; size_t out_bytes = 0;
  // attention split-KV scratch
  float* attn_ws = nullptr; size_t attn_ws_bytes = 0;
  float* part_x = nullptr;     // [splits][T][d] split-K slices of the O / down projections (part_rows rows in all)
  long long part_rows = 0, qkv_rows = 0;
  // options
  int opt_simple = 0, opt_dump = 0, opt_graph = 1, opt_flash = 1, opt_pdl = 1, opt_skinny = 1, opt_pair = 1, opt_tcattn = 1, opt_fuse_rope = 1;
  int opt_trace = 0;
  int opt_mega = 0;            // whole-stack persistent kernel for cached steps of <= 64 tokens: correct, but 4.0 ms per C2 cached step against
                               // 3.19 ms for the per-stage kernels (its grid-wide phase boundaries cost what kernel boundaries cost), so off by default
  CUtensorMap* mega_wmaps = nullptr;   // device array [n_layers][4] of the tiled weight maps
  unsigned int* mega_bar = nullptr;    // its phase counter
  unsigned long long* mega_ts = nullptr, *mega_ts_host = nullptr;   // optional phase timestamps (DLM_OPT_MEGA_PHASE_TS)
  int opt_mega_ts = 0;
  void* u2 = nullptr;          // second RMSNorm output buffer (gate/up input) of the whole-stack kernel
  int opt_tct_min_items = 64;  // fewest (request, KV head, query tile) items for which a step takes the tcgen05 attention kernels
  int opt_mask() const { return opt_simple | (opt_flash << 1) | (opt_pdl << 2) | (opt_skinny << 3) | (opt_pair << 4) | (opt_tcattn << 5) | (opt_fuse_rope << 6) | (opt_trace << 7) | (opt_mega << 8) | (opt_mega_ts << 9); }
  std::map<GraphKey, GraphEntry> graphs;
  unsigned long long graph_clock = 0;
  unsigned paths = 0, last_paths = 0;   // DLM_PATH_* of the step being enqueued / of the last step
  // in-kernel timeline (DLM_OPT_TRACE): one record of 3 x u64 per launch, classes in launch order
  unsigned long long* trace_dev = nullptr;
  std::vector<int> trace_cls, last_trace_cls;
  std::vector<unsigned long long> trace_host;
  int cur_cls = 0;
  TraceSlot tslot() {
    if (!opt_trace || !trace_dev || (int)trace_cls.size() >= kMaxTraceSlots) return TraceSlot{nullptr};
    trace_cls.push_back(cur_cls);
    return TraceSlot{trace_dev + 3 * (trace_cls.size() - 1)};
  }
  // debug dump
  std::map<std::pair<int, int>, void*> dump;   // (layer, which) -> device copy [T, width]
  HostBatch last_batch;
  bool last_refresh = false;
  int dump_T = 0;
  // timing
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  float last_usec = 0.f;
  TmapCache tmaps;
  KProf kprof;

  void* dalloc(size_t bytes) {
    void* p = nullptr;
    bytes = (bytes + 255) & ~(size_t)255;
    if (mem.alloc) p = mem.alloc(bytes, mem.user);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) p = nullptr;
    if (p) allocs.push_back(p);
    return p;
  }
  void dfree_all() {
    for (void* p : allocs) { if (mem.free) mem.free(p, mem.user); else if (!mem.alloc) cudaFree(p); }
    allocs.clear();
  }
};

struct KScope {
  dlm_ctx* c;
  KScope(dlm_ctx* c_, int k) : c(c_) { c->cur_cls = k; if (c->kprof.on) c->kprof.begin(k, c->st); }
  ~KScope() { if (c->kprof.on) c->kprof.end(c->st); }
};

// Every entry point that takes a ctx binds the calling thread to the context's device for the duration of the call (a
// request may be imported into a context on another GPU of the same process) and credits its launches to the context.
static thread_local int g_guard_depth = 0;   // entry points nest (dlm_profile_step_costs_ex -> dlm_refresh_step -> run_step)
struct DevGuard {
  dlm_ctx* c;
  int prev = -1;
  long long l0;
  explicit DevGuard(dlm_ctx* c_) : c(c_), l0(g_launches) {
    if (!c) return;
    ++g_guard_depth;
    cudaGetDevice(&prev);
    if (prev != c->device) cudaSetDevice(c->device);
    g_dev = c->device; g_num_sms = c->num_sms;
  }
  ~DevGuard() {
    if (!c) return;
    if (--g_guard_depth == 0) c->launches += g_launches - l0;      // only the outermost guard credits the launches (once)
    if (prev >= 0 && prev != c->device) cudaSetDevice(prev);
  }
};

static int norm_threads(int d) { return std::min(1024, ((d / 4) + 31) / 32 * 32); }

// a2 / a7 / a10: latency kernel (one block per row) for small steps, warp-per-row throughput kernel from 1024 rows on.
// Same arithmetic per row up to the order of the sum of squares.
template <typename TE>
static void launch_rmsnorm(dlm_ctx* c, TE* u, float* x, const int* row_src, int rows, int d, float eps, const float* part, int n_part,
                           long long part_stride, bool pdl) {
  const TraceSlot tr = c->tslot();
  if (rows >= 1024 && d <= 4096)        // register-resident row: 3.46 -> 2.00 ms per C3 mixed step; slower below ~1000 rows
    launch_k(rmsnorm_warp_kernel<TE>, dim3((rows + 3) / 4), dim3(128), 0, c->st, pdl, u, x, row_src, rows, d, eps, part, n_part, part_stride, tr);
  else if (rows >= 1024)
    launch_k(rmsnorm_rows_kernel<TE>, dim3((rows + 3) / 4), dim3(128), 0, c->st, pdl, u, x, row_src, rows, d, eps, part, n_part, part_stride, tr);
  else
  {
    // more rows than two resident 1024-thread blocks per SM can hold: 256-thread blocks (4 float4 per thread) keep every
    // row of a 512-token step in flight in one wave
    int threads = norm_threads(d);
    if (rows > 2 * g_num_sms && d >= 1024 && d <= 4096) threads = 256;
    launch_k(rmsnorm_kernel<TE>, dim3(rows), dim3(threads), 0, c->st, pdl, u, x, row_src, d, eps, part, n_part, part_stride, tr);
  }
}

static int nqkv(const dlm_arch& a) { return (a.n_heads + 2 * a.n_kv_heads) * a.head_dim; }

// ------------------------------------------------------------------------------------------------
// Init
// ------------------------------------------------------------------------------------------------
template <typename TW>
static void gen_weight(dlm_ctx* c, void* dst, long long n, int tid) {
  unsigned long long key = mix64(c->seed + DLM_GOLD * (unsigned long long)(tid + 1));
  float cst = (float)((double)c->a.init_std / sqrt(4294967295.0 / 3.0));
  int blocks = (int)std::min<long long>((n + 255) / 256, 148 * 16);
  init_weight_kernel<TW><<<blocks, 256, 0, c->st>>>((TW*)dst, n, key, cst, c->a.weight_dtype == DLM_DTYPE_BF16_PRECISE ? 1 : 0);
  DLM_LAUNCH_CHECK();
}
static void gen_weight_any(dlm_ctx* c, void* dst, long long n, int tid) {
  if (c->bf16_model) gen_weight<bf16>(c, dst, n, tid); else gen_weight<float>(c, dst, n, tid);
}
// One [rows, cols] part of a projection matrix (own tensor id, Definition W) from row row0 of the matrix: row-major, and into
// the tiled twin when the matrix has one (its allocation was zeroed, padding stays zero; the twin's row0 is row0t).
static void gen_weight_part(dlm_ctx* c, void* mat, long long row0, long long row0t, long long rows, long long cols, int tid) {
  gen_weight_any(c, (char*)mat + row0 * cols * (c->bf16_model ? 2 : 4), rows * cols, tid);
  const TmapCache::Twin* tw = c->tmaps.twin(mat);
  if (!tw) return;
  unsigned long long key = mix64(c->seed + DLM_GOLD * (unsigned long long)(tid + 1));
  float cst = (float)((double)c->a.init_std / sqrt(4294967295.0 / 3.0));
  int blocks = (int)std::min<long long>((rows * cols + 255) / 256, 148 * 16);
  init_weight_tiled_kernel<bf16><<<blocks, 256, 0, c->st>>>((bf16*)tw->ptr, rows, cols, row0t, tw->rows_pad / 128, key, cst);
  DLM_LAUNCH_CHECK();
}

static int validate_arch(const dlm_arch* a, std::string* err) {
  if (!a) { set_err(err, "arch is NULL"); return DLM_E_ARG; }
#define REQ(cond) if (!(cond)) { set_err(err, "dlm_init: invalid arch: %s", #cond); return DLM_E_ARG; }
  REQ(a->n_layers > 0 && a->d_model > 0 && a->n_heads > 0 && a->n_kv_heads > 0 && a->head_dim > 0 && a->d_ffn > 0);
  REQ(a->vocab > 1 && a->mask_id >= 0 && a->mask_id < a->vocab);
  REQ(a->n_heads % a->n_kv_heads == 0 && a->head_dim % 2 == 0 && a->head_dim <= 256);
  REQ(a->d_model % 4 == 0 && a->d_model <= 16384);
  REQ(a->weight_dtype == DLM_DTYPE_F32 || a->weight_dtype == DLM_DTYPE_BF16 || a->weight_dtype == DLM_DTYPE_BF16_PRECISE);
  REQ(a->max_requests > 0 && a->max_seq > 0 && a->max_block > 0 && a->max_block <= 64);
  REQ(a->kv_page_tokens > 0 && a->max_batch_tokens > 0);
  if (a->weight_dtype == DLM_DTYPE_BF16) {
    REQ(a->d_model % 8 == 0 && a->d_ffn % 8 == 0 && (a->n_heads * a->head_dim) % 8 == 0);
  }
#undef REQ
  return DLM_OK;
}

extern "C" int dlm_init_ex(const dlm_arch* arch, uint64_t seed, const dlm_mem* mem, dlm_ctx** out) {
  if (!out) { set_err(&g_init_error, "out is NULL"); return DLM_E_ARG; }
  *out = nullptr;
  int rc = validate_arch(arch, &g_init_error);
  if (rc) return rc;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    set_err(&g_init_error, "no CUDA device: libdlm has no CPU fallback");
    return DLM_E_CUDA;
  }
  dlm_ctx* c = new dlm_ctx();
  c->a = *arch;
  c->seed = seed;
  if (mem) c->mem = *mem; else memset(&c->mem, 0, sizeof c->mem);
  std::string* err = &g_init_error;
  cudaGetDevice(&c->device);             // the context lives on the caller's current device
#define FAIL(code, ...) do { set_err(err, __VA_ARGS__); dlm_destroy(c); return code; } while (0)
  if (c->mem.cuda_stream) c->st = (cudaStream_t)c->mem.cuda_stream;
  else { if (cudaStreamCreateWithFlags(&c->st, cudaStreamNonBlocking) != cudaSuccess) FAIL(DLM_E_CUDA, "cudaStreamCreate failed"); c->own_stream = true; }
  cudaDeviceProp prop;
  int dev = 0;
  cudaGetDevice(&dev);
  cudaGetDeviceProperties(&prop, dev);
  if (dev < 0 || dev >= kMaxDevices) FAIL(DLM_E_CUDA, "device ordinal %d not supported", dev);
  c->device = dev; c->num_sms = prop.multiProcessorCount;
  g_dev = dev; g_num_sms = c->num_sms;
  const dlm_arch& a = c->a;
  c->bf16_model = a.weight_dtype == DLM_DTYPE_BF16;
  c->esize = c->bf16_model ? 2 : 4;
  if (c->bf16_model && prop.major != 10) FAIL(DLM_E_CUDA, "bf16 path needs an sm_100 device (tcgen05/TMA); found sm_%d%d", prop.major, prop.minor);
  const size_t es = c->esize;
  const long long d = a.d_model, F = a.d_ffn, V = a.vocab, HQ = (long long)a.n_heads * a.head_dim, NQKV = nqkv(a);
#define ALLOC(ptr, bytes) do { ptr = (decltype(ptr))c->dalloc((size_t)(bytes)); if (!ptr) FAIL(DLM_E_CAPACITY, "device allocation of %lld bytes failed (%s)", (long long)(bytes), #ptr); } while (0)
  // ---- weights (Definition W) ----
  // bf16 models keep every layer's projection matrices twice: row-major for the compute-bound kernels (CTA-pair GEMM) and
  // tiled (make_tmap_w_tiled) for the weight-streaming kernels of steps with <= 128 tokens, which gain 5-6 % from the
  // contiguous 16 KB tiles while the pair GEMM loses 7 % on them.  14 GB of 180 GB HBM at the 8B shape.
  c->w_tiled = c->bf16_model;
#define ALLOC_W(ptr, rows, cols, rows_tiled) do { ALLOC(ptr, (long long)(rows) * (cols) * es); \
    if (c->w_tiled) { void* tw_ = nullptr; const long long rp_ = pad_to(rows_tiled, 128), kp_ = pad_to(cols, 64); \
      ALLOC(tw_, rp_ * kp_ * es); cudaMemsetAsync(tw_, 0, (size_t)(rp_ * kp_ * es), c->st); c->tmaps.tiled[ptr] = {tw_, rp_, kp_}; } } while (0)
  const long long Fp = pad_to(F, 128);                       // row of the up projection inside the tiled gate/up matrix
  ALLOC(c->E, V * d * es);
  ALLOC(c->Wlm, V * d * es);        // the LM head's 128-row kernel measured the same on either layout: row-major only
  gen_weight_any(c, c->E, V * d, 0);
  gen_weight_any(c, c->Wlm, V * d, 1);
  c->L.resize(a.n_layers);
  const long long HKV = (long long)a.n_kv_heads * a.head_dim;
  for (int l = 0; l < a.n_layers; ++l) {
    LayerW& w = c->L[l];
    ALLOC_W(w.wqkv, NQKV, d, NQKV);
    ALLOC_W(w.wo, d, HQ, d);
    ALLOC_W(w.wgu, 2 * F, d, Fp + F);
    ALLOC_W(w.wd, d, F, d);
    const int t0 = 16 * (l + 1);
    gen_weight_part(c, w.wqkv, 0, 0, HQ, d, t0 + 0);
    gen_weight_part(c, w.wqkv, HQ, HQ, HKV, d, t0 + 1);
    gen_weight_part(c, w.wqkv, HQ + HKV, HQ + HKV, HKV, d, t0 + 2);
    gen_weight_part(c, w.wo, 0, 0, d, HQ, t0 + 3);
    gen_weight_part(c, w.wgu, 0, 0, F, d, t0 + 4);
    gen_weight_part(c, w.wgu, F, Fp, F, d, t0 + 5);
    gen_weight_part(c, w.wd, 0, 0, d, F, t0 + 6);
  }
#undef ALLOC_W
  // ---- RoPE table ----
  const int half = a.head_dim / 2;
  ALLOC(c->rope_cos, (size_t)a.max_seq * half * 4);
  ALLOC(c->rope_sin, (size_t)a.max_seq * half * 4);
  init_rope_kernel<<<(a.max_seq * half + 255) / 256, 256, 0, c->st>>>(c->rope_cos, c->rope_sin, a.max_seq, half, (double)a.rope_theta);
  DLM_LAUNCH_CHECK();
  // ---- request state + paged K/V store ----
  ALLOC(c->tokens, (size_t)a.max_requests * a.max_seq * 4);
  c->kg.n_kv_heads = a.n_kv_heads; c->kg.head_dim = a.head_dim; c->kg.page_tokens = a.kv_page_tokens;
  c->kg.max_pages_per_req = (a.max_seq + a.kv_page_tokens - 1) / a.kv_page_tokens;
  long long pool_tokens = a.kv_pool_tokens > 0 ? a.kv_pool_tokens : (long long)a.max_requests * a.max_seq;
  c->kg.n_pages = std::min<long long>((pool_tokens + a.kv_page_tokens - 1) / a.kv_page_tokens + a.max_requests,
                                      (long long)a.max_requests * c->kg.max_pages_per_req);
  ALLOC(c->page_table, (size_t)a.max_requests * c->kg.max_pages_per_req * 4);
  ALLOC(c->kv_store, (size_t)a.n_layers * c->kg.n_pages * c->kg.page_elems() * es);
  cudaMemsetAsync(c->page_table, 0, (size_t)a.max_requests * c->kg.max_pages_per_req * 4, c->st);
  c->reqs.resize(a.max_requests);
  for (long long p = c->kg.n_pages - 1; p >= 0; --p) c->free_pages.push_back((int)p);
  // ---- activations ----
  c->Tmax = a.max_batch_tokens;
  c->Rmax = a.max_requests * a.max_block;
  c->n_tiles = c->bf16_model ? (int)((V + 127) / 128) : 1;
  ALLOC(c->x, (size_t)c->Tmax * d * 4);
  // fp32 slice capacity (rows): split-K slices of the skinny path (<= 16 x 128 tokens) and of the pair path (<= 4 x M)
  c->qkv_rows = std::max<long long>(std::max<long long>(c->Tmax, (long long)kSkMaxSplits * kSkMaxTokens), std::min<long long>(3LL * c->Tmax, 4096));
  c->part_rows = std::max<long long>((long long)kSkMaxSplits * kSkMaxTokens, std::min<long long>(4LL * c->Tmax, 8192));
  ALLOC(c->qkv, (size_t)c->qkv_rows * NQKV * 4);
  if (c->bf16_model) ALLOC(c->part_x, (size_t)c->part_rows * d * 4);
  ALLOC(c->u, (size_t)c->Tmax * d * es);
  ALLOC(c->q, (size_t)c->Tmax * HQ * es);
  ALLOC(c->attn, (size_t)c->Tmax * HQ * es);
  ALLOC(c->act, (size_t)c->Tmax * F * es);
  ALLOC(c->hf, (size_t)std::max(c->Rmax, 128) * d * es);
  ALLOC(c->part, (size_t)c->Rmax * std::max(c->n_tiles, 1) * sizeof(RowPartial));
  ALLOC(c->row_src, (size_t)c->Rmax * 4);
  if (c->bf16_model) {      // split-KV partials of the attention kernels: fixed size, so captured graphs stay valid
    c->attn_ws_bytes = (size_t)8 * std::min(c->Tmax, 1024) * a.n_heads * (128 + 2) * 4;
    ALLOC(c->attn_ws, c->attn_ws_bytes);
  }
  c->desc_cap_ints = (size_t)14 * a.max_requests + c->Tmax + 64;      // 13 n + 1 + T used
  ALLOC(c->desc_dev, c->desc_cap_ints * 4);
  if (cudaMallocHost(&c->desc_host, c->desc_cap_ints * 4) != cudaSuccess) FAIL(DLM_E_CUDA, "cudaMallocHost failed");
  c->out_bytes = (size_t)a.max_requests * 4 + (size_t)c->Rmax * 4 * 6 + (size_t)a.max_requests * 5 * 4;     // + confidence features
  ALLOC(c->conf_state, (size_t)a.max_requests * a.max_seq * 4);
  cudaMemsetAsync(c->conf_state, 0, (size_t)a.max_requests * a.max_seq * 4, c->st);
  ALLOC(c->out_dev, c->out_bytes);
  if (cudaMallocHost(&c->out_host, c->out_bytes) != cudaSuccess) FAIL(DLM_E_CUDA, "cudaMallocHost failed");
  ALLOC(c->trace_dev, (size_t)kMaxTraceSlots * 3 * 8);
  if (c->bf16_model) {            // whole-stack kernel: second norm buffer, phase counter, the tiled weight maps of every layer
    ALLOC(c->u2, (size_t)kMgMaxTpad * d * es);
    ALLOC(c->mega_bar, 4096);
    ALLOC(c->mega_ts, (size_t)(kMgPhasesPerLayer * a.n_layers + 2) * 8);
    ALLOC(c->mega_wmaps, (size_t)a.n_layers * 4 * sizeof(CUtensorMap));
    std::vector<CUtensorMap> hm((size_t)a.n_layers * 4);
    bool ok = true;
    for (int l = 0; l < a.n_layers && ok; ++l) {
      const void* w4[4] = {c->L[l].wqkv, c->L[l].wo, c->L[l].wgu, c->L[l].wd};
      for (int gi = 0; gi < 4 && ok; ++gi) {
        const TmapCache::Twin* tw = c->tmaps.twin(w4[gi]);
        ok = tw && make_tmap_w_tiled(&hm[(size_t)l * 4 + gi], tw->ptr, tw->rows_pad, tw->k_pad, gi == 2 ? 64 : 128);
      }
    }
    if (!ok) FAIL(DLM_E_CUDA, "cuTensorMapEncodeTiled failed (tiled weight maps)");
    if (cudaMemcpyAsync(c->mega_wmaps, hm.data(), hm.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, c->st) != cudaSuccess || cudaStreamSynchronize(c->st) != cudaSuccess)
      FAIL(DLM_E_CUDA, "tensor map upload failed");
  }
  cudaEventCreate(&c->ev0);
  cudaEventCreate(&c->ev1);
  cudaError_t e = cudaStreamSynchronize(c->st);
  if (e != cudaSuccess) FAIL(DLM_E_CUDA, "weight generation failed: %s", cudaGetErrorString(e));
#undef ALLOC
#undef FAIL
  c->launches = 0;                       // weight generation is set-up, not step work
  *out = c;
  return DLM_OK;
}

extern "C" int dlm_init(const dlm_arch* arch, uint64_t seed, dlm_ctx** out) { return dlm_init_ex(arch, seed, nullptr, out); }

extern "C" void dlm_destroy(dlm_ctx* c) {
  if (!c) return;
  int prev = -1;
  cudaGetDevice(&prev);
  if (prev != c->device) cudaSetDevice(c->device);
  if (c->st) cudaStreamSynchronize(c->st);
  for (auto& kv : c->dump) cudaFree(kv.second);
  for (auto& g : c->graphs) if (g.second.exec) cudaGraphExecDestroy(g.second.exec);
  if (c->tmp) cudaFree(c->tmp);
  if (c->logits) cudaFree(c->logits);
  c->dfree_all();
  if (c->desc_host) cudaFreeHost(c->desc_host);
  if (c->out_host) cudaFreeHost(c->out_host);
  if (c->ev0) cudaEventDestroy(c->ev0);
  if (c->ev1) cudaEventDestroy(c->ev1);
  if (c->own_stream && c->st) cudaStreamDestroy(c->st);
  if (prev >= 0 && prev != c->device) cudaSetDevice(prev);
  delete c;
}

extern "C" const char* dlm_last_error(dlm_ctx* c) { return c ? c->err.c_str() : g_init_error.c_str(); }
extern "C" int64_t dlm_launch_count(dlm_ctx* c) { return c ? c->launches : 0; }
extern "C" uint32_t dlm_last_step_kernels(dlm_ctx* c) { return c ? c->last_paths : 0; }
extern "C" float dlm_last_step_usec(dlm_ctx* c) { return c ? c->last_usec : 0.f; }

extern "C" int dlm_kernel_times(dlm_ctx* c, dlm_kernel_time* rows, int32_t cap, int32_t* n_rows, int32_t reset) {
  if (!c || !rows || !n_rows) return DLM_E_ARG;
  *n_rows = 0;
  for (int k = 0; k < DLM_K_COUNT && *n_rows < cap; ++k) {
    if (!c->kprof.launches[k]) continue;
    rows[*n_rows].kernel = k; rows[*n_rows].launches = (int32_t)c->kprof.launches[k]; rows[*n_rows].usec = (float)c->kprof.usec[k];
    (*n_rows)++;
  }
  if (reset) c->kprof.reset();
  return DLM_OK;
}

extern "C" int dlm_step_trace(dlm_ctx* c, dlm_trace_row* rows, int32_t cap, int32_t* n_rows) {
  if (!c || !rows || !n_rows) return DLM_E_ARG;
  *n_rows = 0;
  const size_t n = std::min(c->last_trace_cls.size(), c->trace_host.size() / 3);
  unsigned long long t0 = ~0ULL;
  for (size_t i = 0; i < n; ++i) t0 = std::min(t0, c->trace_host[3 * i]);
  for (size_t i = 0; i < n && *n_rows < cap; ++i) {
    const unsigned long long b = c->trace_host[3 * i], w = c->trace_host[3 * i + 1], e = ~c->trace_host[3 * i + 2];
    if (b == ~0ULL) continue;                  // a record that no launch used
    dlm_trace_row& r = rows[(*n_rows)++];
    r.kernel = c->last_trace_cls[i]; r.slot = (int32_t)i;
    r.begin_us = (float)((double)(b - t0) * 1e-3);
    r.wait_us = w == ~0ULL ? r.begin_us : (float)((double)(w - t0) * 1e-3);
    r.end_us = c->trace_host[3 * i + 2] == ~0ULL ? r.wait_us : (float)((double)(e - t0) * 1e-3);
  }
  return DLM_OK;
}

extern "C" int dlm_layer_kernel_phases(dlm_ctx* c, float* usec, int32_t cap) {
  if (!c || !usec || cap <= 0 || !c->mega_ts) return DLM_E_ARG;
  DevGuard dev_guard(c);
  const int n = std::min<int>(cap, kMgPhasesPerLayer * c->a.n_layers + 1);
  std::vector<unsigned long long> h(n);
  if (cudaMemcpy(h.data(), c->mega_ts, (size_t)n * 8, cudaMemcpyDeviceToHost) != cudaSuccess) return DLM_E_CUDA;
  for (int i = 0; i < n; ++i) usec[i] = (float)((double)(h[i] - h[0]) * 1e-3);
  return n;
}

extern "C" int dlm_set_option(dlm_ctx* c, int32_t key, int32_t value) {
  if (!c) return DLM_E_ARG;
  switch (key) {
    case DLM_OPT_SIMPLE_KERNELS: c->opt_simple = value != 0; return DLM_OK;
    case DLM_OPT_DEBUG_DUMP: c->opt_dump = value; return DLM_OK;
    case DLM_OPT_CUDA_GRAPH: c->opt_graph = value != 0; return DLM_OK;
    case DLM_OPT_FLASH_ATTENTION: c->opt_flash = value != 0; return DLM_OK;
    case DLM_OPT_KERNEL_TIMING: c->kprof.on = value != 0; return DLM_OK;
    case DLM_OPT_PDL: c->opt_pdl = value != 0; return DLM_OK;
    case DLM_OPT_SKINNY_GEMM: c->opt_skinny = value != 0; return DLM_OK;
    case DLM_OPT_PAIR_GEMM: c->opt_pair = value != 0; return DLM_OK;
    case DLM_OPT_TC_ATTENTION: c->opt_tcattn = value != 0; return DLM_OK;
    case DLM_OPT_FUSE_ROPE: c->opt_fuse_rope = value != 0; return DLM_OK;
    case DLM_OPT_TRACE: c->opt_trace = value != 0; return DLM_OK;
    case DLM_OPT_LAYER_KERNEL: c->opt_mega = value != 0; return DLM_OK;
    case DLM_OPT_LAYER_KERNEL_PHASE_TS: c->opt_mega_ts = value != 0; return DLM_OK;
    case DLM_OPT_TCT_MIN_ITEMS: {
      // selects the attention kernel a step enqueues but is not part of the graph key: a captured graph of the old selection
      // must not be replayed (an A/B timing on one context would measure the same kernel twice)
      const int v = std::max(1, value);
      if (v != c->opt_tct_min_items) {
        DevGuard dev_guard(c);
        if (c->st) cudaStreamSynchronize(c->st);
        for (auto& g : c->graphs) if (g.second.exec) cudaGraphExecDestroy(g.second.exec);
        c->graphs.clear();
      }
      c->opt_tct_min_items = v;
      return DLM_OK;
    }
  }
  set_err(&c->err, "unknown option %d", key);
  return DLM_E_ARG;
}

// ------------------------------------------------------------------------------------------------
// Requests
// ------------------------------------------------------------------------------------------------
static Req* get_req(dlm_ctx* c, int r) {
  if (!c || r < 0 || r >= (int)c->reqs.size() || !c->reqs[r].used) return nullptr;
  return &c->reqs[r];
}

static void recount(const dlm_arch& a, Req& q, const int* tok) {
  q.n_masked = 0;
  q.cur_block = q.G / q.B;
  q.n_masked_block = 0;
  for (int b = 0; b < q.G / q.B; ++b) {
    int m = 0;
    for (int j = 0; j < q.B; ++j) m += tok[q.P + b * q.B + j] == a.mask_id;
    q.n_masked += m;
    if (m && q.cur_block == q.G / q.B) { q.cur_block = b; q.n_masked_block = m; }
  }
}

extern "C" int dlm_request_add(dlm_ctx* c, const int32_t* prompt, int32_t P, int32_t G, int32_t B, float tau, int32_t* out_req) {
  DevGuard dev_guard(c);
  if (!c) return DLM_E_ARG;
  const dlm_arch& a = c->a;
  if (!prompt || !out_req || P < 0 || G <= 0 || B <= 0 || B > a.max_block || G % B) {
    set_err(&c->err, "dlm_request_add: bad arguments (P=%d G=%d B=%d; G %% B must be 0, B <= max_block=%d)", P, G, B, a.max_block);
    return DLM_E_ARG;
  }
  const int S = P + G;
  if (S > a.max_seq) { set_err(&c->err, "dlm_request_add: S=%d exceeds max_seq=%d", S, a.max_seq); return DLM_E_CAPACITY; }
  for (int i = 0; i < P; ++i)
    if (prompt[i] < 0 || prompt[i] >= a.vocab) { set_err(&c->err, "dlm_request_add: prompt id %d out of range", prompt[i]); return DLM_E_ARG; }
  int slot = -1;
  for (int i = 0; i < (int)c->reqs.size(); ++i) if (!c->reqs[i].used) { slot = i; break; }
  if (slot < 0) { set_err(&c->err, "dlm_request_add: all %d request slots in use", a.max_requests); return DLM_E_CAPACITY; }
  const int need = (S + a.kv_page_tokens - 1) / a.kv_page_tokens;
  if ((int)c->free_pages.size() < need) { set_err(&c->err, "dlm_request_add: K/V pool exhausted (%d pages needed, %zu free)", need, c->free_pages.size()); return DLM_E_CAPACITY; }
  Req& q = c->reqs[slot];
  q = Req();
  q.used = true; q.P = P; q.G = G; q.B = B; q.S = S; q.tau = tau;
  q.cur_block = 0; q.cache_valid = false; q.n_masked = G; q.n_masked_block = B;
  std::vector<int> row(c->kg.max_pages_per_req, 0);
  for (int i = 0; i < need; ++i) { q.pages.push_back(c->free_pages.back()); c->free_pages.pop_back(); row[i] = q.pages[i]; }
  std::vector<int> tok(S);
  for (int i = 0; i < P; ++i) tok[i] = prompt[i];
  for (int i = P; i < S; ++i) tok[i] = a.mask_id;
  cudaError_t e = cudaMemcpyAsync(c->tokens + (size_t)slot * a.max_seq, tok.data(), (size_t)S * 4, cudaMemcpyHostToDevice, c->st);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->conf_state + (size_t)slot * a.max_seq, 0, (size_t)a.max_seq * 4, c->st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(c->page_table + (size_t)slot * c->kg.max_pages_per_req, row.data(), row.size() * 4, cudaMemcpyHostToDevice, c->st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
  if (e != cudaSuccess) {                      // nothing is partially applied: give the slot and its pages back
    for (int pg : q.pages) c->free_pages.push_back(pg);
    q = Req();
    set_err(&c->err, "dlm_request_add: %s", cudaGetErrorString(e));
    return DLM_E_CUDA;
  }
  *out_req = slot;
  return DLM_OK;
}

extern "C" int dlm_request_set_tokens(dlm_ctx* c, int32_t r, const int32_t* tokens, int32_t n, int32_t keep_cache) {
  DevGuard dev_guard(c);
  Req* q = get_req(c, r);
  if (!q || !tokens) { if (c) set_err(&c->err, "dlm_request_set_tokens: bad request %d", r); return DLM_E_ARG; }
  if (n != q->S) { set_err(&c->err, "dlm_request_set_tokens: n=%d != S=%d", n, q->S); return DLM_E_ARG; }
  for (int i = 0; i < n; ++i)
    if (tokens[i] < 0 || tokens[i] >= c->a.vocab || (i < q->P && tokens[i] == c->a.mask_id)) { set_err(&c->err, "dlm_request_set_tokens: bad id at %d", i); return DLM_E_ARG; }
  CU_TRY(&c->err, cudaMemcpyAsync(c->tokens + (size_t)r * c->a.max_seq, tokens, (size_t)n * 4, cudaMemcpyHostToDevice, c->st));
  CU_TRY(&c->err, cudaStreamSynchronize(c->st));
  const int old_block = q->cur_block;
  recount(c->a, *q, tokens);
  if (!keep_cache || q->cur_block != old_block) q->cache_valid = false;
  return DLM_OK;
}

extern "C" int dlm_request_remove(dlm_ctx* c, int32_t r) {
  Req* q = get_req(c, r);
  if (!q) { if (c) set_err(&c->err, "dlm_request_remove: bad request %d", r); return DLM_E_ARG; }
  for (int p : q->pages) c->free_pages.push_back(p);
  *q = Req();
  return DLM_OK;
}

extern "C" int dlm_request_tokens(dlm_ctx* c, int32_t r, int32_t* out, int32_t cap) {
  DevGuard dev_guard(c);
  Req* q = get_req(c, r);
  if (!q || !out) { if (c) set_err(&c->err, "dlm_request_tokens: bad request %d", r); return DLM_E_ARG; }
  if (cap < q->S) { set_err(&c->err, "dlm_request_tokens: cap=%d < S=%d", cap, q->S); return DLM_E_CAPACITY; }
  CU_TRY(&c->err, cudaMemcpyAsync(out, c->tokens + (size_t)r * c->a.max_seq, (size_t)q->S * 4, cudaMemcpyDeviceToHost, c->st));
  CU_TRY(&c->err, cudaStreamSynchronize(c->st));
  return q->S;
}

// ---- migration blob (include/dlm.h): header of 10 words, tokens[S], conf_state[S] ----
namespace {
constexpr int32_t kBlobMagic = 0x524D4C44, kBlobVersion = 1, kBlobHeaderWords = 10;
}

extern "C" int64_t dlm_request_export(dlm_ctx* c, int32_t r, void* blob, int64_t cap) {
  DevGuard dev_guard(c);
  Req* q = get_req(c, r);
  if (!q) { if (c) set_err(&c->err, "dlm_request_export: bad request %d", r); return DLM_E_ARG; }
  const int64_t need = (int64_t)kBlobHeaderWords * 4 + (int64_t)q->S * 8;
  if (!blob || cap < need) return need;
  int32_t* h = static_cast<int32_t*>(blob);
  h[0] = kBlobMagic; h[1] = kBlobVersion; h[2] = q->P; h[3] = q->G; h[4] = q->B; h[5] = q->steps_done;
  h[6] = q->cache_valid ? 1 : 0; h[7] = 0;
  memcpy(&h[8], &q->tau, 4); h[9] = 0;
  CU_TRY(&c->err, cudaMemcpyAsync(h + kBlobHeaderWords, c->tokens + (size_t)r * c->a.max_seq, (size_t)q->S * 4, cudaMemcpyDeviceToHost, c->st));
  CU_TRY(&c->err, cudaMemcpyAsync(h + kBlobHeaderWords + q->S, c->conf_state + (size_t)r * c->a.max_seq, (size_t)q->S * 4, cudaMemcpyDeviceToHost, c->st));
  CU_TRY(&c->err, cudaStreamSynchronize(c->st));
  return need;
}

extern "C" int dlm_request_import(dlm_ctx* c, const void* blob, int64_t bytes, int32_t* out_req) {
  DevGuard dev_guard(c);
  if (!c) return DLM_E_ARG;
  const int32_t* h = static_cast<const int32_t*>(blob);
  if (!blob || !out_req || bytes < (int64_t)kBlobHeaderWords * 4 || h[0] != kBlobMagic || h[1] != kBlobVersion) {
    set_err(&c->err, "dlm_request_import: not a version-%d request blob", kBlobVersion);
    return DLM_E_ARG;
  }
  const int P = h[2], G = h[3], B = h[4], steps = h[5];
  if (P < 0 || G <= 0 || B <= 0 || steps < 0 || bytes != (int64_t)kBlobHeaderWords * 4 + ((int64_t)P + G) * 8) {
    set_err(&c->err, "dlm_request_import: header (P=%d G=%d B=%d) does not match %lld bytes", P, G, B, (long long)bytes);
    return DLM_E_ARG;
  }
  const int S = P + G;
  float tau; memcpy(&tau, &h[8], 4);
  const int32_t* tok = h + kBlobHeaderWords;
  for (int i = 0; i < S; ++i)
    if (tok[i] < 0 || tok[i] >= c->a.vocab || (i < P && tok[i] == c->a.mask_id)) { set_err(&c->err, "dlm_request_import: bad id at %d", i); return DLM_E_ARG; }
  int32_t slot = -1;
  int rc = dlm_request_add(c, tok, P, G, B, tau, &slot);
  if (rc != DLM_OK) return rc;
  rc = dlm_request_set_tokens(c, slot, tok, S, 0);
  if (rc == DLM_OK) {
    cudaError_t e = cudaMemcpyAsync(c->conf_state + (size_t)slot * c->a.max_seq, tok + S, (size_t)S * 4, cudaMemcpyHostToDevice, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) { set_err(&c->err, "dlm_request_import: %s", cudaGetErrorString(e)); rc = DLM_E_CUDA; }
  }
  if (rc != DLM_OK) { dlm_request_remove(c, slot); return rc; }
  c->reqs[slot].steps_done = steps;
  c->reqs[slot].cache_valid = false;
  *out_req = slot;
  return DLM_OK;
}

extern "C" int dlm_request_info(dlm_ctx* c, int32_t r, int32_t* cur_block, int32_t* cache_valid, int32_t* n_masked) {
  Req* q = get_req(c, r);
  if (!q) { if (c) set_err(&c->err, "dlm_request_info: bad request %d", r); return DLM_E_ARG; }
  if (cur_block) *cur_block = q->cur_block;
  if (cache_valid) *cache_valid = q->cache_valid;
  if (n_masked) *n_masked = q->n_masked;
  return DLM_OK;
}

// ------------------------------------------------------------------------------------------------
// One step
// ------------------------------------------------------------------------------------------------
// kind: 0 = cached step, 1 = refresh step, 2 = mixed (each request takes the kind that is due, P:616-618 token-count batching)
static int build_batch(dlm_ctx* c, const dlm_batch* b, const float* thr_override, int kind, HostBatch& hb) {
  const dlm_arch& a = c->a;
  if (!b || b->n <= 0 || !b->req) { set_err(&c->err, "step: empty batch"); return DLM_E_ARG; }
  if (b->n > a.max_requests) { set_err(&c->err, "step: batch of %d exceeds max_requests", b->n); return DLM_E_CAPACITY; }
  hb = HostBatch();
  hb.n = b->n;
  std::vector<char> seen(c->reqs.size(), 0);
  for (int i = 0; i < b->n; ++i) {
    int r = b->req[i];
    Req* q = get_req(c, r);
    if (!q) { set_err(&c->err, "step: unknown request %d", r); return DLM_E_ARG; }
    if (seen[r]) { set_err(&c->err, "step: request %d appears twice in the batch", r); return DLM_E_ARG; }
    seen[r] = 1;
    const bool done = q->cur_block >= q->G / q->B;
    const bool refresh = kind == 1 || (kind == 2 && !done && !q->cache_valid);
    if (!refresh && !done && !q->cache_valid) {
      set_err(&c->err, "dlm_cached_step: request %d has no valid K/V cache (a refresh step is due)", r);
      return DLM_E_STATE;
    }
    const int blk_lo = q->P + std::min(q->cur_block, q->G / q->B - 1) * q->B;
    int qlen, qpos0;
    if (refresh) { qlen = q->S; qpos0 = 0; }
    else { qlen = done ? 0 : q->B; qpos0 = blk_lo; }
    float tau = thr_override ? thr_override[i] : (b->threshold ? b->threshold[i] : q->tau);
    hb.slot.push_back(r); hb.q_off.push_back(hb.T); hb.q_len.push_back(qlen); hb.q_pos0.push_back(qpos0);
    hb.kv_len.push_back(q->S); hb.blk_lo.push_back(blk_lo); hb.blk_len.push_back(done ? 0 : q->B);
    hb.gen_lo.push_back(q->P); hb.gen_len.push_back(q->G);
    hb.row_off.push_back(hb.R); hb.tau.push_back(tau); hb.refresh.push_back(refresh ? 1 : 0);
    for (int t = 0; t < qlen; ++t) hb.tok_bi.push_back(i);
    hb.T += qlen; hb.R += done ? 0 : q->B;
    hb.max_q = std::max(hb.max_q, qlen); hb.max_kv = std::max(hb.max_kv, q->S);
    if (qlen > 0) hb.min_q = std::min(hb.min_q, qlen);
  }
  if (hb.T > c->Tmax) { set_err(&c->err, "step: %d tokens exceed max_batch_tokens=%d", hb.T, c->Tmax); return DLM_E_CAPACITY; }
  // work order of the persistent attention kernels: longest K/V first (requests that compute nothing last); results do not
  // depend on it, every item is computed independently
  hb.order.resize(hb.n);
  for (int i = 0; i < hb.n; ++i) hb.order[i] = i;
  const int rq = c->a.n_heads / c->a.n_kv_heads;
  auto big = [&](int x) { return hb.q_len[x] * rq > 64; };     // kTtNQ: above it the row-major attention kernel takes the request
  std::stable_sort(hb.order.begin(), hb.order.end(), [&](int x, int y) {
    if (big(x) != big(y)) return big(x);
    const long long wx = hb.q_len[x] > 0 ? hb.kv_len[x] : -1, wy = hb.q_len[y] > 0 ? hb.kv_len[y] : -1;
    return wx > wy;
  });
  hb.n_big = 0;
  for (int i = 0; i < hb.n; ++i) hb.n_big += big(i) ? 1 : 0;
  hb.qt_off.assign(hb.n + 1, 0);                               // 128-row query tiles per request, prefix sums over `order`
  for (int i = 0; i < hb.n; ++i) hb.qt_off[i + 1] = hb.qt_off[i] + (hb.q_len[hb.order[i]] * rq + 127) / 128;
  hb.qt_big = hb.qt_off[hb.n_big]; hb.qt_total = hb.qt_off[hb.n];
  return DLM_OK;
}

// Descriptor layout in desc_host / desc_dev (ints): slot, q_off, q_len, q_pos0, kv_len, blk_lo, blk_len, row_off, tau, gen_lo,
// gen_len, order [n each], qt_off [n + 1], then tok_bi [T].  Offsets depend on (n, T) only, so a captured graph of the same batch shape can be replayed.
static size_t fill_desc_host(dlm_ctx* c, const HostBatch& hb) {
  int* h = c->desc_host;
  const size_t n = hb.n;
  const std::vector<int>* v[8] = {&hb.slot, &hb.q_off, &hb.q_len, &hb.q_pos0, &hb.kv_len, &hb.blk_lo, &hb.blk_len, &hb.row_off};
  for (int i = 0; i < 8; ++i) memcpy(h + i * n, v[i]->data(), n * 4);
  memcpy(h + 8 * n, hb.tau.data(), n * 4);
  memcpy(h + 9 * n, hb.gen_lo.data(), n * 4);
  memcpy(h + 10 * n, hb.gen_len.data(), n * 4);
  memcpy(h + 11 * n, hb.order.data(), n * 4);
  memcpy(h + 12 * n, hb.qt_off.data(), (n + 1) * 4);
  memcpy(h + 13 * n + 1, hb.tok_bi.data(), hb.tok_bi.size() * 4);
  return 13 * n + 1 + hb.tok_bi.size();
}
static BatchDesc make_desc(dlm_ctx* c, const HostBatch& hb) {
  BatchDesc d;
  const size_t n = hb.n;
  const int* b = c->desc_dev;
  d.n = hb.n; d.T = hb.T; d.R = hb.R; d.max_q_len = hb.max_q; d.max_kv_len = hb.max_kv; d.min_q_len = std::min(hb.min_q, hb.max_q); d.n_big = hb.n_big; d.qt_big = hb.qt_big; d.qt_total = hb.qt_total;
  d.slot = b; d.q_off = b + n; d.q_len = b + 2 * n; d.q_pos0 = b + 3 * n; d.kv_len = b + 4 * n; d.blk_lo = b + 5 * n;
  d.blk_len = b + 6 * n; d.row_off = b + 7 * n; d.tau = (const float*)(b + 8 * n); d.order = b + 11 * n; d.qt_off = b + 12 * n; d.tok_bi = b + 13 * n + 1;
  return d;
}

static void dump_stage(dlm_ctx* c, int layer, int which, const void* src, size_t row_bytes, int rows) {
  if (!c->opt_dump || rows <= 0) return;
  auto key = std::make_pair(layer, which);
  void*& p = c->dump[key];
  if (p) cudaFree(p);
  p = nullptr;
  if (cudaMalloc(&p, row_bytes * rows) != cudaSuccess) { p = nullptr; return; }
  cudaMemcpyAsync(p, src, row_bytes * rows, cudaMemcpyDeviceToDevice, c->st);
}

// Large-M projection of the bf16 path: the CTA-pair persistent kernel above 128 tokens, the single-CTA kernel below.
// slice_rows_cap > 0 (EPI_F32 into a buffer of that many rows): split-K allowed, *n_slices tells the consumer how
// many [M, ldc] slices to sum.
static int gemm_big(dlm_ctx* c, const void* A, long long a_rows_cap, const void* W, long long w_rows, int M, int N, int K, int epi,
                    float* out_f32, bf16* out_bf16, long long ldc, int up_row0, bool pdl, long long slice_rows_cap = 0, int* n_slices = nullptr) {
  if (n_slices) *n_slices = 1;
  if (M > 128 && c->opt_pair) {
    GemmPairParams p = {};
    p.out_f32 = out_f32; p.out_bf16 = out_bf16; p.ldc = ldc; p.up_row0 = up_row0; p.tr = c->tslot();
    c->paths |= DLM_PATH_GEMM_PAIR;
    const int max_splits = (n_slices && slice_rows_cap > 0) ? (int)std::min<long long>(4, slice_rows_cap / M) : 1;
    return gemm_pair(c->tmaps, &c->err, A, a_rows_cap, W, w_rows, M, N, K, epi, 0, p, c->st, pdl, max_splits, n_slices);
  }
  GemmTcParams p = {};
  p.out_f32 = out_f32; p.out_bf16 = out_bf16; p.ldc = ldc; p.up_row0 = up_row0; p.tr = c->tslot();
  c->paths |= DLM_PATH_GEMM_TC;
  return gemm_tc(c->tmaps, &c->err, A, a_rows_cap, W, w_rows, M, N, K, epi, 0, p, c->st, pdl);
}

// O / down projection of the large-M path: residual add fused in the epilogue, or -- when split-K pays -- fp32 slices
// in part_x that the next RMSNorm folds into the residual stream (*pend = slices pending).
static int gemm_big_resid(dlm_ctx* c, const void* A, const void* W, int M, int N, int K, bool pdl, int* pend) {
  *pend = 0;
  if (M > 128 && c->opt_pair && c->part_x && c->part_rows >= 2LL * M) {
    int bn = 0, sp = 1;
    plan_pair(M, N, K, EPI_F32, (int)std::min<long long>(4, c->part_rows / M), &bn, &sp);
    if (sp > 1) {
      int ns = 1;
      int rc = gemm_big(c, A, c->Tmax, W, N, M, N, K, EPI_F32, c->part_x, nullptr, N, 0, pdl, c->part_rows, &ns);
      *pend = ns;
      return rc;
    }
  }
  return gemm_big(c, A, c->Tmax, W, N, M, N, K, EPI_RESID, c->x, nullptr, N, 0, pdl);
}

// Whole-stack persistent kernel (layer_mega.cuh): can this step take it?
// The whole-stack kernel synchronises its CTAs through a grid-wide counter, so every CTA must be resident at once: it is launched
// cooperatively (the driver refuses the launch instead of letting waiting CTAs spin when the grid does not fit beside other
// work), and a device on which one CTA per SM does not fit never takes this path.
static bool mega_configure(int tpad, int stages) {
  static int state[kMaxDevices] = {};           // 0 unknown, 1 usable, -1 not
  if (!state[g_dev]) {
    int coop = 0, nb = 0;
    bool ok = cudaFuncSetAttribute(layer_mega_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) == cudaSuccess &&
              cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, g_dev) == cudaSuccess && coop &&
              cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, layer_mega_kernel, kMgThreads, (size_t)mega_smem_bytes(tpad, stages)) == cudaSuccess && nb >= 1;
    if (!ok) cudaGetLastError();
    state[g_dev] = ok ? 1 : -1;
  }
  return state[g_dev] > 0;
}

static bool mega_ok(const dlm_ctx* c, const BatchDesc& bd) {
  const dlm_arch& a = c->a;
  if (!c->bf16_model || c->opt_simple || !c->opt_mega || !c->opt_skinny || !c->w_tiled || !c->mega_wmaps) return false;
  if (bd.T <= 0 || bd.T > kMgMaxTpad || a.head_dim != 128 || a.kv_page_tokens != 64) return false;
  const int r = a.n_heads / a.n_kv_heads, NQKV = nqkv(a);
  if (bd.max_q_len * r > 64) return false;                                   // one attention unit = <= 64 stacked rows
  if (a.d_model % 128 || a.d_model > 4096 || (a.n_heads * a.head_dim) % 64 || NQKV % 128 || a.d_ffn % 64) return false;
  if (NQKV / 128 > kMgMaxTiles || a.d_ffn / 64 > kMgMaxTiles || a.d_model / 128 > kMgMaxTiles) return false;
  // a tile is cut into at most ceil(kbt * G / U) + 1 runs: no more than the kernel's fixed-size slice sums take
  const int G = g_num_sms, d = a.d_model, F = a.d_ffn, HQ = a.n_heads * a.head_dim;
  auto max_seg = [&](long long n_tiles, long long kbt) { const long long U = n_tiles * kbt; return (int)((kbt * G + U - 1) / U) + 1; };
  if (max_seg(NQKV / 128, d / 64) > kMgMaxSegQkv || max_seg(F / 64, d / 64) > kMgMaxSegGu || max_seg(d / 128, HQ / 64) > kMgMaxSeg || max_seg(d / 128, F / 64) > kMgMaxSeg) return false;
  // what mega_launch would refuse: the shared-memory plan and the slice buffers -- such a step takes the per-stage kernels instead
  const int tpad = (bd.T + 31) / 32 * 32, stages = mega_stages(tpad);
  if (stages < 2 || stages * (tpad * 128) + kMgScratchOwn < kMgAttnBytes) return false;
  const long long need_a = std::max<long long>((long long)max_seg(NQKV / 128, d / 64) * bd.T * NQKV, (long long)max_seg(F / 64, d / 64) * bd.T * 2 * F);
  const long long need_x = (long long)std::max(max_seg(d / 128, HQ / 64), max_seg(d / 128, F / 64)) * bd.T * d;
  if (need_a > c->qkv_rows * (long long)NQKV || need_x > c->part_rows * (long long)d) return false;
  return mega_configure(tpad, stages);
}

static int mega_launch(dlm_ctx* c, const BatchDesc& bd, int layer0, int n_layers, bool dump, bool pdl) {
  const dlm_arch& a = c->a;
  const int d = a.d_model, F = a.d_ffn, HQ = a.n_heads * a.head_dim, NQKV = nqkv(a);
  MegaParams p = {};
  p.layer0 = layer0; p.n_layers = n_layers; p.T = bd.T; p.tpad = (bd.T + 31) / 32 * 32;
  p.stages = mega_stages(p.tpad);
  p.d = d; p.HQ = HQ; p.NQKV = NQKV; p.F = F; p.Fp = (int)pad_to(F, 128); p.n_heads = a.n_heads;
  p.eps = a.rms_eps; p.scale_log2 = (1.f / sqrtf((float)a.head_dim)) * 1.4426950408889634f;
  p.wmaps = c->mega_wmaps;
  p.x = c->x; p.u = (bf16*)c->u; p.u2 = (bf16*)c->u2; p.attn = (bf16*)c->attn; p.act = (bf16*)c->act;
  p.q = (bf16*)c->q; p.xmid_dump = dump ? c->tmp : nullptr;
  p.part_a = c->qkv; p.part_x = c->part_x;
  p.rope_cos = c->rope_cos; p.rope_sin = c->rope_sin; p.kv_store = (bf16*)c->kv_store; p.page_table = c->page_table;
  p.b = bd; p.g = c->kg; p.bar = c->mega_bar; p.tile_cnt = c->mega_bar + 64;
  p.phase_ts = c->opt_mega_ts ? c->mega_ts : nullptr;
  // attention phase: K/V ranges per (request, KV head) so that about one unit lands on every SM; merged by the last to arrive
  {
    const int units = bd.n * a.n_kv_heads, kv_tiles = (bd.max_kv_len + 63) / 64;
    int nsp = std::max(1, std::min(std::min(kMgMaxAttSplits, g_num_sms / std::max(1, units)), kv_tiles));
    while (nsp > 1 && (size_t)nsp * bd.T * a.n_heads * (128 + 2) * 4 > c->attn_ws_bytes) --nsp;
    p.att_splits = nsp;
    p.ws_o = c->attn_ws; p.ws_ml = c->attn_ws + (size_t)nsp * bd.T * a.n_heads * 128;
  }
  p.tr = c->tslot();
  if (p.stages < 2 || p.stages * (p.tpad * 128) + kMgScratchOwn < kMgAttnBytes) { set_err(&c->err, "layer kernel: shared-memory plan does not fit (tpad %d)", p.tpad); return DLM_E_ARG; }
  // slice capacity: a tile is cut into at most ceil(kbt * G / U) + 1 runs
  const int G = g_num_sms;
  auto max_seg = [&](long long n_tiles, long long kbt) { const long long U = n_tiles * kbt; return (int)((kbt * G + U - 1) / U) + 1; };
  if (max_seg(NQKV / 128, d / 64) > kMgMaxSegQkv || max_seg(F / 64, d / 64) > kMgMaxSegGu || max_seg(d / 128, HQ / 64) > kMgMaxSeg || max_seg(d / 128, F / 64) > kMgMaxSeg) {
    set_err(&c->err, "layer kernel: a tile would be cut into more slices than the kernel sums"); return DLM_E_ARG;
  }
  const long long need_a = std::max<long long>((long long)max_seg(NQKV / 128, d / 64) * bd.T * NQKV, (long long)max_seg(F / 64, d / 64) * bd.T * 2 * F);
  const long long need_x = (long long)std::max(max_seg(d / 128, HQ / 64), max_seg(d / 128, F / 64)) * bd.T * d;
  if (need_a > c->qkv_rows * (long long)NQKV || need_x > c->part_rows * (long long)d) { set_err(&c->err, "layer kernel: slice buffers too small"); return DLM_E_CAPACITY; }
  const CUtensorMap* mu = c->tmaps.get(c->u, c->Tmax, d, p.tpad);
  const CUtensorMap* mu2 = c->tmaps.get(c->u2, kMgMaxTpad, d, p.tpad);
  const CUtensorMap* mat = c->tmaps.get(c->attn, c->Tmax, HQ, p.tpad);
  const CUtensorMap* mac = c->tmaps.get(c->act, c->Tmax, F, p.tpad);
  if (!mu || !mu2 || !mat || !mac) { set_err(&c->err, "cuTensorMapEncodeTiled failed (layer kernel activations)"); return DLM_E_CUDA; }
  if (!mega_configure(p.tpad, p.stages)) { set_err(&c->err, "layer kernel: one CTA per SM does not fit on this device (or no cooperative launch)"); return DLM_E_CUDA; }
  CU_TRY(&c->err, cudaMemsetAsync(c->mega_bar, 0, 4096, c->st));
  cudaError_t e = launch_k_attr(layer_mega_kernel, dim3(G), dim3(kMgThreads), (size_t)mega_smem_bytes(p.tpad, p.stages), c->st, pdl, /*coop=*/true, *mu, *mu2, *mat, *mac, p);
  if (e != cudaSuccess) { set_err(&c->err, "layer kernel launch: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
  c->paths |= DLM_PATH_LAYER_KERNEL;
  return DLM_OK;
}

template <typename TE>
static int forward(dlm_ctx* c, const BatchDesc& bd, bool dry_run) {
  const dlm_arch& a = c->a;
  cudaStream_t st = c->st;
  const int T = bd.T, d = a.d_model, F = a.d_ffn, V = a.vocab, HQ = a.n_heads * a.head_dim, NQKV = nqkv(a);
  const bool tc = c->bf16_model && !c->opt_simple;
  const bool skinny = tc && c->opt_skinny && T <= kSkMaxTokens;      // weight-streaming regime (cached steps of small batches)
  // a3 + a4 in one kernel above 128 tokens: the QKV epilogue rotates, rounds and writes Q and the K/V pages itself
  const bool fuse_rope = tc && !skinny && T > 128 && c->opt_pair && c->opt_fuse_rope && a.head_dim == 128 && NQKV % 256 == 0;
  const bool pdl = c->opt_pdl && !c->kprof.on;                        // event pairs between kernels would serialise anyway
  const float scale = 1.f / sqrtf((float)a.head_dim);
  std::string* err = &c->err;
  if (!tc) {   // scratch of the plain path, allocated on first use
    c->paths |= DLM_PATH_GEMM_PLAIN;
    if (!c->tmp) CU_TRY(err, cudaMalloc(&c->tmp, (size_t)c->Tmax * std::max(d, 2 * F) * 4));
    if (!c->logits) CU_TRY(err, cudaMalloc(&c->logits, (size_t)c->Rmax * V * 4));
  }
  int pend = 0;                                   // split-K slices of x waiting in part_x (folded into the next norm)
  const long long pstride = (long long)T * d;
  // in debug-dump mode x is completed right after each projection so that every dumped tensor is whole
  auto flush_partials = [&]() {
    if (pend > 0 && c->opt_dump) {
      KScope ks(c, DLM_K_RMSNORM);
      launch_k(add_partials_kernel, dim3((unsigned)((pstride + 255) / 256)), dim3(256), 0, st, pdl, c->x, (const float*)c->part_x, pend, pstride, pstride, c->tslot());
      pend = 0;
    }
  };
  if (T > 0) {
    KScope ks(c, DLM_K_EMBED);                    // first kernel of the step: plain launch (stream order vs. the previous step)
    launch_k(embed_kernel<TE>, dim3(T), dim3(256), 0, st, false, c->x, (const TE*)c->E, (const int*)c->tokens, a.max_seq, bd, d, c->tslot());
  }
  const bool mega = tc && T > 0 && mega_ok(c, bd);
  if (mega) {
    // every layer in ONE persistent launch; in debug-dump mode the same kernel runs layer by layer (identical arithmetic) so
    // that each layer's stage tensors can be copied out
    KScope ks(c, DLM_K_LAYERS);
    if (!c->opt_dump) {
      int rc = mega_launch(c, bd, 0, a.n_layers, false, false);      // plain launch: its memset must not overtake the embedding kernel
      if (rc) return rc;
    } else {
      if (!c->tmp) CU_TRY(err, cudaMalloc(&c->tmp, (size_t)c->Tmax * std::max(d, 2 * F) * 4));
      for (int l = 0; l < a.n_layers; ++l) {
        dump_stage(c, l, DLM_T_X_IN, c->x, (size_t)d * 4, T);
        int rc = mega_launch(c, bd, l, 1, true, false);
        if (rc) return rc;
        dump_stage(c, l, DLM_T_NORM1, c->u, (size_t)d * sizeof(TE), T);
        dump_stage(c, l, DLM_T_Q, c->q, (size_t)HQ * sizeof(TE), T);
        dump_stage(c, l, DLM_T_ATTN, c->attn, (size_t)HQ * sizeof(TE), T);
        dump_stage(c, l, DLM_T_X_MID, c->tmp, (size_t)d * 4, T);
        dump_stage(c, l, DLM_T_NORM2, c->u2, (size_t)d * sizeof(TE), T);
        dump_stage(c, l, DLM_T_ACT, c->act, (size_t)F * sizeof(TE), T);
        dump_stage(c, l, DLM_T_X_OUT, c->x, (size_t)d * 4, T);
      }
    }
  }
  for (int l = 0; l < a.n_layers && T > 0 && !mega; ++l) {
    const LayerW& w = c->L[l];
    dump_stage(c, l, DLM_T_X_IN, c->x, (size_t)d * 4, T);
    {
      KScope ks(c, DLM_K_RMSNORM);
      launch_rmsnorm<TE>(c, (TE*)c->u, c->x, (const int*)nullptr, T, d, a.rms_eps, (const float*)c->part_x, pend, pstride, pdl);
      pend = 0;
    }
    dump_stage(c, l, DLM_T_NORM1, c->u, (size_t)d * sizeof(TE), T);
    int nq = 1;                                   // slices of the qkv buffer the RoPE kernel sums
    {
      KScope ks(c, DLM_K_GEMM_QKV);
      if (skinny) {
        SkinnyParams p = {};
        p.out_f32 = c->qkv; p.ldc = NQKV; p.tr = c->tslot();
        c->paths |= DLM_PATH_GEMM_SKINNY;
        int rc = gemm_skinny(c->tmaps, err, c->u, c->Tmax, w.wqkv, NQKV, T, NQKV, d, SK_PARTIAL, 0, p, &nq, st, pdl);
        if (rc) return rc;
      } else if (fuse_rope) {
        GemmPairParams p = {};
        p.rope.q = (bf16*)c->q; p.rope.kv_store = (bf16*)c->kv_store; p.rope.rope_cos = c->rope_cos; p.rope.rope_sin = c->rope_sin;
        p.rope.page_table = c->page_table; p.rope.b = bd; p.rope.g = c->kg; p.rope.layer = l; p.rope.n_heads = a.n_heads;
        p.tr = c->tslot();
        c->paths |= DLM_PATH_GEMM_PAIR | DLM_PATH_ROPE_FUSED;
        int rc = gemm_pair(c->tmaps, err, c->u, c->Tmax, w.wqkv, NQKV, T, NQKV, d, EPI_ROPE, 0, p, st, pdl);
        if (rc) return rc;
      } else if (tc) {
        int rc = gemm_big(c, c->u, c->Tmax, w.wqkv, NQKV, T, NQKV, d, EPI_F32, c->qkv, nullptr, NQKV, 0, pdl, c->qkv_rows, &nq);
        if (rc) return rc;
      } else {
        gemm_plain<TE, TE>(c->qkv, (const TE*)c->u, (const TE*)w.wqkv, T, NQKV, d, st, pdl);
      }
    }
    if (!fuse_rope) {
      KScope ks(c, DLM_K_ROPE_KV);
      const int hpb = std::max(1, 256 / (a.head_dim / 2));       // heads per block
      launch_k(rope_kv_write_kernel<TE>, dim3(T, (a.n_heads + 2 * a.n_kv_heads + hpb - 1) / hpb), dim3(hpb * (a.head_dim / 2)), 0, st, pdl, (TE*)c->q, (TE*)c->kv_store, (const float*)c->qkv, (const float*)c->rope_cos,
               (const float*)c->rope_sin, (const int*)c->page_table, bd, c->kg, l, a.n_heads, nq, (long long)T * NQKV, c->tslot());
    }
    dump_stage(c, l, DLM_T_Q, c->q, (size_t)HQ * sizeof(TE), T);
    bool flash_done = false;
    if (tc && c->opt_flash && c->opt_tcattn) {
      KScope ks(c, DLM_K_ATTENTION);
      const size_t trace_mark = c->trace_cls.size();
      const TraceSlot tr3[3] = {c->tslot(), c->tslot(), c->tslot()};
      int rc = attn_tc_launch(c->tmaps, (bf16*)c->attn, (const bf16*)c->q, (const bf16*)c->kv_store, a.n_layers, c->page_table, bd, c->kg, l,
                              a.n_heads, scale, &c->attn_ws, &c->attn_ws_bytes, st, pdl, err, &flash_done, 0, tr3, &c->paths, c->opt_tct_min_items);
      if (rc) return rc;
      if (!flash_done) c->trace_cls.resize(trace_mark);      // nothing launched: give back the records taken (none once the table is full)
    }
    if (tc && c->opt_flash && !flash_done) {
      KScope ks(c, DLM_K_ATTENTION);
      const size_t trace_mark = c->trace_cls.size();
      const TraceSlot t0 = c->tslot(), t1 = c->tslot();
      int rc = attn_flash_launch((bf16*)c->attn, (const bf16*)c->q, (const bf16*)c->kv_store, c->page_table, bd, c->kg, l,
                                 a.n_heads, scale, &c->attn_ws, &c->attn_ws_bytes, g_num_sms, st, pdl, err, &flash_done, t0, t1);
      if (rc) return rc;
      if (flash_done) c->paths |= DLM_PATH_ATTN_FLASH;
      else c->trace_cls.resize(trace_mark);
    }
    if (!flash_done) {
      KScope ks(c, DLM_K_ATTENTION);
      c->paths |= DLM_PATH_ATTN_PLAIN;
      launch_k(attention_plain_kernel<TE>, dim3(T, a.n_heads), dim3(128), (size_t)bd.max_kv_len * 4, st, pdl, (TE*)c->attn, (const TE*)c->q,
               (const TE*)c->kv_store, (const int*)c->page_table, bd, c->kg, l, a.n_heads, scale);
    }
    dump_stage(c, l, DLM_T_ATTN, c->attn, (size_t)HQ * sizeof(TE), T);
    {
      KScope ks(c, DLM_K_GEMM_O);
      if (skinny) {
        SkinnyParams p = {};
        p.out_f32 = c->part_x; p.ldc = d; p.tr = c->tslot();
        int rc = gemm_skinny(c->tmaps, err, c->attn, c->Tmax, w.wo, d, T, d, HQ, SK_PARTIAL, 0, p, &pend, st, pdl);
        if (rc) return rc;
      } else if (tc) {
        int rc = gemm_big_resid(c, c->attn, w.wo, T, d, HQ, pdl, &pend);
        if (rc) return rc;
      } else {
        gemm_plain<TE, TE>(c->tmp, (const TE*)c->attn, (const TE*)w.wo, T, d, HQ, st, pdl);
        launch_k(add_residual_kernel, dim3((unsigned)(((long long)T * d + 255) / 256)), dim3(256), 0, st, pdl, c->x, (const float*)c->tmp, (long long)T * d);
      }
    }
    flush_partials();
    dump_stage(c, l, DLM_T_X_MID, c->x, (size_t)d * 4, T);
    {
      KScope ks(c, DLM_K_RMSNORM);
      launch_rmsnorm<TE>(c, (TE*)c->u, c->x, (const int*)nullptr, T, d, a.rms_eps, (const float*)c->part_x, pend, pstride, pdl);
      pend = 0;
    }
    dump_stage(c, l, DLM_T_NORM2, c->u, (size_t)d * sizeof(TE), T);
    {
      KScope ks(c, DLM_K_GEMM_GATEUP);
      if (skinny) {
        SkinnyParams p = {};
        p.out_bf16 = (bf16*)c->act; p.ldc = F; p.up_row0 = F; p.tr = c->tslot();
        int rc = gemm_skinny(c->tmaps, err, c->u, c->Tmax, w.wgu, 2LL * F, T, F, d, SK_SWIGLU, 0, p, nullptr, st, pdl);
        if (rc) return rc;
      } else if (tc) {
        int rc = gemm_big(c, c->u, c->Tmax, w.wgu, 2LL * F, T, F, d, EPI_SWIGLU, nullptr, (bf16*)c->act, F, F, pdl);
        if (rc) return rc;
      } else {
        gemm_plain<TE, TE>(c->tmp, (const TE*)c->u, (const TE*)w.wgu, T, 2 * F, d, st, pdl);
        launch_k(swiglu_kernel<TE>, dim3((unsigned)(((long long)T * F + 255) / 256)), dim3(256), 0, st, pdl, (TE*)c->act, (const float*)c->tmp, T, F);
      }
    }
    dump_stage(c, l, DLM_T_ACT, c->act, (size_t)F * sizeof(TE), T);
    {
      KScope ks(c, DLM_K_GEMM_DOWN);
      if (skinny) {
        SkinnyParams p = {};
        p.out_f32 = c->part_x; p.ldc = d; p.tr = c->tslot();
        int rc = gemm_skinny(c->tmaps, err, c->act, c->Tmax, w.wd, d, T, d, F, SK_PARTIAL, 0, p, &pend, st, pdl);
        if (rc) return rc;
      } else if (tc) {
        int rc = gemm_big_resid(c, c->act, w.wd, T, d, F, pdl, &pend);
        if (rc) return rc;
      } else {
        gemm_plain<TE, TE>(c->tmp, (const TE*)c->act, (const TE*)w.wd, T, d, F, st, pdl);
        launch_k(add_residual_kernel, dim3((unsigned)(((long long)T * d + 255) / 256)), dim3(256), 0, st, pdl, c->x, (const float*)c->tmp, (long long)T * d);
      }
    }
    flush_partials();
    dump_stage(c, l, DLM_T_X_OUT, c->x, (size_t)d * 4, T);
  }
  // ---- head: a10 final norm on the block rows, a11 LM head statistics, a12+a13 combine + unmask ----
  const int R = bd.R;
  StepOut so;
  char* ob = c->out_dev;
  so.n_committed = (int*)ob; ob += (size_t)a.max_requests * 4;
  const size_t rb = (size_t)c->Rmax * 4;
  so.pos = (int*)ob; ob += rb; so.tok = (int*)ob; ob += rb; so.conf = (float*)ob; ob += rb;
  so.row_lse = (float*)ob; ob += rb; so.row_conf = (float*)ob; ob += rb; so.row_tok = (int*)ob;
  int n_tiles = 1;
  if (R > 0) {
    {
      KScope ks(c, DLM_K_RMSNORM);
      launch_k(build_row_src_kernel, dim3(bd.n), dim3(64), 0, st, pdl, c->row_src, bd, c->tslot());
      launch_rmsnorm<TE>(c, (TE*)c->hf, c->x, (const int*)c->row_src, R, d, a.rms_eps, (const float*)c->part_x, pend, pstride, pdl);
      pend = 0;
    }
    dump_stage(c, 0, DLM_T_FINAL_NORM, c->hf, (size_t)d * sizeof(TE), R);
    KScope ks(c, DLM_K_LMHEAD);
    if (tc && R > 128 && c->opt_pair) {          // compute-bound head: CTA-pair kernel, 256-wide vocabulary tiles
      n_tiles = (V + 255) / 256;
      GemmPairParams p = {};
      p.part = c->part; p.n_tiles = n_tiles; p.mask_id = a.mask_id; p.scale = a.logit_scale; p.tr = c->tslot();
      c->paths |= DLM_PATH_GEMM_PAIR;
      int rc = gemm_pair(c->tmaps, err, c->hf, std::max(c->Rmax, 128), c->Wlm, V, R, V, d, EPI_LMHEAD, 256, p, st, pdl);
      if (rc) return rc;
    } else if (tc) {
      n_tiles = c->n_tiles;
      GemmTcParams p = {};
      p.part = c->part; p.n_tiles = n_tiles; p.mask_id = a.mask_id; p.scale = a.logit_scale; p.tr = c->tslot();
      c->paths |= DLM_PATH_GEMM_TC;
      int rc = gemm_tc(c->tmaps, err, c->hf, std::max(c->Rmax, 128), c->Wlm, V, R, V, d, EPI_LMHEAD, 128, p, st, pdl);
      if (rc) return rc;
    } else {
      gemm_plain<TE, TE>(c->logits, (const TE*)c->hf, (const TE*)c->Wlm, R, V, d, st, pdl);
      launch_k(row_stats_plain_kernel, dim3(R), dim3(256), 0, st, pdl, c->part, (const float*)c->logits, V, a.mask_id, a.logit_scale);
    }
  }
  {
    KScope ks(c, DLM_K_COMBINE_UNMASK);
    launch_k(combine_unmask_kernel, dim3(bd.n), dim3(1024), 0, st, pdl, so, (const RowPartial*)c->part, n_tiles, c->tokens, a.max_seq, a.max_block, a.mask_id, bd,
             dry_run ? 1 : 0, c->tslot());
    if (c->want_feat) {
      float* feats = (float*)(c->out_dev + (size_t)a.max_requests * 4 + (size_t)c->Rmax * 4 * 6);
      const int* gl = c->desc_dev + 9 * (size_t)bd.n;
      launch_k(conf_features_kernel, dim3(bd.n), dim3(1024), 0, st, pdl, feats, c->conf_state, (const int*)c->tokens, a.max_seq, a.max_block, a.mask_id, so, bd,
               gl, gl + bd.n, dry_run ? 1 : 0, c->tslot());
    }
  }
  CU_TRY(err, cudaGetLastError());
  return DLM_OK;
}

// One step's device work = [descriptor H2D] [kernels between ev0 and ev1] [result D2H].  With DLM_OPT_CUDA_GRAPH the
// whole sequence of a batch shape seen before is replayed from a captured graph (one launch per step).
static int enqueue_step(dlm_ctx* c, const HostBatch& hb, bool dry, size_t desc_ints, bool capturing) {
  std::string* err = &c->err;
  CU_TRY(err, cudaMemcpyAsync(c->desc_dev, c->desc_host, desc_ints * 4, cudaMemcpyHostToDevice, c->st));
  c->paths = 0;
  c->trace_cls.clear();
  if (c->opt_trace) CU_TRY(err, cudaMemsetAsync(c->trace_dev, 0xFF, (size_t)kMaxTraceSlots * 3 * 8, c->st));   // all three words are minima
  BatchDesc bd = make_desc(c, hb);
  if (capturing) CU_TRY(err, cudaEventRecordWithFlags(c->ev0, c->st, cudaEventRecordExternal));
  else CU_TRY(err, cudaEventRecord(c->ev0, c->st));        // device time of the step: first kernel .. last kernel
  int rc = c->bf16_model ? forward<bf16>(c, bd, dry) : forward<float>(c, bd, dry);
  if (rc) return rc;
  if (capturing) CU_TRY(err, cudaEventRecordWithFlags(c->ev1, c->st, cudaEventRecordExternal));
  else CU_TRY(err, cudaEventRecord(c->ev1, c->st));
  CU_TRY(err, cudaMemcpyAsync(c->out_host, c->out_dev, c->out_bytes, cudaMemcpyDeviceToHost, c->st));
  return DLM_OK;
}

static int run_step(dlm_ctx* c, const dlm_batch* b, const float* thr_override, dlm_result* res, int kind) {
  if (!c) return DLM_E_ARG;
  DevGuard dev_guard(c);
  if (!res || !res->n_committed || !res->pos || !res->tok || !res->conf) { set_err(&c->err, "step: result buffers missing"); return DLM_E_ARG; }
  HostBatch hb;
  int rc = build_batch(c, b, thr_override, kind, hb);
  if (rc) return rc;
  const dlm_arch& a = c->a;
  const bool dry = (b->flags & DLM_DRY_RUN) != 0;
  if (res->capacity < hb.R) { set_err(&c->err, "step: result capacity %d < %d block rows", res->capacity, hb.R); return DLM_E_CAPACITY; }
  if (res->features)
    for (int i = 0; i < hb.n; ++i)
      if (c->reqs[hb.slot[i]].G > kFeatMaxGen) {
        set_err(&c->err, "step: the Step Predictor features support at most %d output positions per request (request %d has %d)", kFeatMaxGen, hb.slot[i], c->reqs[hb.slot[i]].G);
        return DLM_E_CAPACITY;
      }
  std::string* err = &c->err;
  const size_t desc_ints = fill_desc_host(c, hb);
  c->want_feat = res->features != nullptr;
  const bool use_graph = c->opt_graph && !c->kprof.on && !c->opt_dump;
  bool launched = false;
  if (use_graph) {
    GraphKey key = std::make_tuple(kind, dry ? 1 : 0, hb.n, hb.T, hb.R, hb.max_q, hb.max_kv, c->opt_mask() | (c->want_feat ? 1 << 16 : 0) | (std::min(hb.min_q, 255) << 20), hb.n_big, hb.qt_big, hb.qt_total);
    GraphEntry& g = c->graphs[key];
    g.used = ++c->graph_clock;
    if (g.seen == 1) {                         // second sighting of this batch shape: capture it
      const long long l0 = g_launches;
      cudaGraph_t graph = nullptr;
      if (cudaStreamBeginCapture(c->st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        rc = enqueue_step(c, hb, dry, desc_ints, true);
        cudaError_t e = cudaStreamEndCapture(c->st, &graph);
        if (rc == DLM_OK && e == cudaSuccess && graph && cudaGraphInstantiate(&g.exec, graph, 0) == cudaSuccess) {
          g.launches = g_launches - l0;
          g.paths = c->paths; g.trace_cls = c->trace_cls;
          g.seen = 2;
        } else {
          g.seen = 3;                            // capture not possible for this shape: stay on eager launches
          cudaGetLastError();
        }
        if (graph) cudaGraphDestroy(graph);
        g_launches = l0;
        if (rc) return rc;
      } else { g.seen = 3; cudaGetLastError(); }
    }
    if (g.seen == 2) {
      CU_TRY(err, cudaGraphLaunch(g.exec, c->st));
      g_launches += g.launches;
      c->paths = g.paths | DLM_PATH_GRAPH_REPLAY; c->trace_cls = g.trace_cls;
      launched = true;
    } else if (g.seen == 0) {
      g.seen = 1;
    }
    // bounded cache: a serving loop with drifting ragged shapes must not grow host / device memory without limit.  The
    // least recently used entry goes (its executable graph is destroyed; the shape is captured again if it comes back).
    while (c->graphs.size() > kMaxGraphs) {
      auto victim = c->graphs.end();
      for (auto it = c->graphs.begin(); it != c->graphs.end(); ++it)
        if (&it->second != &g && (victim == c->graphs.end() || it->second.used < victim->second.used)) victim = it;
      if (victim == c->graphs.end()) break;
      if (victim->second.exec) {
        if (launched) cudaStreamSynchronize(c->st);          // never destroy a graph the stream may still be running
        cudaGraphExecDestroy(victim->second.exec);
      }
      c->graphs.erase(victim);
    }
  }
  if (!launched) {
    rc = enqueue_step(c, hb, dry, desc_ints, false);
    if (rc) { cudaStreamSynchronize(c->st); c->kprof.cls.clear(); c->kprof.used = 0; return rc; }
  }
  CU_TRY(err, cudaStreamSynchronize(c->st));
  cudaEventElapsedTime(&c->last_usec, c->ev0, c->ev1);
  c->last_usec *= 1000.f;
  if (c->kprof.on) c->kprof.collect();
  c->last_paths = c->paths;
  c->last_trace_cls = c->trace_cls;
  if (c->opt_trace && !c->last_trace_cls.empty()) {
    c->trace_host.resize(c->last_trace_cls.size() * 3);
    CU_TRY(err, cudaMemcpy(c->trace_host.data(), c->trace_dev, c->trace_host.size() * 8, cudaMemcpyDeviceToHost));
  } else {
    c->trace_host.clear();
  }
  // ---- unpack, update host-side request state ----
  const char* ob = c->out_host;
  const int* n_comm = (const int*)ob; ob += (size_t)a.max_requests * 4;
  const size_t rb = (size_t)c->Rmax * 4;
  const int* pos = (const int*)ob; ob += rb; const int* tok = (const int*)ob; ob += rb; const float* conf = (const float*)ob; ob += rb;
  const float* rlse = (const float*)ob; ob += rb; const float* rconf = (const float*)ob; ob += rb; const int* rtok = (const int*)ob; ob += rb;
  const float* feats = (const float*)ob;
  int total = 0;
  for (int i = 0; i < hb.n; ++i) {
    Req& q = c->reqs[hb.slot[i]];
    const int k = hb.blk_len[i] ? n_comm[i] : 0;
    res->n_committed[i] = k;
    for (int j = 0; j < k; ++j) {
      res->pos[total + j] = pos[i * a.max_block + j];
      res->tok[total + j] = tok[i * a.max_block + j];
      res->conf[total + j] = conf[i * a.max_block + j];
    }
    total += k;
    for (int j = 0; j < a.max_block; ++j) {
      const bool v = j < hb.blk_len[i];
      if (res->lse) res->lse[i * a.max_block + j] = v ? rlse[i * a.max_block + j] : 0.f;
      if (res->row_conf) res->row_conf[i * a.max_block + j] = v ? rconf[i * a.max_block + j] : 0.f;
      if (res->row_tok) res->row_tok[i * a.max_block + j] = v ? rtok[i * a.max_block + j] : -1;
    }
    if (hb.refresh[i] && hb.blk_len[i]) q.cache_valid = true;      // K/V of all positions now match the pre-step tokens
    if (!dry && hb.blk_len[i]) {
      q.n_masked -= k; q.n_masked_block -= k;
      q.steps_done++;
      if (q.n_masked_block == 0) {                            // P:109 block complete -> recompute before the next block
        q.cache_valid = false;
        q.cur_block++;
        q.n_masked_block = q.cur_block < q.G / q.B ? q.B : 0;
      }
    }
    if (res->n_masked_left) res->n_masked_left[i] = q.n_masked;
    if (res->features) {          // App. A order; the request's state AFTER this step.  A dry run reports the state the step WOULD
      float* f = res->features + (size_t)i * DLM_N_FEATURES;      // leave (progress from the reported commits) without mutating anything
      const int nb = q.G / q.B;
      int steps = q.steps_done, n_masked = q.n_masked, n_masked_block = q.n_masked_block, cur_block = q.cur_block;
      if (dry && hb.blk_len[i]) {
        steps++; n_masked -= k; n_masked_block -= k;
        if (n_masked_block == 0) { cur_block++; n_masked_block = cur_block < nb ? q.B : 0; }
      }
      const bool fin = cur_block >= nb;
      f[0] = hb.tau[i]; f[1] = (float)q.G; f[2] = (float)steps / q.G; f[3] = (float)(q.G - n_masked) / q.G;
      f[4] = fin ? 1.f : (float)cur_block / nb; f[5] = fin ? 1.f : (float)(q.B - n_masked_block) / q.B;
      for (int j = 0; j < 5; ++j) f[6 + j] = feats[i * 5 + j];
    }
  }
  res->total = total;
  c->last_batch = hb;
  c->last_refresh = kind == 1;
  return DLM_OK;
}

extern "C" int dlm_refresh_step(dlm_ctx* c, const dlm_batch* b, dlm_result* r) { return run_step(c, b, nullptr, r, 1); }
extern "C" int dlm_cached_step(dlm_ctx* c, const dlm_batch* b, const float* thr, dlm_result* r) { return run_step(c, b, thr, r, 0); }
extern "C" int dlm_mixed_step(dlm_ctx* c, const dlm_batch* b, const float* thr, dlm_result* r) { return run_step(c, b, thr, r, 2); }

// ------------------------------------------------------------------------------------------------
// Debug tensors
// ------------------------------------------------------------------------------------------------
static void to_f32_host(const void* src, float* dst, size_t n, bool is_bf16) {
  if (!is_bf16) { memcpy(dst, src, n * 4); return; }
  const uint16_t* s = (const uint16_t*)src;
  for (size_t i = 0; i < n; ++i) { uint32_t u = (uint32_t)s[i] << 16; memcpy(dst + i, &u, 4); }
}

extern "C" int64_t dlm_debug_tensor(dlm_ctx* c, int32_t r, int32_t layer, int32_t which, float* out, int64_t cap) {
  DevGuard dev_guard(c);
  Req* q = get_req(c, r);
  if (!q || !out) { if (c) set_err(&c->err, "dlm_debug_tensor: bad request %d", r); return DLM_E_ARG; }
  const dlm_arch& a = c->a;
  const int HQ = a.n_heads * a.head_dim, HKV = a.n_kv_heads * a.head_dim;
  if (which == DLM_T_KCACHE || which == DLM_T_VCACHE || which == DLM_T_K || which == DLM_T_V) {
    // K (post-RoPE) / V as they sit in the request's pages: all S positions (DLM_T_*CACHE), or the rows the last step
    // computed for this request (DLM_T_K / DLM_T_V: the step wrote exactly those slots)
    if (layer < 0 || layer >= a.n_layers) { set_err(&c->err, "dlm_debug_tensor: bad layer"); return DLM_E_ARG; }
    int p0 = 0, rows = q->S;
    if (which == DLM_T_K || which == DLM_T_V) {
      int bi = -1;
      for (int i = 0; i < c->last_batch.n; ++i) if (c->last_batch.slot[i] == r) bi = i;
      if (bi < 0) { set_err(&c->err, "dlm_debug_tensor: request %d was not in the last step", r); return DLM_E_STATE; }
      p0 = c->last_batch.q_pos0[bi]; rows = c->last_batch.q_len[bi];
    }
    const int64_t n = (int64_t)rows * HKV;
    if (cap < n) { set_err(&c->err, "dlm_debug_tensor: cap too small"); return DLM_E_CAPACITY; }
    std::vector<char> page((size_t)c->kg.page_elems() * c->esize);
    const int PT = a.kv_page_tokens, kv = (which == DLM_T_VCACHE || which == DLM_T_V);
    for (int pi = p0 / PT; pi * PT < p0 + rows; ++pi) {
      const char* src = (const char*)c->kv_store + (size_t)c->kg.offset(layer, q->pages[pi], 0, 0, 0) * c->esize;
      if (cudaMemcpy(page.data(), src, page.size(), cudaMemcpyDeviceToHost) != cudaSuccess) { set_err(&c->err, "dlm_debug_tensor: copy failed"); return DLM_E_CUDA; }
      for (int h = 0; h < a.n_kv_heads; ++h)
        for (int t = 0; t < PT; ++t) {
          const int pos = pi * PT + t;
          if (pos < p0 || pos >= p0 + rows) continue;
          size_t so = ((size_t)(kv * a.n_kv_heads + h) * PT + t) * a.head_dim;
          to_f32_host(page.data() + so * c->esize, out + ((size_t)(pos - p0) * HKV + (size_t)h * a.head_dim), a.head_dim, c->bf16_model);
        }
    }
    return n;
  }
  // stage tensors of the last step
  int bi = -1;
  for (int i = 0; i < c->last_batch.n; ++i) if (c->last_batch.slot[i] == r) bi = i;
  if (bi < 0) { set_err(&c->err, "dlm_debug_tensor: request %d was not in the last step", r); return DLM_E_STATE; }
  int width, rows, off;
  bool f32 = false;
  switch (which) {
    case DLM_T_X_IN: case DLM_T_X_MID: case DLM_T_X_OUT: width = a.d_model; f32 = true; break;
    case DLM_T_NORM1: case DLM_T_NORM2: case DLM_T_FINAL_NORM: width = a.d_model; break;
    case DLM_T_Q: case DLM_T_ATTN: width = HQ; break;
    case DLM_T_ACT: width = a.d_ffn; break;
    default: set_err(&c->err, "dlm_debug_tensor: unsupported tensor %d", which); return DLM_E_ARG;
  }
  if (which == DLM_T_FINAL_NORM) { rows = c->last_batch.blk_len[bi]; off = c->last_batch.row_off[bi]; layer = 0; }
  else { rows = c->last_batch.q_len[bi]; off = c->last_batch.q_off[bi]; }
  auto it = c->dump.find(std::make_pair(layer, which));
  if (it == c->dump.end() || !it->second) { set_err(&c->err, "dlm_debug_tensor: nothing dumped for layer %d tensor %d (set DLM_OPT_DEBUG_DUMP before the step)", layer, which); return DLM_E_STATE; }
  const int64_t n = (int64_t)rows * width;
  if (cap < n) { set_err(&c->err, "dlm_debug_tensor: cap too small"); return DLM_E_CAPACITY; }
  const size_t es = f32 ? 4 : c->esize;
  std::vector<char> buf((size_t)n * es);
  if (cudaMemcpy(buf.data(), (const char*)it->second + (size_t)off * width * es, buf.size(), cudaMemcpyDeviceToHost) != cudaSuccess) { set_err(&c->err, "dlm_debug_tensor: copy failed"); return DLM_E_CUDA; }
  to_f32_host(buf.data(), out, (size_t)n, !f32 && c->bf16_model);
  return n;
}

// ------------------------------------------------------------------------------------------------
// a15  cost table (P:123 one-time latency profiling; P:599-618 LP[tp][tokens], tp = 1)
// ------------------------------------------------------------------------------------------------
// Median of `reps` timed dry-run steps after two untimed ones (the second sighting of a shape captures its CUDA graph).
static int time_steps(dlm_ctx* c, const dlm_batch* b, dlm_result* res, int kind, int reps, float* usec) {
  std::vector<float> t;
  for (int it = 0; it < reps + 2; ++it) {
    int rc = kind == DLM_KIND_REFRESH ? dlm_refresh_step(c, b, res) : dlm_cached_step(c, b, nullptr, res);
    if (rc) return rc;
    if (it >= 2) t.push_back(c->last_usec);
  }
  std::sort(t.begin(), t.end());
  *usec = t.size() % 2 ? t[t.size() / 2] : 0.5f * (t[t.size() / 2 - 1] + t[t.size() / 2]);
  return DLM_OK;
}

extern "C" int dlm_profile_step_costs_ex(dlm_ctx* c, int32_t block_len, int32_t repeats, dlm_cost_row* rows, int32_t cap, int32_t* n_rows) {
  if (!c || !rows || !n_rows) return DLM_E_ARG;
  DevGuard dev_guard(c);
  const dlm_arch& a = c->a;
  *n_rows = 0;
  const int B = block_len;
  if (B <= 0 || B > a.max_block) { set_err(&c->err, "dlm_profile_step_costs: block length %d outside [1, max_block=%d]", B, a.max_block); return DLM_E_ARG; }
  const int reps = std::max(10, repeats);                       // median of >= 10 timed repeats
  static const int kv_lens[] = {512, 1024, 2048, 4608};
  static const int ns[] = {1, 2, 4, 8, 16, 32, 64};
  int free_slots = 0;
  for (auto& q : c->reqs) free_slots += !q.used;
  std::vector<int32_t> n_comm(a.max_requests), pos(c->Rmax), tok(c->Rmax);
  std::vector<float> conf(c->Rmax);
  dlm_result res = {};
  res.n_committed = n_comm.data(); res.pos = pos.data(); res.tok = tok.data(); res.conf = conf.data(); res.capacity = c->Rmax;
  std::vector<int32_t> ids;
  auto drop = [&]() { for (int r : ids) dlm_request_remove(c, r); ids.clear(); };
  auto add = [&](int n, int S) {                                 // n scratch requests of S positions, the last B of them one MASK block
    std::vector<int32_t> prompt(S - B);
    for (int i = 0; i < n; ++i) {
      for (int j = 0; j < S - B; ++j) prompt[j] = (int32_t)(mix64(0x5eedULL + 977ULL * i + j) % (unsigned)(a.vocab - 1));
      for (auto& t : prompt) if (t >= a.mask_id) t++;
      int32_t id;
      int rc = dlm_request_add(c, prompt.data(), S - B, B, B, 2.0f, &id);
      if (rc) { drop(); return rc; }
      ids.push_back(id);
    }
    return (int)DLM_OK;
  };
  auto fits = [&](long long n, long long S) {
    return n <= free_slots && S <= a.max_seq && S > B && n * ((S + a.kv_page_tokens - 1) / a.kv_page_tokens) <= (long long)c->free_pages.size();
  };
  // ---- cache steps: n requests x per-request K/V length (the paper's LP is indexed by cacheBlockSize x numReqs, P:615-617;
  // the K/V length is added because the cached step's attention reads all of it).  The caches are built by untimed refresh
  // steps over as many requests as max_batch_tokens admits at a time.
  for (int kv : kv_lens) {
    for (int n : ns) {
      if (!fits(n, kv) || (long long)n * B > c->Tmax || kv > c->Tmax) continue;
      if (*n_rows + 1 > cap) return DLM_OK;
      int rc = add(n, kv);
      if (rc) return rc;
      const int per = std::max(1, c->Tmax / kv);
      for (int i0 = 0; i0 < n && !rc; i0 += per) {
        dlm_batch rb = {std::min(per, n - i0), ids.data() + i0, nullptr, DLM_DRY_RUN};
        rc = dlm_refresh_step(c, &rb, &res);
      }
      float us = 0.f;
      dlm_batch b = {n, ids.data(), nullptr, DLM_DRY_RUN};
      if (!rc) rc = time_steps(c, &b, &res, DLM_KIND_CACHED, reps, &us);
      drop();
      if (rc) return rc;
      rows[(*n_rows)++] = {DLM_KIND_CACHED, n, n * B, kv, us};
    }
  }
  // ---- recompute steps: total tokens in powers of two (LP[tp][numTokens]), as ONE request up to max_seq, then as
  // several requests of the largest power of two that fits
  int s_big = 128;
  while (2 * s_big <= a.max_seq) s_big *= 2;
  for (long long t = 128; t <= 32768; t *= 2) {
    const long long S = std::min<long long>(t, s_big), n = t / S;
    if (t > c->Tmax || !fits(n, S)) continue;
    if (*n_rows + 1 > cap) return DLM_OK;
    int rc = add((int)n, (int)S);
    if (rc) return rc;
    float us = 0.f;
    dlm_batch b = {(int)n, ids.data(), nullptr, DLM_DRY_RUN};
    rc = time_steps(c, &b, &res, DLM_KIND_REFRESH, reps, &us);
    drop();
    if (rc) return rc;
    rows[(*n_rows)++] = {DLM_KIND_REFRESH, (int)n, (int)t, (int)S, us};
  }
  return DLM_OK;
}

extern "C" int dlm_profile_step_costs(dlm_ctx* c, dlm_cost_row* rows, int32_t cap, int32_t* n_rows) {
  return dlm_profile_step_costs_ex(c, c ? std::min(32, c->a.max_block) : 32, 10, rows, cap, n_rows);
}

// ------------------------------------------------------------------------------------------------
// Kernel-level entry points (include/dlm_ops.h)
// ------------------------------------------------------------------------------------------------
static TmapCache g_op_tmaps;

static int op_check_device() {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    set_err(&g_init_error, "no CUDA device: libdlm has no CPU fallback");
    return DLM_E_CUDA;
  }
  static int sms[kMaxDevices] = {};
  int d = 0;
  cudaGetDevice(&d);
  if (d < 0 || d >= kMaxDevices) { set_err(&g_init_error, "device ordinal %d not supported", d); return DLM_E_CUDA; }
  if (!sms[d]) { cudaDeviceProp p; cudaGetDeviceProperties(&p, d); sms[d] = p.multiProcessorCount; }
  g_dev = d; g_num_sms = sms[d];
  return DLM_OK;
}

extern "C" int dlm_op_gemm_bf16(const void* A, const void* W, void* out, int32_t M, int32_t N, int32_t K, int32_t epi, int32_t bn, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!A || !W || !out || M <= 0 || N <= 0 || K <= 0 || epi < 0 || epi > 3) { set_err(&g_init_error, "dlm_op_gemm_bf16: bad arguments"); return DLM_E_ARG; }
  GemmTcParams p = {};
  p.ldc = N;
  p.up_row0 = N;
  if (epi == EPI_F32 || epi == EPI_RESID) p.out_f32 = (float*)out; else p.out_bf16 = (bf16*)out;
  g_op_tmaps.m.clear(); g_op_tmaps.mo.clear();   // caller buffers come and go; never reuse a stale map
  return gemm_tc(g_op_tmaps, &g_init_error, A, M, W, epi == EPI_SWIGLU ? 2LL * N : N, M, N, K, epi, bn, p, (cudaStream_t)stream);
}

extern "C" int dlm_op_gemm_pair_bf16(const void* A, const void* W, void* out, int32_t M, int32_t N, int32_t K, int32_t epi, int32_t bn,
                                     int32_t splits, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!A || !W || !out || M <= 0 || N <= 0 || K <= 0 || epi < 0 || epi > 3 || splits < 0 || splits > 8 || (splits > 1 && epi != EPI_F32)) {
    set_err(&g_init_error, "dlm_op_gemm_pair_bf16: bad arguments"); return DLM_E_ARG;
  }
  cudaStream_t st = (cudaStream_t)stream;
  GemmPairParams p = {};
  p.ldc = N;
  p.up_row0 = N;
  g_op_tmaps.m.clear(); g_op_tmaps.mo.clear();
  if (epi != EPI_F32 || splits == 1) {
    if (epi == EPI_F32 || epi == EPI_RESID) p.out_f32 = (float*)out; else p.out_bf16 = (bf16*)out;
    rc = gemm_pair(g_op_tmaps, &g_init_error, A, M, W, epi == EPI_SWIGLU ? 2LL * N : N, M, N, K, epi, bn, p, st);
    return rc < 0 ? rc : 1;
  }
  // split-K: slices in a scratch buffer, summed in slice order into `out`
  const long long n = (long long)M * N;
  const int cap = splits ? splits : 4;
  float* part = nullptr;
  if (cudaMalloc(&part, (size_t)cap * n * 4) != cudaSuccess) { set_err(&g_init_error, "dlm_op_gemm_pair_bf16: allocation failed"); return DLM_E_CAPACITY; }
  p.out_f32 = part;
  int ns = 0;
  if (splits == 0) rc = gemm_pair(g_op_tmaps, &g_init_error, A, M, W, N, M, N, K, epi, 0, p, st, false, cap, &ns);
  else rc = gemm_pair(g_op_tmaps, &g_init_error, A, M, W, N, M, N, K, epi, bn > 0 ? bn : 256, p, st, false, -splits, &ns);
  if (!rc) {
    cudaMemsetAsync(out, 0, (size_t)n * 4, st);
    launch_k(add_partials_kernel, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, st, false, (float*)out, (const float*)part, ns, n, n);
  }
  cudaError_t e = cudaStreamSynchronize(st);
  cudaFree(part);
  if (!rc && e != cudaSuccess) { set_err(&g_init_error, "dlm_op_gemm_pair_bf16: %s", cudaGetErrorString(e)); rc = DLM_E_CUDA; }
  return rc < 0 ? rc : ns;
}

extern "C" int dlm_op_gemm_pair_plan(int32_t M, int32_t N, int32_t K, int32_t epi, int32_t* bn, int32_t* bn2, int32_t* n_wide) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!bn || !bn2 || !n_wide || M <= 0 || N <= 0 || K <= 0 || epi < 0 || epi > 3) { set_err(&g_init_error, "dlm_op_gemm_pair_plan: bad arguments"); return DLM_E_ARG; }
  int b = 0, sp = 1, b1 = 0, b2 = 0, na = 0, nb = 0;
  plan_pair(M, N, K, epi, 1, &b, &sp);
  *bn = b; *bn2 = 0; *n_wide = 0;
  if (plan_pair_mixed(M, N, K, epi, b, &b1, &b2, &na, &nb)) { *bn = b1; *bn2 = b2; *n_wide = na; }
  return DLM_OK;
}

extern "C" int dlm_op_gemm_skinny_bf16(const void* X, const void* W, void* out, int32_t T, int32_t N, int32_t K, int32_t epi, int32_t splits, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!X || !W || !out || T <= 0 || T > kSkMaxTokens || N <= 0 || K <= 0 || (epi != EPI_F32 && epi != EPI_SWIGLU)) {
    set_err(&g_init_error, "dlm_op_gemm_skinny_bf16: bad arguments (T must be in [1, %d])", kSkMaxTokens); return DLM_E_ARG;
  }
  cudaStream_t st = (cudaStream_t)stream;
  g_op_tmaps.m.clear(); g_op_tmaps.mo.clear();
  SkinnyParams p = {};
  p.ldc = N; p.up_row0 = N;
  if (epi == EPI_SWIGLU) {
    p.out_bf16 = (bf16*)out;
    return gemm_skinny(g_op_tmaps, &g_init_error, X, T, W, 2LL * N, T, N, K, SK_SWIGLU, 0, p, nullptr, st, false);
  }
  float* part = nullptr;
  const long long n = (long long)T * N;
  if (cudaMalloc(&part, (size_t)kSkMaxSplits * n * 4) != cudaSuccess) { set_err(&g_init_error, "dlm_op_gemm_skinny_bf16: allocation failed"); return DLM_E_CAPACITY; }
  p.out_f32 = part;
  int ns = 0;
  rc = gemm_skinny(g_op_tmaps, &g_init_error, X, T, W, N, T, N, K, SK_PARTIAL, splits, p, &ns, st, false);
  if (!rc) {
    cudaMemsetAsync(out, 0, (size_t)n * 4, st);
    launch_k(add_partials_kernel, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, st, false, (float*)out, (const float*)part, ns, n, n);
  }
  cudaError_t e = cudaStreamSynchronize(st);
  cudaFree(part);
  if (!rc && e != cudaSuccess) { set_err(&g_init_error, "dlm_op_gemm_skinny_bf16: %s", cudaGetErrorString(e)); rc = DLM_E_CUDA; }
  return rc < 0 ? rc : ns;
}

extern "C" int dlm_op_gemm_plain_bf16(const void* A, const void* W, float* out, int32_t M, int32_t N, int32_t K, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!A || !W || !out || M <= 0 || N <= 0 || K <= 0) { set_err(&g_init_error, "dlm_op_gemm_plain_bf16: bad arguments"); return DLM_E_ARG; }
  gemm_plain<bf16, bf16>(out, (const bf16*)A, (const bf16*)W, M, N, K, (cudaStream_t)stream);
  return cudaGetLastError() == cudaSuccess ? DLM_OK : DLM_E_CUDA;
}

extern "C" int64_t dlm_op_lmhead_scratch_bytes(int32_t R, int32_t V) {
  return (int64_t)std::max(R, 1) * ((V + 127) / 128) * (int64_t)sizeof(RowPartial) + (int64_t)R * 64 + 4096;
}

// batch descriptor for the stand-alone head ops: n requests of B rows, block = positions [0, B) of a private token row
static int op_head(const void* hidden, const void* Wlm, int n, int B, int V, int K, float scale, int mask_id, const float* tau,
                   int* tokens_io, StepOut so, void* scratch, cudaStream_t st, int dry) {
  const int R = n * B;
  int n_tiles = (V + 127) / 128;
  RowPartial* part = (RowPartial*)scratch;
  int* meta = (int*)((char*)scratch + (size_t)R * n_tiles * sizeof(RowPartial));
  // meta: slot[n], blk_lo[n], blk_len[n], row_off[n]  (+ tau passed separately)
  std::vector<int> h(4 * n);
  for (int i = 0; i < n; ++i) { h[i] = i; h[n + i] = 0; h[2 * n + i] = B; h[3 * n + i] = i * B; }
  cudaMemcpyAsync(meta, h.data(), h.size() * 4, cudaMemcpyHostToDevice, st);
  cudaStreamSynchronize(st);   // h is a stack-lifetime staging buffer
  g_op_tmaps.m.clear(); g_op_tmaps.mo.clear();
  int rc;
  if (R > 128) {                 // as in the engine: the CTA-pair kernel with 256-wide vocabulary tiles above 128 rows
    n_tiles = (V + 255) / 256;
    GemmPairParams p = {};
    p.part = part; p.n_tiles = n_tiles; p.mask_id = mask_id; p.scale = scale;
    rc = gemm_pair(g_op_tmaps, &g_init_error, hidden, R, Wlm, V, R, V, K, EPI_LMHEAD, 256, p, st);
  } else {
    GemmTcParams p = {};
    p.part = part; p.n_tiles = n_tiles; p.mask_id = mask_id; p.scale = scale;
    rc = gemm_tc(g_op_tmaps, &g_init_error, hidden, R, Wlm, V, R, V, K, EPI_LMHEAD, 128, p, st);
  }
  if (rc) return rc;
  BatchDesc bd = {};
  bd.n = n; bd.R = R; bd.slot = meta; bd.blk_lo = meta + n; bd.blk_len = meta + 2 * n; bd.row_off = meta + 3 * n; bd.tau = tau;
  combine_unmask_kernel<<<n, 1024, 0, st>>>(so, part, n_tiles, tokens_io, B, B, mask_id, bd, dry);
  DLM_LAUNCH_CHECK();
  return cudaGetLastError() == cudaSuccess ? DLM_OK : DLM_E_CUDA;
}

extern "C" int dlm_op_lmhead_unmask_bf16(const void* hidden, const void* Wlm, int32_t n, int32_t B, int32_t V, int32_t K, float scale,
                                          int32_t mask_id, const float* tau, int32_t* tokens_io, int32_t* n_committed, int32_t* pos,
                                          int32_t* tok, float* conf, void* scratch, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!hidden || !Wlm || !tau || !tokens_io || !n_committed || !pos || !tok || !conf || !scratch || n <= 0 || B <= 0 || B > 64 || K % 8) {
    set_err(&g_init_error, "dlm_op_lmhead_unmask_bf16: bad arguments"); return DLM_E_ARG;
  }
  // row statistics land after the metadata in scratch
  const int R = n * B;
  char* extra = (char*)scratch + (size_t)R * ((V + 127) / 128) * sizeof(RowPartial) + (size_t)16 * n + 256;
  StepOut so;
  so.n_committed = n_committed; so.pos = pos; so.tok = tok; so.conf = conf;
  so.row_lse = (float*)extra; so.row_conf = (float*)extra + R; so.row_tok = (int*)extra + 2 * R;
  return op_head(hidden, Wlm, n, B, V, K, scale, mask_id, tau, tokens_io, so, scratch, (cudaStream_t)stream, 0);
}

extern "C" int dlm_op_lmhead_bf16(const void* hidden, const void* Wlm, int32_t R, int32_t V, int32_t K, float scale, int32_t mask_id,
                                   int32_t* tok, float* conf, float* lse, void* scratch, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!hidden || !Wlm || !tok || !conf || !lse || !scratch || R <= 0 || K % 8) { set_err(&g_init_error, "dlm_op_lmhead_bf16: bad arguments"); return DLM_E_ARG; }
  // every row is its own "request" of one block row; commits are discarded (dry run), only row stats are kept
  const int n_tiles = (V + 127) / 128;
  char* extra = (char*)scratch + (size_t)R * n_tiles * sizeof(RowPartial) + (size_t)16 * R + 256;
  int* dummy = (int*)extra;                 // n_committed[R], pos[R], tok[R], conf[R], tokens[R], tau[R]
  StepOut so;
  so.n_committed = dummy; so.pos = dummy + R; so.tok = dummy + 2 * R; so.conf = (float*)(dummy + 3 * R);
  so.row_lse = lse; so.row_conf = conf; so.row_tok = tok;
  int* tokens = dummy + 4 * R;
  float* tau = (float*)(dummy + 5 * R);
  cudaMemsetAsync(tokens, 0, (size_t)R * 4, (cudaStream_t)stream);
  cudaMemsetAsync(tau, 0, (size_t)R * 4, (cudaStream_t)stream);
  return op_head(hidden, Wlm, R, 1, V, K, scale, mask_id, tau, tokens, so, scratch, (cudaStream_t)stream, 1);
}

extern "C" int dlm_op_attention_bf16(const void* q, const void* k, const void* v, void* out, int32_t Tq, int32_t S, int32_t H,
                                      int32_t Hkv, int32_t dh, int32_t flash, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  return attn_op_contiguous(q, k, v, out, Tq, S, H, Hkv, dh, flash, (cudaStream_t)stream, &g_init_error);
}

// ------------------------------------------------------------------------------------------------
// dlm_op_lmhead_static_bf16 (dlm_ops.h): the fused LM head for callers that cannot allocate device memory.
// Its scratch is the file-scope array below, part of the module image: every GPU that loads libdlm.so holds
// DLM_LMHEAD_STATIC_SCRATCH_BYTES for it until the process exits, and all calls on a device share it.
// In host code the name `g_lmhead_static` is only the host-side handle of that array, not a device address: the
// address comes from cudaGetSymbolAddress, looked up once per device with that device current.  Device code in this
// file may name the array directly (lmhead_static_meta_kernel does).
// Layout of one call's use (every region a multiple of 256 bytes):
//   RowPartial part[R][n_tiles] | int slot[R] blk_lo[R] blk_len[R] row_off[R] | int n_committed[R] pos[R] tok[R]
//   float conf[R] | int tokens[R] | float tau[R]
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_lmhead_static[DLM_LMHEAD_STATIC_SCRATCH_BYTES];

static inline size_t static_align256(size_t b) { return (b + 255) & ~(size_t)255; }
constexpr int kStaticHeadIntRows = 10;    // the ten R-long rows that follow the partials

extern "C" int64_t dlm_op_lmhead_static_bytes(int32_t R, int32_t V) {
  if (R <= 0 || V <= 0) return 0;
  return (int64_t)(static_align256((size_t)R * ((V + 127) / 128) * sizeof(RowPartial)) + kStaticHeadIntRows * static_align256((size_t)R * 4));
}

// Row metadata of "R requests of one block row each" and the rows that have to start at zero (token ids: nothing is
// masked, nothing committed from an earlier call; thresholds), rewritten by every call because the array keeps the
// previous call's contents.  Names the array directly: in device code the symbol IS the device array.
__global__ void lmhead_static_meta_kernel(long long meta_off, int R, int stride) {
  int* meta = reinterpret_cast<int*>(g_lmhead_static + meta_off);
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= R) return;
  meta[i] = i;                    // slot
  meta[stride + i] = 0;           // blk_lo
  meta[2 * stride + i] = 1;       // blk_len
  meta[3 * stride + i] = i;       // row_off
  meta[8 * stride + i] = 0;       // tokens
  meta[9 * stride + i] = 0;       // tau = 0.0f
}

// Device address of g_lmhead_static on the current device; looked up on the first call per device.
static int lmhead_static_base(unsigned char** base) {
  static unsigned char* ptrs[kMaxDevices] = {};
  const int d = g_dev;            // set by op_check_device() from cudaGetDevice()
  if (!ptrs[d]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_lmhead_static);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      set_err(&g_init_error, "dlm_op_lmhead_static_bf16: cudaGetSymbolAddress on device %d failed: %s", d, cudaGetErrorString(e));
      return DLM_E_CUDA;
    }
    ptrs[d] = (unsigned char*)p;
  }
  *base = ptrs[d];
  return DLM_OK;
}

extern "C" int dlm_op_lmhead_static_bf16(const void* hidden, const void* Wlm, int32_t R, int32_t V, int32_t K, float scale,
                                          int32_t mask_id, int32_t* tok, float* conf, float* lse, void* stream) {
  int rc = op_check_device();
  if (rc) return rc;
  if (!hidden || !Wlm || !tok || !conf || !lse || R <= 0 || V <= 0 || K <= 0 || K % 8) {
    set_err(&g_init_error, "dlm_op_lmhead_static_bf16: bad arguments"); return DLM_E_ARG;
  }
  const long long need = dlm_op_lmhead_static_bytes(R, V);
  if (R > DLM_LMHEAD_STATIC_MAX_ROWS || need > (long long)DLM_LMHEAD_STATIC_SCRATCH_BYTES) {
    set_err(&g_init_error, "dlm_op_lmhead_static_bf16: R = %d rows x V = %d columns needs %lld bytes of scratch; the built-in array "
            "holds %d bytes and at most %d rows (use dlm_op_lmhead_bf16 with a caller-owned scratch buffer)",
            R, V, need, (int)DLM_LMHEAD_STATIC_SCRATCH_BYTES, (int)DLM_LMHEAD_STATIC_MAX_ROWS);
    return DLM_E_CAPACITY;
  }
  unsigned char* base = nullptr;
  if ((rc = lmhead_static_base(&base)) != DLM_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int n_tiles = (V + 127) / 128;
  const size_t meta_off = static_align256((size_t)R * n_tiles * sizeof(RowPartial));
  const int stride = (int)(static_align256((size_t)R * 4) / 4);
  RowPartial* part = (RowPartial*)base;
  int* meta = (int*)(base + meta_off);

  lmhead_static_meta_kernel<<<(R + 127) / 128, 128, 0, st>>>((long long)meta_off, R, stride);
  DLM_LAUNCH_CHECK();

  // the single-CTA-per-tile tcgen05 GEMM with the split-vocab epilogue, as op_head / gemm_tc set it up for R <= 128;
  // tensor maps live on this stack frame (kernel parameters are copied at launch)
  GemmTcParams p = {};
  p.M = R; p.N = V; p.K = K; p.bn = 128;
  p.a_box_rows = R <= 32 ? 32 : (R <= 64 ? 64 : 128);
  const int num_kb = (K + kBK - 1) / kBK;
  p.stages = std::max(2, std::min(std::min(num_kb, 12), (200 * 1024) / gemm_tc_stage_bytes(128)));
  p.w_policy = DLM_L2_EVICT_FIRST;
  p.part = part; p.n_tiles = n_tiles; p.mask_id = mask_id; p.scale = scale;
  CUtensorMap ma, mb;
  if (!make_tmap_bf16(&ma, hidden, R, K, p.a_box_rows) || !make_tmap_bf16(&mb, Wlm, V, K, 128)) {
    set_err(&g_init_error, "dlm_op_lmhead_static_bf16: cuTensorMapEncodeTiled failed"); return DLM_E_CUDA;
  }
  cudaError_t e = launch_gemm_tc_t<EPI_LMHEAD>(&ma, &mb, p, n_tiles, st, false);
  if (e != cudaSuccess) { set_err(&g_init_error, "dlm_op_lmhead_static_bf16: launch failed: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }

  // every row is its own request of one block row; the commit lists go to the array and are dropped (dry run)
  StepOut so;
  so.n_committed = meta + 4 * stride; so.pos = meta + 5 * stride; so.tok = meta + 6 * stride; so.conf = (float*)(meta + 7 * stride);
  so.row_lse = lse; so.row_conf = conf; so.row_tok = tok;
  BatchDesc bd = {};
  bd.n = R; bd.R = R; bd.slot = meta; bd.blk_lo = meta + stride; bd.blk_len = meta + 2 * stride; bd.row_off = meta + 3 * stride;
  bd.tau = (const float*)(meta + 9 * stride);
  combine_unmask_kernel<<<R, 1024, 0, st>>>(so, part, n_tiles, meta + 8 * stride, 1, 1, mask_id, bd, 1);
  DLM_LAUNCH_CHECK();
  e = cudaGetLastError();
  if (e != cudaSuccess) { set_err(&g_init_error, "dlm_op_lmhead_static_bf16: %s", cudaGetErrorString(e)); return DLM_E_CUDA; }
  return DLM_OK;
}
