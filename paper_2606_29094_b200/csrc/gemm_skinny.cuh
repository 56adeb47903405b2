// Weight-streaming tcgen05 GEMM for small token counts (T <= 128): the cached step's a3/a6/a8/a9.
//
//   D[T, N] = X[T, K] . W[N, K]^T        X = activations (bf16), W = weights ([out, in] row-major, bf16)
//
// With 32..128 tokens the contraction is HBM-bound (each weight byte is used once per step), so the kernel is
// organised around keeping weight bytes in flight, not around MMA efficiency:
//   * swap-AB: the WEIGHT tile is the MMA's M operand (128 output features = 128 TMEM lanes), the tokens are
//     the MMA's N (tpad = 32/64/96/128 columns).  All 128 lanes and all four epilogue warps do useful work and
//     one 128 x tpad x 16 MMA costs tpad/2 cycles per 4 KB of weights.
//   * split-K: work item = (128-feature tile, K range).  Splits are chosen on the host so that ~2 CTAs per SM
//     (296 items) stream concurrently even when N / 128 is only 32 (O / down projections).  Every split writes
//     an fp32 partial slice [split][T][N]; the consumer kernel (RMSNorm / RoPE) sums the slices in a fixed
//     order, so results are deterministic (no atomics).
//   * programmatic dependent launch: weights do not depend on the previous kernel, so the producer warp fills
//     the whole shared-memory ring with weight tiles BEFORE griddepcontrol.wait and only the activation tiles
//     wait for the upstream kernel.  HBM stays busy across kernel boundaries.
//   * SwiGLU epilogue (a8): a tile holds 64 gate rows and 64 up rows of the same features; the gate half
//     passes silu(g) to the up half through shared memory; act = silu(g) * u goes out as bf16.
// Token columns >= T hold stale activations; each D column depends on its own X row only and is never stored.
#pragma once
#include "common.cuh"
#include "kernels_basic.cuh"
#include "ptx_sm100.cuh"

namespace dlm {

enum { SK_PARTIAL = 0, SK_SWIGLU = 1 };

struct SkinnyParams {
  int T, N, K;            // N = output features (SwiGLU: F)
  int tpad;               // MMA N: multiple of 32 in [32, 128], >= T
  int splits;             // K splits (grid.y)
  int kb_per_split;       // 64-wide K blocks per split
  int stages;
  int up_row0;            // SwiGLU: first row of the up projection inside W (= F)
  float* out_f32;         // SK_PARTIAL: [splits][T][ldc]
  bf16* out_bf16;         // SK_SWIGLU:  [T][ldc]
  long long ldc;
  unsigned long long w_policy;
  int w_box;              // 0: W row-major (2-D map); else tiled storage, rows per TMA box (ptx::tma_load_w_tiled)
  TraceSlot tr;           // DLM_OPT_TRACE record of this launch (null: off)
};

constexpr int kSkThreads = 192;
constexpr int kSkWBytes = 128 * 128;     // 128 weight rows x 64 bf16

__host__ __device__ inline int skinny_stage_bytes(int tpad) { return kSkWBytes + tpad * 128; }
__host__ inline int skinny_smem_bytes(int tpad, int stages, int epi) {
  return stages * skinny_stage_bytes(tpad) + 1024 + 256 + (epi == SK_SWIGLU ? 32 * 65 * 4 : 0);
}

template <int EPI>
__global__ void __launch_bounds__(kSkThreads, 2)
gemm_skinny_kernel(const __grid_constant__ CUtensorMap mapW, const __grid_constant__ CUtensorMap mapX, const SkinnyParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const int stages = p.stages;
  const uint32_t stage_bytes = skinny_stage_bytes(p.tpad);
  const uint32_t bar_base = base + stages * stage_bytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (stages + s); };
  const uint32_t tmem_full_bar = bar_base + 16u * stages;
  const uint32_t tmem_ptr_addr = tmem_full_bar + 8u;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tile = blockIdx.x, split = blockIdx.y;
  const int num_kb_total = (p.K + 63) / 64;
  const int kb0 = split * p.kb_per_split;
  const int nkb = min(p.kb_per_split, num_kb_total - kb0);      // >= 1 by construction of the grid
  const uint32_t tmem_cols = p.tpad <= 32 ? 32u : (p.tpad <= 64 ? 64u : 128u);

  ptx::pdl_launch_dependents();            // the next kernel may start its own weight prefetch
  if (threadIdx.x == 0) trace_begin(p.tr);
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&mapW);
    ptx::prefetch_tmap(&mapX);
    for (int s = 0; s < stages; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    ptx::mbar_init(tmem_full_bar, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 1) {
    ptx::tmem_alloc(tmem_ptr_addr, tmem_cols);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr));

  if (warp == 0) {
    if (ptx::elect_one()) {        // one elected lane of the converged warp: TMA issues compile straight-line
      // ---------------- TMA producer ----------------
      const uint32_t tx = (uint32_t)kSkWBytes + (uint32_t)p.tpad * 128u;
      auto load_w = [&](int kb, int s) {
        const uint32_t sw = base + s * stage_bytes;
        const int kcol = (kb0 + kb) * 64;
        ptx::mbar_expect_tx(full_bar(s), tx);
        if (p.w_box) {
          if (EPI == SK_SWIGLU) {
            ptx::tma_load_w_tiled(sw, &mapW, kb0 + kb, tile * 64, 64, p.w_box, full_bar(s), p.w_policy);
            ptx::tma_load_w_tiled(sw + 64 * 128, &mapW, kb0 + kb, p.up_row0 + tile * 64, 64, p.w_box, full_bar(s), p.w_policy);
          } else {
            ptx::tma_load_w_tiled(sw, &mapW, kb0 + kb, tile * 128, 128, p.w_box, full_bar(s), p.w_policy);
          }
        } else if (EPI == SK_SWIGLU) {
          ptx::tma_load_2d(sw, &mapW, kcol, tile * 64, full_bar(s), p.w_policy);
          ptx::tma_load_2d(sw + 64 * 128, &mapW, kcol, p.up_row0 + tile * 64, full_bar(s), p.w_policy);
        } else {
          ptx::tma_load_2d(sw, &mapW, kcol, tile * 128, full_bar(s), p.w_policy);
        }
      };
      auto load_x = [&](int kb, int s) {
        ptx::tma_load_2d(base + s * stage_bytes + kSkWBytes, &mapX, (kb0 + kb) * 64, 0, full_bar(s), DLM_L2_EVICT_LAST);
      };
      const int pre = min(stages, nkb);
      for (int kb = 0; kb < pre; ++kb) load_w(kb, kb);          // weights: independent of the upstream kernel
      ptx::pdl_wait();                                           // activations: written by the upstream kernel
      trace_wait(p.tr);
      for (int kb = 0; kb < pre; ++kb) load_x(kb, kb);
      // ring position as running (stage, phase) counters (no run-time division per K block); pre == stages here
      for (int kb = pre, s = 0, ph = 1; kb < nkb; ++kb, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1 : 0)) {
        ptx::mbar_wait(empty_bar(s), (uint32_t)ph ^ 1u);
        load_w(kb, s);
        load_x(kb, s);
      }
    }
  } else if (warp == 1) {
    // ---------------- MMA issuer: D[128 features, tpad tokens] += W_tile . X_tile^T (whole warp walks, one elected lane issues) ----------------
    const uint32_t idesc = ptx::umma_idesc_bf16(128, p.tpad);
    for (int kb = 0, s = 0, ph = 0; kb < nkb; ++kb, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1 : 0)) {
      ptx::mbar_wait(full_bar(s), (uint32_t)ph);
      ptx::tc_fence_after();
      if (ptx::elect_one()) {
        const uint32_t sw = base + s * stage_bytes;
        const uint32_t w_lo = ptx::umma_desc_lo(sw), x_lo = ptx::umma_desc_lo(sw + kSkWBytes);
#pragma unroll
        for (int k = 0; k < 4; ++k)
          ptx::umma_bf16_lo(tmem_base, w_lo + 2 * k, x_lo + 2 * k, idesc, (kb | k) != 0 ? 1u : 0u);
        ptx::umma_commit(empty_bar(s));
        if (kb + 1 == nkb) ptx::umma_commit(tmem_full_bar);
      }
      __syncwarp();
    }
  } else {
    // ---------------- epilogue (warps 2..5; TMEM lane quarter = warp % 4; lane = output feature) ----------------
    const int quarter = warp & 3;
    ptx::mbar_wait(tmem_full_bar, 0);
    ptx::tc_fence_after();
    const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16);
    uint32_t r[32];
    if (EPI == SK_PARTIAL) {
      const int f = tile * 128 + quarter * 32 + lane;
      float* o = p.out_f32 + (long long)split * p.T * p.ldc + f;
      for (int c = 0; c < p.tpad / 32; ++c) {
        __syncwarp();
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_wait();
        if (f < p.N) {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const int tok = c * 32 + j;
            if (tok < p.T) o[(long long)tok * p.ldc] = __uint_as_float(r[j]);     // 32 lanes -> 128 contiguous bytes
          }
        }
      }
    } else {
      // rows 0..63 of the tile = gate features f0..f0+63 (quarters 0, 1), rows 64..127 = up features (quarters 2, 3)
      float* xch = reinterpret_cast<float*>(smem_raw + (base - ptx::smem_u32(smem_raw)) + stages * stage_bytes + 256);   // [32 tokens][65]
      const int fl = (quarter & 1) * 32 + lane;        // feature inside the tile, 0..63
      const int f = tile * 64 + fl;
      const bool is_gate = quarter < 2;
      for (int c = 0; c < p.tpad / 32; ++c) {
        __syncwarp();
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_wait();
        if (is_gate) {
#pragma unroll
          for (int j = 0; j < 32; ++j) xch[j * 65 + fl] = silu_f(__uint_as_float(r[j]));
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (!is_gate && f < p.N) {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const int tok = c * 32 + j;
            if (tok < p.T) p.out_bf16[(long long)tok * p.ldc + f] = __float2bfloat16_rn(xch[j * 65 + fl] * __uint_as_float(r[j]));
          }
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) trace_end(p.tr);
  if (warp == 1) ptx::tmem_dealloc(tmem_base, tmem_cols);
}

}  // namespace dlm
