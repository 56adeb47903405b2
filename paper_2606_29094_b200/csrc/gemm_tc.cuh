// tcgen05 / TMEM GEMM fed by TMA:  D[M, N] = A[M, K] . W[N, K]^T,  A = activations (bf16, K-major),
// W = weights (bf16, [out, in] row-major = K-major), fp32 accumulation in tensor memory.
// Rows a3, a6, a8, a9, a11 of DESIGN.md's hot-path table.
//
// One CTA computes one 128 x BN output tile (BN a runtime multiple of 16/32, 32..256):
//   warp 0      TMA producer: per 64-wide K block, one box of A (a_box_rows x 64) and one (two for SwiGLU) of W
//               into a `stages`-deep shared-memory ring (SWIZZLE_128B), completion on full[stage]
//   warp 1      TMEM allocation; one elected lane issues 4 x tcgen05.mma (128 x BN x 16) per K block and
//               tcgen05.commit's the stage back to the producer; the last commit signals the epilogue
//   warps 2..5  epilogue: tcgen05.ld the accumulator (lane = row, 32 columns at a time) and apply the fused
//               epilogue: fp32 store | bf16 store | residual add into the fp32 stream | SwiGLU -> bf16 |
//               LM-head split-vocab statistics (max, sum exp, argmax) -- logits never reach HBM.
// Rows >= M of a tile hold stale activations; each D row depends on its own A row only and is never stored.
#pragma once
#include "common.cuh"
#include "kernels_basic.cuh"
#include "ptx_sm100.cuh"

namespace dlm {

enum { EPI_F32 = 0, EPI_BF16 = 1, EPI_RESID = 2, EPI_SWIGLU = 3, EPI_LMHEAD = 4 };

struct GemmTcParams {
  int M, N, K;        // N = output features (SwiGLU: F; a tile covers bn/2 of them)
  int bn;             // MMA N of the CTA tile
  int a_box_rows;     // rows the A tensor map's box loads (<= 128)
  int stages;
  int up_row0;        // SwiGLU: first row of the up projection inside W (= F)
  float* out_f32;     // EPI_F32 / EPI_RESID
  bf16* out_bf16;     // EPI_BF16 / EPI_SWIGLU
  long long ldc;
  RowPartial* part;   // EPI_LMHEAD: [M, n_tiles]
  int n_tiles;
  int mask_id;
  float scale;
  unsigned long long w_policy;   // L2 cache hint for the weight stream
  TraceSlot tr;                  // DLM_OPT_TRACE record of this launch (null: off)
};

constexpr int kGemmThreads = 192;
constexpr int kBK = 64;                 // K block = one 128-byte swizzle row of bf16
constexpr int kATileBytes = 128 * 128;  // 128 rows x 64 bf16

__host__ __device__ inline int gemm_tc_stage_bytes(int bn) { return kATileBytes + bn * 128; }
__host__ inline int gemm_tc_smem_bytes(int bn, int stages) { return stages * gemm_tc_stage_bytes(bn) + 1024 + 256; }

template <int EPI>
__global__ void __launch_bounds__(kGemmThreads, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const GemmTcParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const int BN = p.bn;
  const int stages = p.stages;
  const uint32_t stage_bytes = gemm_tc_stage_bytes(BN);
  const uint32_t bar_base = base + stages * stage_bytes;        // full[stages], empty[stages], tmem_full, tmem_ptr
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (stages + s); };
  const uint32_t tmem_full_bar = bar_base + 16u * stages;
  const uint32_t tmem_ptr_addr = tmem_full_bar + 8u;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.y * 128;
  const int tile_n = blockIdx.x;
  const int num_kb = (p.K + kBK - 1) / kBK;
  uint32_t tmem_cols = 32;
  while ((int)tmem_cols < BN) tmem_cols <<= 1;

  ptx::pdl_launch_dependents();
  if (threadIdx.x == 0) trace_begin(p.tr);
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&mapA);
    ptx::prefetch_tmap(&mapB);
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
      const uint32_t a_bytes = (uint32_t)p.a_box_rows * 128u;
      const uint32_t tx = a_bytes + (uint32_t)BN * 128u;
      auto load_w = [&](int kb, int s) {
        const uint32_t sb = base + s * stage_bytes + kATileBytes;
        ptx::mbar_expect_tx(full_bar(s), tx);
        if (EPI == EPI_SWIGLU) {
          const int f0 = tile_n * (BN / 2);
          ptx::tma_load_2d(sb, &mapB, kb * kBK, f0, full_bar(s), p.w_policy);
          ptx::tma_load_2d(sb + (BN / 2) * 128, &mapB, kb * kBK, p.up_row0 + f0, full_bar(s), p.w_policy);
        } else {
          ptx::tma_load_2d(sb, &mapB, kb * kBK, tile_n * BN, full_bar(s), p.w_policy);
        }
      };
      auto load_a = [&](int kb, int s) { ptx::tma_load_2d(base + s * stage_bytes, &mapA, kb * kBK, m0, full_bar(s), DLM_L2_EVICT_LAST); };
      // weights do not depend on the upstream kernel: fill the ring with them before the PDL wait
      const int pre = min(stages, num_kb);
      for (int kb = 0; kb < pre; ++kb) load_w(kb, kb);
      ptx::pdl_wait();
      trace_wait(p.tr);
      for (int kb = 0; kb < pre; ++kb) load_a(kb, kb);
      // ring position as running (stage, phase) counters (no run-time division per K block); pre == stages here
      for (int kb = pre, s = 0, ph = 1; kb < num_kb; ++kb, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1 : 0)) {
        ptx::mbar_wait(empty_bar(s), (uint32_t)ph ^ 1u);
        load_w(kb, s);
        load_a(kb, s);
      }
    }
  } else if (warp == 1) {
    // ---------------- MMA issuer (the whole warp walks the loop, one elected lane issues) ----------------
    const uint32_t idesc = ptx::umma_idesc_bf16(128, BN);
    for (int kb = 0, s = 0, ph = 0; kb < num_kb; ++kb, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1 : 0)) {
      ptx::mbar_wait(full_bar(s), (uint32_t)ph);
      ptx::tc_fence_after();
      if (ptx::elect_one()) {
        const uint32_t sa = base + s * stage_bytes;
        const uint32_t a_lo = ptx::umma_desc_lo(sa), b_lo = ptx::umma_desc_lo(sa + kATileBytes);
#pragma unroll
        for (int k = 0; k < kBK / 16; ++k)            // +32 bytes along K inside the 128-byte swizzle row = +2 in the encoded address
          ptx::umma_bf16_lo(tmem_base, a_lo + 2 * k, b_lo + 2 * k, idesc, (kb | k) != 0 ? 1u : 0u);
        ptx::umma_commit(empty_bar(s));            // frees the stage once these MMAs have read it
        if (kb + 1 == num_kb) ptx::umma_commit(tmem_full_bar);       // accumulator complete
      }
      __syncwarp();
    }
  } else {
    // ---------------- epilogue (warps 2..5; TMEM lane quarter = warp % 4) ----------------
    const int quarter = warp & 3;
    const int row = m0 + quarter * 32 + lane;
    const bool row_ok = row < p.M;
    ptx::mbar_wait(tmem_full_bar, 0);
    ptx::tc_fence_after();
    const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16);
    uint32_t r[32];
    if (EPI == EPI_F32 || EPI == EPI_RESID || EPI == EPI_BF16) {
      const int n0 = tile_n * BN;
      for (int c = 0; c < BN / 32; ++c) {
        __syncwarp();
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_wait();
        const int col0 = n0 + c * 32;
        if (!row_ok || col0 >= p.N) {
          // nothing to store for this thread / chunk (keeps the warp converged for the next tcgen05.ld)
        } else if (EPI == EPI_BF16) {
          bf16* o = p.out_bf16 + (long long)row * p.ldc + col0;
          if (col0 + 32 <= p.N) {
#pragma unroll
            for (int j = 0; j < 32; j += 8) {
              uint4 v;
              __nv_bfloat162 t0 = __floats2bfloat162_rn(__uint_as_float(r[j]), __uint_as_float(r[j + 1]));
              __nv_bfloat162 t1 = __floats2bfloat162_rn(__uint_as_float(r[j + 2]), __uint_as_float(r[j + 3]));
              __nv_bfloat162 t2 = __floats2bfloat162_rn(__uint_as_float(r[j + 4]), __uint_as_float(r[j + 5]));
              __nv_bfloat162 t3 = __floats2bfloat162_rn(__uint_as_float(r[j + 6]), __uint_as_float(r[j + 7]));
              v.x = *reinterpret_cast<uint32_t*>(&t0); v.y = *reinterpret_cast<uint32_t*>(&t1);
              v.z = *reinterpret_cast<uint32_t*>(&t2); v.w = *reinterpret_cast<uint32_t*>(&t3);
              *reinterpret_cast<uint4*>(o + j) = v;
            }
          } else {
            #pragma unroll
            for (int j = 0; j < 32; ++j) if (col0 + j < p.N) o[j] = __float2bfloat16_rn(__uint_as_float(r[j]));
          }
        } else {
          float* o = p.out_f32 + (long long)row * p.ldc + col0;
          if (col0 + 32 <= p.N) {
#pragma unroll
            for (int j = 0; j < 32; j += 4) {
              float4 v = make_float4(__uint_as_float(r[j]), __uint_as_float(r[j + 1]), __uint_as_float(r[j + 2]),
                                     __uint_as_float(r[j + 3]));
              if (EPI == EPI_RESID) {
                float4 x = *reinterpret_cast<float4*>(o + j);
                v.x += x.x; v.y += x.y; v.z += x.z; v.w += x.w;
              }
              *reinterpret_cast<float4*>(o + j) = v;
            }
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              if (col0 + j < p.N) {
                float v = __uint_as_float(r[j]);
                o[j] = (EPI == EPI_RESID) ? o[j] + v : v;
              }
            }
          }
        }
      }
    } else if (EPI == EPI_SWIGLU) {
      const int half = BN / 2;
      const int f0 = tile_n * half;
      uint32_t u[32];
      for (int c = 0; c < half / 32; ++c) {
        __syncwarp();
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_32x32(taddr + half + c * 32, u);
        ptx::tmem_ld_wait();
        const int fc = f0 + c * 32;
        bf16* o = p.out_bf16 + (long long)row * p.ldc + fc;
        if (!row_ok || fc >= p.N) {
        } else if (fc + 32 <= p.N) {
#pragma unroll
          for (int j = 0; j < 32; j += 8) {
            uint32_t w[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              float a0 = silu_f(__uint_as_float(r[j + 2 * q])) * __uint_as_float(u[j + 2 * q]);
              float a1 = silu_f(__uint_as_float(r[j + 2 * q + 1])) * __uint_as_float(u[j + 2 * q + 1]);
              __nv_bfloat162 t = __floats2bfloat162_rn(a0, a1);
              w[q] = *reinterpret_cast<uint32_t*>(&t);
            }
            *reinterpret_cast<uint4*>(o + j) = make_uint4(w[0], w[1], w[2], w[3]);
          }
        } else {
#pragma unroll
          for (int j = 0; j < 32; ++j)
            if (fc + j < p.N) o[j] = __float2bfloat16_rn(silu_f(__uint_as_float(r[j])) * __uint_as_float(u[j]));
        }
      }
    } else if (EPI == EPI_LMHEAD) {
      // a11: split-vocab online (max, sum exp(z - max), argmax); z = scale * acc; mask_id and columns >= V excluded.
      const int n0 = tile_n * BN;
      float m = -CUDART_INF_F, ssum = 0.f;
      int idx = 0x7fffffff;
      for (int c = 0; c < BN / 32; ++c) {
        __syncwarp();
        ptx::tmem_ld_32x32(taddr + c * 32, r);
        ptx::tmem_ld_wait();
        const int col0 = n0 + c * 32;
        float cm = -CUDART_INF_F;
        int ci = 0x7fffffff;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const int col = col0 + j;
          float z = __uint_as_float(r[j]) * p.scale;
          if (col >= p.N || col == p.mask_id) z = -CUDART_INF_F;
          r[j] = __float_as_uint(z);
          if (z > cm) { cm = z; ci = col; }        // strict > keeps the lowest column on ties
        }
        if (cm != -CUDART_INF_F) {
          if (cm > m) { ssum *= __expf(m - cm); m = cm; idx = ci; }
          float cs = 0.f;
#pragma unroll
          for (int j = 0; j < 32; ++j) cs += __expf(__uint_as_float(r[j]) - m);
          ssum += cs;
        }
      }
      if (row_ok) {
        RowPartial o;
        o.m = m; o.s = ssum; o.idx = idx; o.pad = 0;
        *reinterpret_cast<int4*>(p.part + (long long)row * p.n_tiles + tile_n) = *reinterpret_cast<int4*>(&o);
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) trace_end(p.tr);
  if (warp == 1) ptx::tmem_dealloc(tmem_base, tmem_cols);
}

}  // namespace dlm
