// a5  Fused non-causal block attention (bf16, d_h = 128): current-block (or whole-sequence) Q against the paged
// K/V store, online softmax in fp32, GQA-aware, ragged lengths, split-KV for small batches.
//
// The cached step is HBM-bound here (arithmetic intensity = query rows per K/V byte pair, 32-64 flop/B, far
// under the ridge), so the kernel is organised around streaming K/V pages once through shared memory with
// cp.async double buffering; the contractions run on the warp-level tensor-core path (mma.sync m16n8k16),
// which is ample for the bytes it has to keep up with.
//
// Work item = (request, KV head, 64-row query tile, KV split).  Query rows of the r = H/H_kv heads that share a
// KV head are stacked (row rho -> token rho / r, head rho % r) so one pass over K/V serves the whole group.
// 4 warps x 16 rows; K/V tile = 64 tokens (one page slice, contiguous 16 KB per head).
#pragma once
#include <math_constants.h>

#include <algorithm>
#include <string>

#include "common.cuh"

namespace dlm {

constexpr int kFaDh = 128;
constexpr int kFaBM = 64;
constexpr int kFaBN = 64;
constexpr int kFaThreads = 128;
constexpr int kFaSmem = (kFaBM * kFaDh + 4 * kFaBN * kFaDh) * 2;   // Q + 2 x (K, V) = 80 KB

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
  int sz = valid ? 16 : 0;   // src-size 0 => zero fill
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&t);
}
// [rows][128] bf16 tile, 16-byte chunks XOR-swizzled by row%8 (conflict-free ldmatrix)
__device__ __forceinline__ uint32_t tile_off(int row, int chunk) { return (uint32_t)(row * 256 + ((chunk ^ (row & 7)) << 4)); }

struct FaParams {
  bf16* out;                // [T, H, 128]
  const bf16* q;            // [T, H, 128]
  const bf16* kv_store;
  const int* page_table;
  BatchDesc b;
  KvGeom g;
  int layer, n_heads, splits;
  float scale_log2;         // (1/sqrt(d_h)) * log2(e)
  float* ws_o;              // [splits, T*H, 128] unnormalised partial outputs (splits > 1)
  float* ws_ml;             // [splits, T*H, 2]   (running max in log2 units, running sum)
  TraceSlot tr;             // DLM_OPT_TRACE record of this launch (null: off)
};

__global__ void __launch_bounds__(kFaThreads) attn_flash_kernel(const FaParams p) {
  extern __shared__ __align__(128) uint8_t fa_smem[];
  DLM_PROLOGUE(p.tr);
  const int bi = blockIdx.z / p.splits, split = blockIdx.z % p.splits;
  const int kvh = blockIdx.y;
  const int r = p.n_heads / p.g.n_kv_heads;
  const int q_len = p.b.q_len[bi];
  const int n_rows = q_len * r;                       // stacked query rows of this (request, KV head)
  const int row0 = blockIdx.x * kFaBM;
  if (row0 >= n_rows) return;
  const int S = p.b.kv_len[bi];
  const int n_tiles = (S + kFaBN - 1) / kFaBN;
  const int tiles_per = (n_tiles + p.splits - 1) / p.splits;
  const int t_begin = split * tiles_per, t_end = min(n_tiles, t_begin + tiles_per);
  const int q_off = p.b.q_off[bi];
  const int* pt = p.page_table + (long long)p.b.slot[bi] * p.g.max_pages_per_req;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t sQ = (uint32_t)__cvta_generic_to_shared(fa_smem);
  const uint32_t sK = sQ + kFaBM * 256, sV = sK + 2 * kFaBN * 256;
  const int H = p.n_heads;

  // ---- load the Q tile (zero-fill rows past the end) ----
  for (int i = tid; i < kFaBM * 16; i += kFaThreads) {
    const int row = i >> 4, ch = i & 15;
    const int rho = row0 + row;
    const bool ok = rho < n_rows;
    const int tok = ok ? rho / r : 0, hh = ok ? rho % r : 0;
    const bf16* src = p.q + ((long long)(q_off + tok) * H + kvh * r + hh) * kFaDh + ch * 8;
    cp_async16(sQ + tile_off(row, ch), src, ok);
  }
  auto load_kv = [&](int tile, int buf) {
    const int j0 = tile * kFaBN;
    const int page = pt[j0 / p.g.page_tokens];
    const int in_page = j0 % p.g.page_tokens;
    const bf16* kb = p.kv_store + p.g.offset(p.layer, page, 0, kvh, in_page);
    const bf16* vb = p.kv_store + p.g.offset(p.layer, page, 1, kvh, in_page);
    for (int i = tid; i < kFaBN * 16; i += kFaThreads) {
      const int row = i >> 4, ch = i & 15;
      const bool ok = j0 + row < S;
      cp_async16(sK + buf * kFaBN * 256 + tile_off(row, ch), kb + row * kFaDh + ch * 8, ok);
      cp_async16(sV + buf * kFaBN * 256 + tile_off(row, ch), vb + row * kFaDh + ch * 8, ok);
    }
  };
  if (t_begin < t_end) load_kv(t_begin, 0);
  cp_async_commit();

  float o[16][4];
#pragma unroll
  for (int i = 0; i < 16; ++i) { o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f; }
  float m0 = -CUDART_INF_F, m1 = -CUDART_INF_F, l0 = 0.f, l1 = 0.f;   // rows g and g+8 of this warp's 16
  uint32_t qf[8][4];
  const int wrow = warp * 16;

  for (int t = t_begin; t < t_end; ++t) {
    const int buf = (t - t_begin) & 1;
    if (t + 1 < t_end) load_kv(t + 1, buf ^ 1);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();
    if (t == t_begin) {
#pragma unroll
      for (int ks = 0; ks < 8; ++ks)
        ldsm_x4(sQ + tile_off(wrow + (lane & 7) + ((lane >> 3) & 1) * 8, ks * 2 + (lane >> 4)), qf[ks][0], qf[ks][1], qf[ks][2], qf[ks][3]);
    }
    const uint32_t kbase = sK + buf * kFaBN * 256, vbase = sV + buf * kFaBN * 256;
    // ---- S = Q K^T (16 x 64 per warp) ----
    float s[8][4];
#pragma unroll
    for (int j = 0; j < 8; ++j) { s[j][0] = s[j][1] = s[j][2] = s[j][3] = 0.f; }
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) {
#pragma unroll
      for (int jp = 0; jp < 4; ++jp) {            // pairs of 8-wide kv tiles
        uint32_t b0, b1, b2, b3;
        ldsm_x4(kbase + tile_off(jp * 16 + (lane & 7) + (lane >> 4) * 8, ks * 2 + ((lane >> 3) & 1)), b0, b1, b2, b3);
        mma_bf16_16816(s[2 * jp], qf[ks], b0, b1);
        mma_bf16_16816(s[2 * jp + 1], qf[ks], b2, b3);
      }
    }
    // ---- online softmax (log2 domain) ----
    const int j0 = t * kFaBN;
    float tm0 = -CUDART_INF_F, tm1 = -CUDART_INF_F;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int col = j0 + j * 8 + (lane & 3) * 2;
      s[j][0] = (col < S) ? s[j][0] * p.scale_log2 : -CUDART_INF_F;
      s[j][1] = (col + 1 < S) ? s[j][1] * p.scale_log2 : -CUDART_INF_F;
      s[j][2] = (col < S) ? s[j][2] * p.scale_log2 : -CUDART_INF_F;
      s[j][3] = (col + 1 < S) ? s[j][3] * p.scale_log2 : -CUDART_INF_F;
      tm0 = fmaxf(tm0, fmaxf(s[j][0], s[j][1]));
      tm1 = fmaxf(tm1, fmaxf(s[j][2], s[j][3]));
    }
    tm0 = fmaxf(tm0, __shfl_xor_sync(0xffffffffu, tm0, 1)); tm0 = fmaxf(tm0, __shfl_xor_sync(0xffffffffu, tm0, 2));
    tm1 = fmaxf(tm1, __shfl_xor_sync(0xffffffffu, tm1, 1)); tm1 = fmaxf(tm1, __shfl_xor_sync(0xffffffffu, tm1, 2));
    const float nm0 = fmaxf(m0, tm0), nm1 = fmaxf(m1, tm1);       // finite: every tile has >= 1 valid column
    const float c0 = exp2f(m0 - nm0), c1 = exp2f(m1 - nm1);
    m0 = nm0; m1 = nm1;
    float rs0 = 0.f, rs1 = 0.f;
    uint32_t pf[4][4];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const float p0 = exp2f(s[j][0] - nm0), p1 = exp2f(s[j][1] - nm0);
      const float p2 = exp2f(s[j][2] - nm1), p3 = exp2f(s[j][3] - nm1);
      rs0 += p0 + p1; rs1 += p2 + p3;
      pf[j >> 1][(j & 1) * 2 + 0] = pack_bf16(p0, p1);
      pf[j >> 1][(j & 1) * 2 + 1] = pack_bf16(p2, p3);
    }
    l0 = l0 * c0 + rs0; l1 = l1 * c1 + rs1;
#pragma unroll
    for (int i = 0; i < 16; ++i) { o[i][0] *= c0; o[i][1] *= c0; o[i][2] *= c1; o[i][3] *= c1; }
    // ---- O += P V ----
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
#pragma unroll
      for (int np = 0; np < 8; ++np) {            // pairs of 8-wide d tiles
        uint32_t b0, b1, b2, b3;
        ldsm_x4_t(vbase + tile_off(kk * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, np * 2 + (lane >> 4)), b0, b1, b2, b3);
        mma_bf16_16816(o[2 * np], pf[kk], b0, b1);
        mma_bf16_16816(o[2 * np + 1], pf[kk], b2, b3);
      }
    }
    __syncthreads();      // everyone is done with `buf` before the next prefetch overwrites it
  }
  cp_async_wait<0>();
  // ---- finish: quad-reduce the row sums, normalise (or emit a split partial) ----
  l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
  const int g = lane >> 2, tq = lane & 3;
#pragma unroll
  for (int hr = 0; hr < 2; ++hr) {
    const int rho = row0 + wrow + g + hr * 8;
    if (rho >= n_rows) continue;
    const int tok = rho / r, hh = rho % r;
    const long long orow = (long long)(q_off + tok) * H + kvh * r + hh;
    const float l = hr ? l1 : l0, m = hr ? m1 : m0;
    if (p.splits == 1) {
      const float inv = 1.f / l;
      bf16* dst = p.out + orow * kFaDh;
#pragma unroll
      for (int i = 0; i < 16; ++i)
        *reinterpret_cast<uint32_t*>(dst + i * 8 + tq * 2) = pack_bf16(o[i][hr * 2] * inv, o[i][hr * 2 + 1] * inv);
    } else {
      const long long TH = (long long)p.b.T * H;
      float* dst = p.ws_o + ((long long)split * TH + orow) * kFaDh;
#pragma unroll
      for (int i = 0; i < 16; ++i)
        *reinterpret_cast<float2*>(dst + i * 8 + tq * 2) = make_float2(o[i][hr * 2], o[i][hr * 2 + 1]);
      if (tq == 0) {
        float* ml = p.ws_ml + ((long long)split * TH + orow) * 2;
        ml[0] = (t_begin < t_end) ? m : -CUDART_INF_F;
        ml[1] = (t_begin < t_end) ? l : 0.f;
      }
    }
  }
}

// merge split partials: out = sum_s o_s 2^(m_s - m) / sum_s l_s 2^(m_s - m)
__global__ void __launch_bounds__(kFaDh) attn_combine_kernel(bf16* __restrict__ out, const float* __restrict__ ws_o,
                                                             const float* __restrict__ ws_ml, long long TH, int splits,
                                                             TraceSlot tr = TraceSlot{nullptr}) {
  DLM_PROLOGUE(tr);
  const long long row = blockIdx.x;
  const int e = threadIdx.x;
  float m = -CUDART_INF_F;
  for (int s = 0; s < splits; ++s) m = fmaxf(m, ws_ml[(s * TH + row) * 2]);
  float acc = 0.f, l = 0.f;
  for (int s = 0; s < splits; ++s) {
    const float ms = ws_ml[(s * TH + row) * 2];
    if (ms == -CUDART_INF_F) continue;
    const float w = exp2f(ms - m);
    l += ws_ml[(s * TH + row) * 2 + 1] * w;
    acc += ws_o[(s * TH + row) * kFaDh + e] * w;
  }
  out[row * kFaDh + e] = __float2bfloat16_rn(acc / l);
  DLM_EPILOGUE(tr);
}

// Host launcher.  *done = false when the shape is not supported (caller falls back to the plain kernel).
static int attn_flash_launch(bf16* out, const bf16* q, const bf16* kv_store, const int* page_table, const BatchDesc& bd,
                             const KvGeom& g, int layer, int n_heads, float scale, float** ws, size_t* ws_bytes, int num_sms,
                             cudaStream_t st, bool pdl, std::string* err, bool* done, TraceSlot tr0 = TraceSlot{nullptr},
                             TraceSlot tr1 = TraceSlot{nullptr}) {
  *done = false;
  if (g.head_dim != kFaDh || g.page_tokens % kFaBN != 0 || bd.T <= 0) return 0;
  static bool configured[kMaxDevices] = {};
  if (!configured[g_dev]) {
    cudaError_t e = cudaFuncSetAttribute(attn_flash_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kFaSmem);
    if (e != cudaSuccess) { *err = std::string("attn_flash: ") + cudaGetErrorString(e); return -4; }
    configured[g_dev] = true;
  }
  const int r = n_heads / g.n_kv_heads;
  const int q_tiles = (bd.max_q_len * r + kFaBM - 1) / kFaBM;
  const long long items = (long long)q_tiles * g.n_kv_heads * bd.n;
  const int kv_tiles = (bd.max_kv_len + kFaBN - 1) / kFaBN;
  // Split-KV when the items alone cannot fill the GPU: ~4 K/V tiles (256 positions) per CTA, between one and two CTAs per
  // SM (measured on single-request cached steps at S = 512 ... 4608: one tile per CTA is all ramp, one CTA per SM starves
  // long sequences).  No empty split.
  int splits = 1;
  if (items < 2LL * num_sms) {
    const long long lo = std::max<long long>(1, num_sms / items), hi = (2LL * num_sms + items - 1) / items;
    const int want = (int)std::min<long long>(kv_tiles, std::max(lo, std::min<long long>(hi, kv_tiles / 4)));
    const int tiles_per = (kv_tiles + want - 1) / want;
    splits = (kv_tiles + tiles_per - 1) / tiles_per;
  }
  splits = std::max(1, std::min(splits, 32));
  FaParams p;
  p.out = out; p.q = q; p.kv_store = kv_store; p.page_table = page_table; p.b = bd; p.g = g; p.layer = layer; p.n_heads = n_heads;
  p.splits = splits; p.scale_log2 = scale * 1.4426950408889634f; p.ws_o = nullptr; p.ws_ml = nullptr; p.tr = tr0;
  const long long TH = (long long)bd.T * n_heads;
  // the split-KV workspace is allocated once by the caller (captured CUDA graphs keep its address): fit the split to it
  while (splits > 1 && (size_t)splits * TH * (kFaDh + 2) * 4 > *ws_bytes) --splits;
  p.splits = splits;
  if (splits > 1) {
    p.ws_o = *ws;
    p.ws_ml = *ws + (size_t)splits * TH * kFaDh;
  }
  dim3 grid(q_tiles, g.n_kv_heads, bd.n * splits);
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.stream = st; cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  cfg.gridDim = grid; cfg.blockDim = dim3(kFaThreads); cfg.dynamicSmemBytes = kFaSmem;
  cudaError_t e = cudaLaunchKernelEx(&cfg, attn_flash_kernel, p);
  DLM_LAUNCH_CHECK();
  if (splits > 1 && e == cudaSuccess) {
    cfg.gridDim = dim3((unsigned)TH); cfg.blockDim = dim3(kFaDh); cfg.dynamicSmemBytes = 0;
    e = cudaLaunchKernelEx(&cfg, attn_combine_kernel, out, (const float*)p.ws_o, (const float*)p.ws_ml, TH, splits, tr1);
    DLM_LAUNCH_CHECK();
  }
  if (e != cudaSuccess) { *err = std::string("attn_flash launch: ") + cudaGetErrorString(e); return -4; }
  *done = true;
  return 0;
}

}  // namespace dlm
