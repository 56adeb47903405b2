// Plain CUDA kernels of the denoising step: weight generation (Definition W), embedding gather, RMSNorm,
// RoPE + paged K/V write, SIMT GEMM / attention (the all-fp32 path of config 1 and the on-device debugging
// reference of the bf16 path), SwiGLU, residual add, LM-head row statistics, combine + threshold unmask.
// Row numbers a0..a13 refer to DESIGN.md's hot-path table.
#pragma once
#include <math_constants.h>

#include "common.cuh"

namespace dlm {

// ------------------------------------------------------------------------------------------------
// Definition W: counter-based weight generation, bit-identical to the written definition.
// ------------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
#define DLM_GOLD 0x9E3779B97F4A7C15ULL

// round_bf16 (fp32 storage only): the value is rounded to bf16 first, so an fp32-activation instance (DLM_DTYPE_BF16_PRECISE)
// holds exactly the weights of the bf16 model.
template <typename TW>
__global__ void init_weight_kernel(TW* __restrict__ w, long long n, unsigned long long key, float c, int round_bf16) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long stride = (long long)gridDim.x * blockDim.x;
  for (; i < n; i += stride) {
    unsigned long long h = mix64(key + DLM_GOLD * (unsigned long long)(i + 1));
    int s = (int)(h & 0xFFFF) + (int)((h >> 16) & 0xFFFF) + (int)((h >> 32) & 0xFFFF) + (int)(h >> 48) - 131070;
    float v = __fmul_rn((float)s, c);
    if (round_bf16) v = __bfloat162float(__float2bfloat16_rn(v));
    w[i] = from_f32<TW>(v);
  }
}

// Same values into tiled storage (engine.cu make_tmap_w_tiled): element (row, col) of a [rows, cols] matrix whose first row
// sits at storage row row0 goes to tile (col / 64, row / 128); rb_pad = padded storage rows of the whole matrix / 128.  The value depends on the logical
// index row * cols + col only, so the weights are those of Definition W whatever the layout.
__host__ __device__ inline long long w_tiled_index(long long row, long long col, long long rb_pad) {
  return (((col >> 6) * rb_pad + (row >> 7)) << 13) + ((row & 127) << 6) + (col & 63);
}
template <typename TW>
__global__ void init_weight_tiled_kernel(TW* __restrict__ w, long long rows, long long cols, long long row0, long long rb_pad,
                                         unsigned long long key, float c) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long stride = (long long)gridDim.x * blockDim.x;
  const long long n = rows * cols;
  for (; i < n; i += stride) {
    unsigned long long h = mix64(key + DLM_GOLD * (unsigned long long)(i + 1));
    int s = (int)(h & 0xFFFF) + (int)((h >> 16) & 0xFFFF) + (int)((h >> 32) & 0xFFFF) + (int)(h >> 48) - 131070;
    w[w_tiled_index(row0 + i / cols, i % cols, rb_pad)] = from_f32<TW>(__fmul_rn((float)s, c));
  }
}

// RoPE table: cos/sin(pos * theta^(-2i/d_h)) computed in double, stored fp32. [max_seq, d_h/2]
__global__ void init_rope_kernel(float* __restrict__ cs, float* __restrict__ sn, int max_seq, int half, double theta) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= max_seq * half) return;
  int pos = idx / half, i = idx % half;
  double ang = (double)pos * pow(theta, -2.0 * (double)i / (double)(2 * half));
  cs[idx] = (float)cos(ang);
  sn[idx] = (float)sin(ang);
}

// ------------------------------------------------------------------------------------------------
// a1  embedding gather: x[t, :] = E[token_t, :]   (residual stream is fp32 in both paths)
// ------------------------------------------------------------------------------------------------
template <typename TW>
__global__ void embed_kernel(float* __restrict__ x, const TW* __restrict__ E, const int* __restrict__ tokens,
                             int max_seq, BatchDesc b, int d, TraceSlot tr = TraceSlot{nullptr}) {
  DLM_PROLOGUE(tr);
  int t = blockIdx.x;
  int bi = b.tok_bi[t];
  int pos = b.q_pos0[bi] + (t - b.q_off[bi]);
  int tok = tokens[(long long)b.slot[bi] * max_seq + pos];
  const TW* e = E + (long long)tok * d;
  float* xr = x + (long long)t * d;
  if (sizeof(TW) == 2 && d % 8 == 0) {           // 16-byte loads of 8 bf16
    for (int i = threadIdx.x * 8; i < d; i += blockDim.x * 8) {
      uint4 raw = *reinterpret_cast<const uint4*>(reinterpret_cast<const bf16*>(e) + i);
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&raw);
      float2 a = __bfloat1622float2(h[0]), bq = __bfloat1622float2(h[1]), cq = __bfloat1622float2(h[2]), dq = __bfloat1622float2(h[3]);
      *reinterpret_cast<float4*>(xr + i) = make_float4(a.x, a.y, bq.x, bq.y);
      *reinterpret_cast<float4*>(xr + i + 4) = make_float4(cq.x, cq.y, dq.x, dq.y);
    }
  } else {
    for (int i = threadIdx.x; i < d; i += blockDim.x) xr[i] = to_f32(e[i]);
  }
  DLM_EPILOGUE(tr);
}

// ------------------------------------------------------------------------------------------------
// a2/a7/a10  RMSNorm: u = x * rsqrt(mean(x^2) + eps), gains 1.  One block per row.  row_src (optional)
// gathers rows (a10: the block rows of each request).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float block_sum(float v, float* red) {
  v = warp_sum(v);
  int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) red[w] = v;
  __syncthreads();
  float t = (threadIdx.x < (blockDim.x >> 5)) ? red[threadIdx.x] : 0.f;
  if (w == 0) { t = warp_sum(t); if (l == 0) red[0] = t; }
  __syncthreads();
  return red[0];
}

// Split-K partials of the previous O / down projection (gemm_skinny) are folded in here, in a fixed order:
//   x[row] = ((x[row] + part[0][row]) + part[1][row]) + ... ; then u = RMSNorm(x[row]).
// One block per row, one float4 per thread per 4*blockDim chunk (d = 4096 -> 1024 threads, everything in flight at
// once: the kernel sits on the critical path between two weight-streaming GEMMs and is pure latency).
constexpr int kNormMaxChunks = 4;     // d <= 4 * 4 * 1024

template <typename TA>
__global__ void __launch_bounds__(1024) rmsnorm_kernel(TA* __restrict__ u, float* __restrict__ x, const int* __restrict__ row_src,
                                                      int d, float eps, const float* __restrict__ part, int n_part,
                                                      long long part_stride, TraceSlot tr = TraceSlot{nullptr}) {
  __shared__ float red[33];
  DLM_PROLOGUE(tr);
  const int r = blockIdx.x;
  const long long sr = row_src ? row_src[r] : r;
  float4* xr = reinterpret_cast<float4*>(x + sr * d);
  const int nvec = d >> 2;
  float4 v[kNormMaxChunks];
  float ss = 0.f;
#pragma unroll
  for (int k = 0; k < kNormMaxChunks; ++k) {
    const int i = threadIdx.x + k * blockDim.x;
    if (i < nvec) {
      float4 a = xr[i];
      if (n_part > 0) {
        const float4* pr = reinterpret_cast<const float4*>(part + sr * d) + i;
        const long long ps4 = part_stride >> 2;
        // eight slice loads in flight at a time (the kernel is one dependent L2 round trip after the other); slices are still
        // added in slice order, a slice past n_part is not read and adds an exact zero
        if (n_part > 4) {          // weight-streaming regime (8-9 slices, one chunk per thread)
          for (int s0 = 0; s0 < n_part; s0 += 8) {
            float4 q[8];
#pragma unroll
            for (int s = 0; s < 8; ++s) q[s] = s0 + s < n_part ? __ldcg(pr + (s0 + s) * ps4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int s = 0; s < 8; ++s) { a.x += q[s].x; a.y += q[s].y; a.z += q[s].z; a.w += q[s].w; }
          }
        } else {                   // CTA-pair regime (<= 4 slices, up to 4 chunks per thread): keep the register footprint small
#pragma unroll 4
          for (int s = 0; s < n_part; ++s) {
            const float4 q = __ldcg(pr + s * ps4);
            a.x += q.x; a.y += q.y; a.z += q.z; a.w += q.w;
          }
        }
        xr[i] = a;
      }
      v[k] = a;
      ss += a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w;
    }
  }
  ss = block_sum(ss, red);
  const float rs = rsqrtf(ss / (float)d + eps);
  TA* ur = u + (long long)r * d;
#pragma unroll
  for (int k = 0; k < kNormMaxChunks; ++k) {
    const int i = threadIdx.x + k * blockDim.x;
    if (i < nvec) {
      const float4 a = v[k];
      if (sizeof(TA) == 2) {
        __nv_bfloat162 lo = __floats2bfloat162_rn(a.x * rs, a.y * rs), hi = __floats2bfloat162_rn(a.z * rs, a.w * rs);
        uint2 w;
        w.x = *reinterpret_cast<uint32_t*>(&lo); w.y = *reinterpret_cast<uint32_t*>(&hi);
        *reinterpret_cast<uint2*>(reinterpret_cast<bf16*>(ur) + 4 * i) = w;
      } else {
        *reinterpret_cast<float4*>(reinterpret_cast<float*>(ur) + 4 * i) = make_float4(a.x * rs, a.y * rs, a.z * rs, a.w * rs);
      }
    }
  }
  DLM_EPILOGUE(tr);
}

// Throughput variant for large token counts (T >= 1024): one WARP per row, no block barrier, two passes (sum of
// squares while folding the split-K slices into x; then re-read x -- an L2 hit -- scale and round).  At 512..36 864 rows the
// one-block-per-row kernel above is latency-bound (~0.7 TB/s at 2048 rows); this one keeps up to 64 rows per SM in flight.
template <typename TA>
__global__ void __launch_bounds__(512) rmsnorm_rows_kernel(TA* __restrict__ u, float* __restrict__ x, const int* __restrict__ row_src,
                                                           int n_rows, int d, float eps, const float* __restrict__ part, int n_part,
                                                           long long part_stride, TraceSlot tr = TraceSlot{nullptr}) {
  DLM_PROLOGUE(tr);
  const int r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (r >= n_rows) return;
  const int lane = threadIdx.x & 31;
  const long long sr = row_src ? row_src[r] : r;
  float4* xr = reinterpret_cast<float4*>(x + sr * d);
  const int nvec = d >> 2;
  const long long ps4 = part_stride >> 2;
  float ss = 0.f;
#pragma unroll 4
  for (int i = lane; i < nvec; i += 32) {
    float4 a = xr[i];
    if (n_part > 0) {
      const float4* pr = reinterpret_cast<const float4*>(part + sr * d) + i;
      for (int s = 0; s < n_part; ++s) {
        const float4 q = __ldcg(pr + s * ps4);
        a.x += q.x; a.y += q.y; a.z += q.z; a.w += q.w;
      }
      xr[i] = a;
    }
    ss += a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w;
  }
  ss = warp_sum(ss);
  const float rs = rsqrtf(ss / (float)d + eps);
  TA* ur = u + (long long)r * d;
#pragma unroll 4
  for (int i = lane; i < nvec; i += 32) {
    const float4 a = xr[i];
    if (sizeof(TA) == 2) {
      __nv_bfloat162 lo = __floats2bfloat162_rn(a.x * rs, a.y * rs), hi = __floats2bfloat162_rn(a.z * rs, a.w * rs);
      uint2 w;
      w.x = *reinterpret_cast<uint32_t*>(&lo); w.y = *reinterpret_cast<uint32_t*>(&hi);
      *reinterpret_cast<uint2*>(reinterpret_cast<bf16*>(ur) + 4 * i) = w;
    } else {
      *reinterpret_cast<float4*>(reinterpret_cast<float*>(ur) + 4 * i) = make_float4(a.x * rs, a.y * rs, a.z * rs, a.w * rs);
    }
  }
  DLM_EPILOGUE(tr);
}

// Same result (same per-lane summation order), one pass: d <= 4096, the whole row lives in the warp's registers (32 float4 per
// lane, every load of a row issued before the first use), so x is read once and the second pass costs no memory traffic.
template <typename TA>
__global__ void __launch_bounds__(128) rmsnorm_warp_kernel(TA* __restrict__ u, float* __restrict__ x, const int* __restrict__ row_src,
                                                           int n_rows, int d, float eps, const float* __restrict__ part, int n_part,
                                                           long long part_stride, TraceSlot tr = TraceSlot{nullptr}) {
  DLM_PROLOGUE(tr);
  const int r = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (r >= n_rows) return;
  const int lane = threadIdx.x & 31;
  const long long sr = row_src ? row_src[r] : r;
  float4* xr = reinterpret_cast<float4*>(x + sr * d);
  const int nvec = d >> 2;
  float4 a[32];
#pragma unroll
  for (int k = 0; k < 32; ++k) {
    const int i = k * 32 + lane;
    a[k] = i < nvec ? xr[i] : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  if (n_part > 0) {
    const float4* pr = reinterpret_cast<const float4*>(part + sr * d);
    const long long ps4 = part_stride >> 2;
    for (int s = 0; s < n_part; ++s) {
#pragma unroll
      for (int k = 0; k < 32; ++k) {
        const int i = k * 32 + lane;
        if (i < nvec) {
          const float4 q = __ldcg(pr + s * ps4 + i);
          a[k].x += q.x; a[k].y += q.y; a[k].z += q.z; a[k].w += q.w;
        }
      }
    }
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const int i = k * 32 + lane;
      if (i < nvec) xr[i] = a[k];
    }
  }
  float ss = 0.f;
#pragma unroll
  for (int k = 0; k < 32; ++k)
    if (k * 32 + lane < nvec) ss += a[k].x * a[k].x + a[k].y * a[k].y + a[k].z * a[k].z + a[k].w * a[k].w;
  ss = warp_sum(ss);
  const float rs = rsqrtf(ss / (float)d + eps);
  TA* ur = u + (long long)r * d;
#pragma unroll
  for (int k = 0; k < 32; ++k) {
    const int i = k * 32 + lane;
    if (i >= nvec) continue;
    if (sizeof(TA) == 2) {
      __nv_bfloat162 lo = __floats2bfloat162_rn(a[k].x * rs, a[k].y * rs), hi = __floats2bfloat162_rn(a[k].z * rs, a[k].w * rs);
      uint2 w;
      w.x = *reinterpret_cast<uint32_t*>(&lo); w.y = *reinterpret_cast<uint32_t*>(&hi);
      *reinterpret_cast<uint2*>(reinterpret_cast<bf16*>(ur) + 4 * i) = w;
    } else {
      *reinterpret_cast<float4*>(reinterpret_cast<float*>(ur) + 4 * i) = make_float4(a[k].x * rs, a[k].y * rs, a[k].z * rs, a[k].w * rs);
    }
  }
  DLM_EPILOGUE(tr);
}

// x[row] += sum of split-K partials (debug-dump mode only: makes x complete right after the projection)
__global__ void add_partials_kernel(float* __restrict__ x, const float* __restrict__ part, int n_part, long long part_stride, long long n, TraceSlot tr = TraceSlot{nullptr}) {
  DLM_PROLOGUE(tr);
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float v = x[i];
  for (int s = 0; s < n_part; ++s) v += part[s * part_stride + i];
  x[i] = v;
  DLM_EPILOGUE(tr);
}

// ------------------------------------------------------------------------------------------------
// a4  RoPE + K/V write.  qkv fp32 [T, (H+2H_kv) d_h] -> q [T, H d_h] (TA), K (rotated) and V into the pages.
// Half-split pairing (i, i + d_h/2), angle = pos * theta^(-2i/d_h) from the table.  One block per token.
// ------------------------------------------------------------------------------------------------
// Grid (token, group of 256/half heads); thread = (head, pair index i): every load of the kernel is in flight at once.
template <typename TA>
__global__ void __launch_bounds__(256) rope_kv_write_kernel(TA* __restrict__ q, TA* __restrict__ kv_store, const float* __restrict__ qkv,
                                                           const float* __restrict__ rope_cos, const float* __restrict__ rope_sin,
                                                           const int* __restrict__ page_table, BatchDesc b, KvGeom g, int layer,
                                                           int n_heads, int n_part, long long part_stride, TraceSlot tr = TraceSlot{nullptr}) {
  DLM_PROLOGUE(tr);
  const int t = blockIdx.x;
  const int dh = g.head_dim, half = dh >> 1;
  const int h = blockIdx.y * (blockDim.x / half) + threadIdx.x / half;       // 0..H-1 query, then K heads, then V heads
  const int i = threadIdx.x % half;
  if (h >= n_heads + 2 * g.n_kv_heads) return;
  const int bi = b.tok_bi[t];
  const int pos = b.q_pos0[bi] + (t - b.q_off[bi]);
  const int nq = n_heads * dh, nkv = g.n_kv_heads * dh;
  const float* row = qkv + (long long)t * (nq + 2 * nkv) + (long long)h * dh;
  float a = row[i], c = row[i + half];
#pragma unroll 4
  for (int s = 1; s < n_part; ++s) { a += __ldcg(row + s * part_stride + i); c += __ldcg(row + s * part_stride + i + half); }
  if (h < n_heads + g.n_kv_heads) {               // rotate Q and K
    const float cs = rope_cos[(long long)pos * half + i], sn = rope_sin[(long long)pos * half + i];
    const float ra = a * cs - c * sn, rc = c * cs + a * sn;
    a = ra; c = rc;
  }
  TA* dst;
  if (h < n_heads) {
    dst = q + (long long)t * nq + h * dh;
  } else {
    const int page = page_table[(long long)b.slot[bi] * g.max_pages_per_req + pos / g.page_tokens];
    const int kvh = h - n_heads;
    dst = kv_store + (kvh < g.n_kv_heads ? g.offset(layer, page, 0, kvh, pos % g.page_tokens)
                                         : g.offset(layer, page, 1, kvh - g.n_kv_heads, pos % g.page_tokens));
  }
  dst[i] = from_f32<TA>(a);
  dst[i + half] = from_f32<TA>(c);
  DLM_EPILOGUE(tr);
}

// ------------------------------------------------------------------------------------------------
// a5 (plain)  attention, one block per (query token, head): softmax_j(q.k_j / sqrt(d_h)) v_j over ALL
// j in [0, S_r), no mask; K/V read from the pages (the block's own slots were just rewritten by a4).
// Scores live in dynamic shared memory ([max_kv_len] floats).
// ------------------------------------------------------------------------------------------------
template <typename TA>
__global__ void attention_plain_kernel(TA* __restrict__ out, const TA* __restrict__ q, const TA* __restrict__ kv_store,
                                       const int* __restrict__ page_table, BatchDesc b, KvGeom g, int layer,
                                       int n_heads, float scale) {
  extern __shared__ float sc[];
  __shared__ float red[33];
  __shared__ float qs[256];
  pdl_launch_dependents();
  pdl_wait();
  int t = blockIdx.x, h = blockIdx.y;
  int bi = b.tok_bi[t];
  int S = b.kv_len[bi];
  int dh = g.head_dim;
  int kvh = (h * g.n_kv_heads) / n_heads;
  const int* pt = page_table + (long long)b.slot[bi] * g.max_pages_per_req;
  const TA* qr = q + ((long long)t * n_heads + h) * dh;
  for (int e = threadIdx.x; e < dh; e += blockDim.x) qs[e] = to_f32(qr[e]);
  __syncthreads();
  float lmax = -CUDART_INF_F;
  for (int j = threadIdx.x; j < S; j += blockDim.x) {
    const TA* kr = kv_store + g.offset(layer, pt[j / g.page_tokens], 0, kvh, j % g.page_tokens);
    float s = 0.f;
    for (int e = 0; e < dh; ++e) s += qs[e] * to_f32(kr[e]);
    s *= scale;
    sc[j] = s;
    lmax = fmaxf(lmax, s);
  }
  lmax = warp_max(lmax);
  int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) red[w] = lmax;
  __syncthreads();
  float m = red[0];
  for (int i = 1; i < (int)(blockDim.x >> 5); ++i) m = fmaxf(m, red[i]);
  float lsum = 0.f;
  for (int j = threadIdx.x; j < S; j += blockDim.x) {
    float p = expf(sc[j] - m);
    sc[j] = p;
    lsum += p;
  }
  float tot = block_sum(lsum, red);
  float inv = 1.f / tot;
  for (int e = threadIdx.x; e < dh; e += blockDim.x) {
    float acc = 0.f;
    for (int j = 0; j < S; ++j) {
      const TA* vr = kv_store + g.offset(layer, pt[j / g.page_tokens], 1, kvh, j % g.page_tokens);
      acc += sc[j] * to_f32(vr[e]);
    }
    out[((long long)t * n_heads + h) * dh + e] = from_f32<TA>(acc * inv);
  }
}

// ------------------------------------------------------------------------------------------------
// a3/a6/a8/a9/a11 (plain)  C[M,N] = A[M,K] . W[N,K]^T, fp32 accumulate, fp32 out.  64x64 tile, 4x4 per thread.
// ------------------------------------------------------------------------------------------------
template <typename TA, typename TW>
__global__ void __launch_bounds__(256) gemm_plain_kernel(float* __restrict__ C, const TA* __restrict__ A,
                                                         const TW* __restrict__ W, int M, int N, int K, int lda,
                                                         int ldw, int ldc) {
  __shared__ float As[16][65];
  __shared__ float Ws[16][65];
  pdl_launch_dependents();
  pdl_wait();
  int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  int m0 = blockIdx.y * 64, n0 = blockIdx.x * 64;
  float acc[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += 16) {
    for (int i = threadIdx.x; i < 1024; i += 256) {
      int r = i >> 4, c = i & 15;
      As[c][r] = (m0 + r < M && k0 + c < K) ? to_f32(A[(long long)(m0 + r) * lda + k0 + c]) : 0.f;
      Ws[c][r] = (n0 + r < N && k0 + c < K) ? to_f32(W[(long long)(n0 + r) * ldw + k0 + c]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      float a[4], w[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = As[kk][ty * 4 + i]; w[i] = Ws[kk][tx * 4 + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], w[j], acc[i][j]);
    }
    __syncthreads();
  }
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) {
      int m = m0 + ty * 4 + i, n = n0 + tx * 4 + j;
      if (m < M && n < N) C[(long long)m * ldc + n] = acc[i][j];
    }
}

// x += y   (fp32 residual stream)
__global__ void add_residual_kernel(float* __restrict__ x, const float* __restrict__ y, long long n) {
  pdl_launch_dependents();
  pdl_wait();
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] += y[i];
}

__device__ __forceinline__ float silu_f(float g) { return g / (1.f + __expf(-g)); }

// act[t, f] = silu(gu[t, f]) * gu[t, F + f]
template <typename TA>
__global__ void swiglu_kernel(TA* __restrict__ act, const float* __restrict__ gu, int T, int F) {
  pdl_launch_dependents();
  pdl_wait();
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)T * F) return;
  int t = (int)(i / F), f = (int)(i % F);
  const float* r = gu + (long long)t * 2 * F;
  act[i] = from_f32<TA>(silu_f(r[f]) * r[F + f]);
}

// row_src[r] for a10: index into [T, d] of each block row
__global__ void build_row_src_kernel(int* __restrict__ row_src, BatchDesc b, TraceSlot tr = TraceSlot{nullptr}) {
  DLM_PROLOGUE(tr);
  int bi = blockIdx.x;
  int base = b.q_off[bi] + (b.blk_lo[bi] - b.q_pos0[bi]);
  for (int j = threadIdx.x; j < b.blk_len[bi]; j += blockDim.x) row_src[b.row_off[bi] + j] = base + j;
  DLM_EPILOGUE(tr);
}

// ------------------------------------------------------------------------------------------------
// a11 (plain)  per-row statistics of materialised logits: z = scale * logits, z[mask_id] excluded.
// Writes ONE partial (max, sum exp(z - max), argmax) per row, the format the tcgen05 epilogue writes per tile.
// ------------------------------------------------------------------------------------------------
struct RowPartial { float m, s; int idx; int pad; };

__device__ __forceinline__ void partial_merge(float& m, float& s, int& idx, float m2, float s2, int idx2) {
  // lowest index wins ties (reading G8)
  if (m2 > m || (m2 == m && idx2 < idx)) idx = idx2;
  float nm = fmaxf(m, m2);
  if (nm == -CUDART_INF_F) { s = 0.f; m = nm; return; }
  s = s * __expf(m - nm) + s2 * __expf(m2 - nm);
  m = nm;
}

__global__ void row_stats_plain_kernel(RowPartial* __restrict__ part, const float* __restrict__ logits, int V,
                                       int mask_id, float scale) {
  __shared__ float sm[32], ss[32];
  __shared__ int si[32];
  pdl_launch_dependents();
  pdl_wait();
  int r = blockIdx.x;
  const float* z = logits + (long long)r * V;
  float m = -CUDART_INF_F, s = 0.f;
  int idx = 0x7fffffff;
  for (int v = threadIdx.x; v < V; v += blockDim.x) {
    if (v == mask_id) continue;
    partial_merge(m, s, idx, z[v] * scale, 1.f, v);
  }
  for (int o = 16; o > 0; o >>= 1) {
    float m2 = __shfl_xor_sync(0xffffffffu, m, o), s2 = __shfl_xor_sync(0xffffffffu, s, o);
    int i2 = __shfl_xor_sync(0xffffffffu, idx, o);
    partial_merge(m, s, idx, m2, s2, i2);
  }
  int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { sm[w] = m; ss[w] = s; si[w] = idx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < (int)(blockDim.x >> 5); ++i) partial_merge(m, s, idx, sm[i], ss[i], si[i]);
    part[r].m = m; part[r].s = s; part[r].idx = idx; part[r].pad = 0;
  }
}

// ------------------------------------------------------------------------------------------------
// a12 + a13  combine split-vocab partials, then threshold-unmask.  One block (128 threads) per request.
//   tok = argmax_v z (lowest id on ties), lse = m + log(sum), conf = 1 / sum = exp(z_tok - lse)
//   M = MASK positions of the current block; C = {i in M : conf_i >= tau} U {argmax_{i in M} conf_i, lowest i}
//   tokens[i] = tok_i for i in C (unless dry run); commits written in ascending position.
// ------------------------------------------------------------------------------------------------
struct StepOut {              // device-side result arrays, fixed stride max_block per request
  int* n_committed;           // [n]
  int* pos;                   // [n, max_block]
  int* tok;                   // [n, max_block]
  float* conf;                // [n, max_block]
  float* row_lse;             // [n, max_block]
  float* row_conf;            // [n, max_block]
  int* row_tok;               // [n, max_block]
};

__global__ void __launch_bounds__(1024) combine_unmask_kernel(StepOut o, const RowPartial* __restrict__ part,
                                                             int n_tiles, int* __restrict__ tokens, int max_seq,
                                                             int max_block, int mask_id, BatchDesc b, int dry_run, TraceSlot tr = TraceSlot{nullptr}) {
  __shared__ float s_conf[64];
  __shared__ int s_tok[64];
  DLM_PROLOGUE(tr);
  int bi = blockIdx.x;
  int B = b.blk_len[bi];
  int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int n_warps = blockDim.x >> 5;
  for (int j = w; j < B; j += n_warps) {
    const int4* p = reinterpret_cast<const int4*>(part + (long long)(b.row_off[bi] + j) * n_tiles);
    float m = -CUDART_INF_F, s = 0.f;
    int idx = 0x7fffffff;
    int t = l;
    for (; t + 96 < n_tiles; t += 128) {          // four 16-byte loads in flight per lane
      const int4 q0 = __ldcg(p + t), q1 = __ldcg(p + t + 32), q2 = __ldcg(p + t + 64), q3 = __ldcg(p + t + 96);
      partial_merge(m, s, idx, __int_as_float(q0.x), __int_as_float(q0.y), q0.z);
      partial_merge(m, s, idx, __int_as_float(q1.x), __int_as_float(q1.y), q1.z);
      partial_merge(m, s, idx, __int_as_float(q2.x), __int_as_float(q2.y), q2.z);
      partial_merge(m, s, idx, __int_as_float(q3.x), __int_as_float(q3.y), q3.z);
    }
    for (; t < n_tiles; t += 32) {
      const int4 q0 = __ldcg(p + t);
      partial_merge(m, s, idx, __int_as_float(q0.x), __int_as_float(q0.y), q0.z);
    }
    for (int off = 16; off > 0; off >>= 1) {
      float m2 = __shfl_xor_sync(0xffffffffu, m, off), s2 = __shfl_xor_sync(0xffffffffu, s, off);
      int i2 = __shfl_xor_sync(0xffffffffu, idx, off);
      partial_merge(m, s, idx, m2, s2, i2);
    }
    if (l == 0) {
      float conf = 1.f / s;
      s_conf[j] = conf;
      s_tok[j] = idx;
      o.row_lse[bi * max_block + j] = m + logf(s);
      o.row_conf[bi * max_block + j] = conf;
      o.row_tok[bi * max_block + j] = idx;
    }
  }
  __syncthreads();
  if (w != 0) return;
  int* trow = tokens + (long long)b.slot[bi] * max_seq + b.blk_lo[bi];
  float tau = b.tau[bi];
  // best MASK position: max conf, lowest j on ties
  float bc = -1.f;
  int bj = 0x7fffffff;
  for (int j = l; j < B; j += 32)
    if (trow[j] == mask_id && (s_conf[j] > bc)) { bc = s_conf[j]; bj = j; }   // ascending j keeps the lowest on ties
  for (int off = 16; off > 0; off >>= 1) {
    float c2 = __shfl_xor_sync(0xffffffffu, bc, off);
    int j2 = __shfl_xor_sync(0xffffffffu, bj, off);
    if (c2 > bc || (c2 == bc && j2 < bj)) { bc = c2; bj = j2; }
  }
  int count = 0;
  for (int j0 = 0; j0 < B; j0 += 32) {
    int j = j0 + l;
    bool masked = (j < B) && trow[j] == mask_id;
    bool commit = masked && (s_conf[j] >= tau || j == bj);
    unsigned bal = __ballot_sync(0xffffffffu, commit);
    if (commit) {
      int k = count + __popc(bal & ((1u << l) - 1));
      o.pos[bi * max_block + k] = b.blk_lo[bi] + j;
      o.tok[bi * max_block + k] = s_tok[j];
      o.conf[bi * max_block + k] = s_conf[j];
      if (!dry_run) trow[j] = s_tok[j];
    }
    count += __popc(bal);
  }
  if (l == 0) o.n_committed[bi] = count;
  DLM_EPILOGUE(tr);
}

// ------------------------------------------------------------------------------------------------
// NEXT-1  Step Predictor confidence features ("confidence statistics", App. A; reading G22).
// conf_state[slot][pos] = the confidence the model last gave position pos while it was masked (frozen at commit, 0
// before any step evaluated it).  After the unmask: positions of the current block that were masked before the step
// take this step's row confidence; then min / q25 / median / mean / q75 over the G output positions (bitonic sort in
// shared memory, quartiles by linear interpolation between order statistics).  One block per request.
// ------------------------------------------------------------------------------------------------
constexpr int kFeatMaxGen = 2048;
__global__ void __launch_bounds__(1024) conf_features_kernel(float* __restrict__ feats, float* __restrict__ conf_state,
                                                            const int* __restrict__ tokens, int max_seq, int max_block, int mask_id,
                                                            StepOut o, BatchDesc b, const int* __restrict__ gen_lo,
                                                            const int* __restrict__ gen_len, int dry_run, TraceSlot tr = TraceSlot{nullptr}) {
  __shared__ float s[kFeatMaxGen];
  __shared__ float red[33];
  DLM_PROLOGUE(tr);
  const int bi = blockIdx.x, tid = threadIdx.x;
  const int P = gen_lo[bi], G = gen_len[bi], B = b.blk_len[bi], lo = b.blk_lo[bi];
  float* f = feats + bi * 5;
  if (G > kFeatMaxGen || G <= 0) {
    if (tid < 5) f[tid] = __int_as_float(0x7fc00000);
    return;
  }
  int n2 = 1;
  while (n2 < G) n2 <<= 1;
  const long long row = (long long)b.slot[bi] * max_seq;
  const int n_comm = B > 0 ? o.n_committed[bi] : 0;
  float part = 0.f;
  for (int j = tid; j < n2; j += blockDim.x) {
    float v = CUDART_INF_F;
    if (j < G) {
      const int pos = P + j;
      v = conf_state[row + pos];
      if (pos >= lo && pos < lo + B) {
        bool was_masked = tokens[row + pos] == mask_id;
        if (!was_masked && !dry_run)
          for (int k = 0; k < n_comm; ++k) was_masked |= o.pos[bi * max_block + k] == pos;      // committed by this very step
        if (was_masked) {
          v = o.row_conf[bi * max_block + (pos - lo)];
          if (!dry_run) conf_state[row + pos] = v;
        }
      }
      part += v;
    }
    s[j] = v;
  }
  const float total = block_sum(part, red);
  for (int k = 2; k <= n2; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = tid; i < n2; i += blockDim.x) {
        const int ixj = i ^ j;
        if (ixj > i) {
          const float a = s[i], c = s[ixj];
          const bool up = (i & k) == 0;
          if ((a > c) == up) { s[i] = c; s[ixj] = a; }
        }
      }
      __syncthreads();
    }
  }
  if (tid == 0) {
    auto quant = [&](float q) {
      const float h = (float)(G - 1) * q;
      const int l = (int)floorf(h);
      const int u = min(l + 1, G - 1);
      return s[l] + (h - (float)l) * (s[u] - s[l]);
    };
    f[0] = s[0]; f[1] = quant(0.25f); f[2] = quant(0.5f); f[3] = total / (float)G; f[4] = quant(0.75f);
  }
  DLM_EPILOGUE(tr);
}

}  // namespace dlm
