// a5  Non-causal block attention on tcgen05 / TMEM (bf16, d_h = 128, 64-token K/V pages): the kernel the engine uses
// whenever a step has enough (request, head) work to fill the GPU -- large cached batches (HBM-bound: every K/V
// byte of a request crosses HBM once per KV head) and refresh steps (tensor-bound).
//
// Work item = (request, KV head, tile of 128 stacked query rows, KV split); query rows of the r = H / H_kv heads that
// share a KV head are stacked (row rho -> token rho / r, head rho % r).  A persistent CTA (one per SM) walks items;
// inside an item K/V is consumed in tiles of 128 tokens (two pages):
//   warp 0        TMA producer: K ring (3 x 32 KB) and V ring (2 x 32 KB) straight from the paged store through one
//                 2-D tensor map over [all page rows, 128] (box 64 x 64, SWIZZLE_128B) -- a (page, head) slice is a
//                 contiguous 16 KB run per K and per V
//   warp 1        MMA issuer: S_j = Q K_j^T (M 128, N 128, K 128) into one of two TMEM score buffers, then
//                 O += P_{j-1} V_{j-1} (V is the MN-major B operand: no transpose needed), software-pipelined so the
//                 tensor pipe always has the next QK^T queued behind the current PV
//   warp 2        TMEM allocation; loads the 128 x 128 Q tile of the next item (cp.async, manual 128-B swizzle)
//   warps 4..7    softmax: thread = query row = TMEM lane; two passes over the score row (max, then exp2 / sum / bf16
//                 P into shared memory); the running max is only raised when it grows by more than 2^8 ("lazy
//                 rescale"), in which case O is rescaled in TMEM; epilogue normalises O (or emits a split partial)
// Rows >= S of the last K/V tile hold whatever the page holds: their scores are replaced by -inf and their V rows
// are zeroed in shared memory before the PV product.
#pragma once
#include <math_constants.h>

#include "attn_flash.cuh"
#include "common.cuh"
#include "gemm_pair.cuh"
#include "ptx_sm100.cuh"

namespace dlm {

constexpr int kTaThreads = 256;
constexpr int kTaKStages = 3, kTaVStages = 2;
constexpr int kTaTile = 128;                       // query rows per item and K/V tokens per tile
constexpr int kTaTileBytes = 128 * 128 * 2;        // 32 KB: two [128 x 64] swizzled boxes
constexpr int kTaSmem = (2 + kTaKStages + kTaVStages) * kTaTileBytes + 1024 + 256;   // Q, P, K ring, V ring
constexpr float kTaRescaleThreshold = 8.f;         // log2 units

struct TaParams {
  bf16* out;                // [T, H, 128]
  const bf16* q;            // [T, H, 128]
  const int* page_table;
  BatchDesc b;
  KvGeom g;
  int layer, n_heads, splits, q_tiles_max;
  int n_items;              // n * H_kv * q_tiles_max * splits
  float scale_log2;
  float* ws_o;              // [splits, T*H, 128] (splits > 1)
  float* ws_ml;             // [splits, T*H, 2]
  unsigned long long kv_policy;
  int row_filter;           // mixed steps: 0 all requests, 1 only those with <= 64 stacked rows, 2 only those with more
  int req_lo, req_n;        // entries [req_lo, req_lo + req_n) of BatchDesc::order are this launch's requests
  int ragged_q;             // 1: items enumerate the requests' own query tiles (BatchDesc::qt_off), no empty slots for short requests
  TraceSlot tr;             // DLM_OPT_TRACE record of this launch (null: off)
};

namespace ptx {
// A from shared memory, cta_group::1; descriptors given as (lo, hi) words
__device__ __forceinline__ void umma_bf16_desc2(uint32_t tmem_d, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi, uint32_t idesc,
                                                uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\t"
      "setp.ne.b32 p, %6, 0;\n\t"
      "mov.b64 da, {%1, %2};\n\t"
      "mov.b64 db, {%3, %4};\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %5, p;\n\t}"
      ::"r"(tmem_d), "r"(a_lo), "r"(a_hi), "r"(b_lo), "r"(b_hi), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_st_32x32(uint32_t taddr, const uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]),
        "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]),
        "r"(r[30]), "r"(r[31])
      : "memory");
}
__device__ __forceinline__ float ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
}  // namespace ptx

// item -> (batch index, KV head, query tile, split).  Items are numbered request-major (each request with its own number of
// query tiles) over the requests in order of
// DECREASING K/V length (BatchDesc::order, sorted on the host) and dealt to the persistent CTAs in a snake (round k runs
// left to right for even k, right to left for odd k): longest-first + alternating direction keeps the CTAs' K/V tile totals
// within a few tiles of each other on ragged batches (plain round-robin over unsorted requests: +25 % on the slowest CTA).
struct TaItem { int bi, kvh, qt, split; };
__device__ __forceinline__ TaItem ta_item(int it, const TaParams& p) {
  TaItem r;
  r.split = it % p.splits; it /= p.splits;
  r.kvh = it % p.g.n_kv_heads; it /= p.g.n_kv_heads;
  if (p.ragged_q) {
    // `it` is a query-tile index over the launch's requests: find the request by its prefix sum (n <= a few dozen)
    const int* off = p.b.qt_off + p.req_lo;
    const int base = off[0];
    int lo = 0, hi = p.req_n;                       // off[lo] - base <= it < off[hi] - base
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (off[mid] - base <= it) lo = mid; else hi = mid;
    }
    r.qt = it - (off[lo] - base);
    r.bi = p.b.order[p.req_lo + lo];
    return r;
  }
  r.qt = it % p.q_tiles_max;
  r.bi = p.b.order[p.req_lo + it / p.q_tiles_max];
  return r;
}
// k-th item of this CTA, or -1 when it has none left
__device__ __forceinline__ int ta_sched(int k, int n_items) {
  const int G = (int)gridDim.x, base = k * G;
  if (base >= n_items) return -1;
  const int it = base + ((k & 1) ? G - 1 - (int)blockIdx.x : (int)blockIdx.x);
  return it < n_items ? it : -1;
}
// K/V tiles [t_begin, t_end) of an item; empty when the query tile is past the request's rows
__device__ __forceinline__ void ta_range(const TaItem& im, const TaParams& p, int* t_begin, int* t_end, int* n_rows, int* S) {
  const int r = p.n_heads / p.g.n_kv_heads;
  *n_rows = p.b.q_len[im.bi] * r;
  *S = p.b.kv_len[im.bi];
  const int n_tiles = (*S + kTaTile - 1) / kTaTile;
  const int per = (n_tiles + p.splits - 1) / p.splits;
  *t_begin = im.split * per;
  *t_end = min(n_tiles, *t_begin + per);
  if (im.qt * kTaTile >= *n_rows) { *t_begin = 0; *t_end = 0; }
  if ((p.row_filter == 1 && *n_rows > 64) || (p.row_filter == 2 && *n_rows <= 64)) { *t_begin = 0; *t_end = 0; *n_rows = 0; }   // the other launch's request
}

__global__ void __launch_bounds__(kTaThreads, 1) attn_tc_kernel(const __grid_constant__ CUtensorMap mapKV, const TaParams p) {
  extern __shared__ uint8_t ta_smem[];
  const uint32_t base = (ptx::smem_u32(ta_smem) + 1023u) & ~1023u;
  const uint32_t sQ = base, sP = base + kTaTileBytes;
  const uint32_t sK = sP + kTaTileBytes, sV = sK + kTaKStages * kTaTileBytes;
  const uint32_t bar = sV + kTaVStages * kTaTileBytes;
  auto k_full = [&](int s) { return bar + 8u * s; };
  auto k_empty = [&](int s) { return bar + 8u * (kTaKStages + s); };
  const uint32_t vb = bar + 16u * kTaKStages;
  auto v_full = [&](int s) { return vb + 8u * s; };
  auto v_empty = [&](int s) { return vb + 8u * (kTaVStages + s); };
  const uint32_t ob = vb + 16u * kTaVStages;
  const uint32_t q_full = ob, q_empty = ob + 8, p_full = ob + 16, pv_done = ob + 24, o_empty = ob + 32;
  auto s_full = [&](int b) { return ob + 40u + 8u * b; };
  auto s_empty = [&](int b) { return ob + 56u + 8u * b; };
  const uint32_t tmem_ptr_addr = ob + 72;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r = p.n_heads / p.g.n_kv_heads;
  const int H = p.n_heads;

  pdl_launch_dependents();
  if (threadIdx.x == 0) trace_begin(p.tr);
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&mapKV);
    for (int s = 0; s < kTaKStages; ++s) { ptx::mbar_init(k_full(s), 1); ptx::mbar_init(k_empty(s), 1); }
    for (int s = 0; s < kTaVStages; ++s) { ptx::mbar_init(v_full(s), 1); ptx::mbar_init(v_empty(s), 1); }
    ptx::mbar_init(q_full, 1); ptx::mbar_init(q_empty, 1);
    ptx::mbar_init(p_full, 128); ptx::mbar_init(pv_done, 1); ptx::mbar_init(o_empty, 128);
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(s_full(b), 1); ptx::mbar_init(s_empty(b), 128); }
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc(tmem_ptr_addr, 512);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr));
  const uint32_t tmem_o = tmem_base + 256;          // S buffers at columns 0 and 128, O at 256
  pdl_wait();                                       // q and the block's fresh K/V come from the upstream kernels
  if (threadIdx.x == 0) trace_wait(p.tr);

  if (warp == 0) {
    if (ptx::elect_one()) {        // one elected lane of the converged warp: TMA issues compile straight-line
      // ---------------- TMA producer: K ring and V ring ----------------
      int kc = 0, vc = 0;
      for (int k = 0, it; (it = ta_sched(k, p.n_items)) >= 0; ++k) {
        const TaItem im = ta_item(it, p);
        int t0, t1, n_rows, S;
        ta_range(im, p, &t0, &t1, &n_rows, &S);
        const int* pt = p.page_table + (long long)p.b.slot[im.bi] * p.g.max_pages_per_req;
        const int n_pages_req = (S + 63) >> 6;
        for (int t = t0; t < t1; ++t) {
          const int pg0 = pt[2 * t];
          const int pg1 = (2 * t + 1 < n_pages_req) ? pt[2 * t + 1] : pg0;     // second page past the end: any valid page (masked)
          const int rk0 = (int)(p.g.offset(p.layer, pg0, 0, im.kvh, 0) >> 7), rk1 = (int)(p.g.offset(p.layer, pg1, 0, im.kvh, 0) >> 7);
          const int rv0 = (int)(p.g.offset(p.layer, pg0, 1, im.kvh, 0) >> 7), rv1 = (int)(p.g.offset(p.layer, pg1, 1, im.kvh, 0) >> 7);
          {
            const int s = kc % kTaKStages;
            ptx::mbar_wait(k_empty(s), ((uint32_t)(kc / kTaKStages) & 1u) ^ 1u);
            ptx::mbar_expect_tx(k_full(s), kTaTileBytes);
            const uint32_t d = sK + s * kTaTileBytes;
            ptx::tma_load_2d(d, &mapKV, 0, rk0, k_full(s), p.kv_policy);
            ptx::tma_load_2d(d + 8192, &mapKV, 0, rk1, k_full(s), p.kv_policy);
            ptx::tma_load_2d(d + 16384, &mapKV, 64, rk0, k_full(s), p.kv_policy);
            ptx::tma_load_2d(d + 24576, &mapKV, 64, rk1, k_full(s), p.kv_policy);
            ++kc;
          }
          {
            const int s = vc % kTaVStages;
            ptx::mbar_wait(v_empty(s), ((uint32_t)(vc / kTaVStages) & 1u) ^ 1u);
            ptx::mbar_expect_tx(v_full(s), kTaTileBytes);
            const uint32_t d = sV + s * kTaTileBytes;
            ptx::tma_load_2d(d, &mapKV, 0, rv0, v_full(s), p.kv_policy);
            ptx::tma_load_2d(d + 8192, &mapKV, 0, rv1, v_full(s), p.kv_policy);
            ptx::tma_load_2d(d + 16384, &mapKV, 64, rv0, v_full(s), p.kv_policy);
            ptx::tma_load_2d(d + 24576, &mapKV, 64, rv1, v_full(s), p.kv_policy);
            ++vc;
          }
        }
      }
    }
  } else if (warp == 1) {
    // ---------------- MMA issuer (whole warp walks the loop, one elected lane issues) ----------------
    const uint32_t idesc_qk = ptx::umma_idesc_bf16(128, 128);
    const uint32_t idesc_pv = idesc_qk | (1u << 16);               // B (= V) is MN-major
    const uint32_t hi = ptx::kDescHiSw128;
    int kc = 0, vc = 0, qc = 0, sc = 0, pc = 0, oc = 0;
    auto issue_pv = [&](bool first) {
      const int s = vc % kTaVStages;
      ptx::mbar_wait(v_full(s), (uint32_t)(vc / kTaVStages) & 1u);
      ptx::mbar_wait(p_full, (uint32_t)pc & 1u);
      if (first) ptx::mbar_wait(o_empty, ((uint32_t)oc & 1u) ^ 1u);
      ptx::tc_fence_after();
      if (ptx::elect_one()) {
        const uint32_t v0 = sV + s * kTaTileBytes;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t a_lo = ptx::umma_desc_lo(sP + (kk >> 2) * 16384 + (kk & 3) * 32);
          const uint32_t b_lo = (((v0 + kk * 2048) & 0x3FFFFu) >> 4) | ((16384u >> 4) << 16);
          ptx::umma_bf16_desc2(tmem_o, a_lo, hi, b_lo, hi, idesc_pv, (first && kk == 0) ? 0u : 1u);
        }
        ptx::umma_commit(v_empty(s));
        ptx::umma_commit(pv_done);
      }
      __syncwarp();
      ++vc; ++pc;
    };
    for (int k = 0, it; (it = ta_sched(k, p.n_items)) >= 0; ++k) {
      const TaItem im = ta_item(it, p);
      int t0, t1, n_rows, S;
      ta_range(im, p, &t0, &t1, &n_rows, &S);
      const int n = t1 - t0;
      if (n <= 0) continue;
      ptx::mbar_wait(q_full, (uint32_t)qc & 1u);
      for (int j = 0; j < n; ++j) {
        const int s = kc % kTaKStages, b = sc & 1;
        ptx::mbar_wait(k_full(s), (uint32_t)(kc / kTaKStages) & 1u);
        ptx::mbar_wait(s_empty(b), ((uint32_t)(sc >> 1) & 1u) ^ 1u);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
          const uint32_t k0 = sK + s * kTaTileBytes;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint32_t off = (kk >> 2) * 16384 + (kk & 3) * 32;
            ptx::umma_bf16_desc2(tmem_base + b * 128, ptx::umma_desc_lo(sQ + off), hi, ptx::umma_desc_lo(k0 + off), hi, idesc_qk, kk ? 1u : 0u);
          }
          ptx::umma_commit(k_empty(s));
          ptx::umma_commit(s_full(b));
          if (j + 1 == n) ptx::umma_commit(q_empty);
        }
        __syncwarp();
        ++kc; ++sc;
        if (j >= 1) issue_pv(j == 1);
      }
      issue_pv(n == 1);
      ++qc; ++oc;
    }
  } else if (warp == 2) {
    // ---------------- Q loader: 128 stacked rows x 128 into two swizzled [128 x 64] boxes ----------------
    int qc = 0;
    for (int k = 0, it; (it = ta_sched(k, p.n_items)) >= 0; ++k) {
      const TaItem im = ta_item(it, p);
      int t0, t1, n_rows, S;
      ta_range(im, p, &t0, &t1, &n_rows, &S);
      if (t1 - t0 <= 0) continue;
      ptx::mbar_wait(q_empty, ((uint32_t)qc & 1u) ^ 1u);
      const int q_off = p.b.q_off[im.bi];
      for (int i = lane; i < 128 * 16; i += 32) {
        const int row = i >> 4, ch = i & 15;
        const int rho = im.qt * kTaTile + row;
        const bool ok = rho < n_rows;
        const int tok = ok ? rho / r : 0, hh = ok ? rho % r : 0;
        const bf16* src = p.q + ((long long)(q_off + tok) * H + im.kvh * r + hh) * 128 + ch * 8;
        cp_async16(sQ + (ch >> 3) * 16384 + row * 128 + (((ch & 7) ^ (row & 7)) << 4), src, ok);
      }
      cp_async_commit();
      cp_async_wait<0>();
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(q_full);
      ++qc;
    }
  } else if (warp >= 4) {
    // ---------------- softmax + epilogue (thread = stacked query row = TMEM lane) ----------------
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    const uint32_t p_row = sP + row * 128;
    const int sw = row & 7;
    int sc = 0, pc = 0;
    uint32_t rg[32];
    for (int k = 0, it; (it = ta_sched(k, p.n_items)) >= 0; ++k) {
      const TaItem im = ta_item(it, p);
      int t0, t1, n_rows, S;
      ta_range(im, p, &t0, &t1, &n_rows, &S);
      const int n = t1 - t0;
      const int rho = im.qt * kTaTile + row;
      const bool row_ok = rho < n_rows;
      const int tok = row_ok ? rho / r : 0, hh = row_ok ? rho % r : 0;
      const long long orow = (long long)(p.b.q_off[im.bi] + tok) * H + im.kvh * r + hh;
      const long long TH = (long long)p.b.T * H;
      if (n <= 0) {
        if (p.splits > 1 && row_ok) {             // empty K/V range of a valid row: a partial the combine pass ignores
          float* ml = p.ws_ml + ((long long)im.split * TH + orow) * 2;
          ml[0] = -CUDART_INF_F; ml[1] = 0.f;
        }
        continue;
      }
      const bool warp_live = im.qt * kTaTile + quarter * 32 < n_rows;     // warp-uniform: any valid row in this warp
      float m_used = -CUDART_INF_F, l = 0.f;
      for (int j = 0; j < n; ++j) {
        const int b = sc & 1;
        const int j0 = (t0 + j) * kTaTile;
        const int n_valid = min(kTaTile, S - j0);
        const uint32_t s_addr = tmem_base + lane_addr + b * 128;
        ptx::mbar_wait(s_full(b), (uint32_t)(sc >> 1) & 1u);
        ptx::tc_fence_after();
        // P_j = exp2(S_j * scale - m) in bf16, held in registers.  This is the MUFU-bound part (16 ex2 per clock per SM) and
        // it overlaps the PV product of the previous tile, which still owns the shared-memory P buffer.  After the
        // first tile the previous reference max is used speculatively (one pass over the scores, loads of the next 32
        // columns in flight while the current ones are exponentiated); only a row whose scores outgrow it by more than
        // 2^kTaRescaleThreshold takes a second pass with the new max and rescales O.
        float m_new = m_used;
        bool need = false;
        uint32_t pk[64];
        float rs = 0.f;
        if (warp_live) {
          uint32_t ra[32], rb[32];
          const bool full = n_valid == kTaTile;       // warp-uniform
          if (j == 0) {
            float mx = -CUDART_INF_F;
            ptx::tmem_ld_32x32(s_addr, ra);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              ptx::tmem_ld_wait();
              if (c < 3) ptx::tmem_ld_32x32(s_addr + (c + 1) * 32, (c & 1) ? ra : rb);
              const uint32_t(&cur)[32] = (c & 1) ? rb : ra;
#pragma unroll
              for (int i = 0; i < 32; ++i) if (full || c * 32 + i < n_valid) mx = fmaxf(mx, __uint_as_float(cur[i]));
            }
            m_new = mx * p.scale_log2;
          }
          for (int pass = 0; pass < 2; ++pass) {
            float mx = -CUDART_INF_F;
            rs = 0.f;
            ptx::tmem_ld_32x32(s_addr, ra);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              ptx::tmem_ld_wait();
              if (c < 3) ptx::tmem_ld_32x32(s_addr + (c + 1) * 32, (c & 1) ? ra : rb);
              const uint32_t(&cur)[32] = (c & 1) ? rb : ra;
              if (full) {
#pragma unroll
                for (int i = 0; i < 32; i += 2) {
                  const float s0 = __uint_as_float(cur[i]), s1 = __uint_as_float(cur[i + 1]);
                  mx = fmaxf(mx, fmaxf(s0, s1));
                  const float p0 = ptx::ex2(fmaf(s0, p.scale_log2, -m_new)), p1 = ptx::ex2(fmaf(s1, p.scale_log2, -m_new));
                  rs += p0 + p1;
                  pk[c * 16 + (i >> 1)] = pack_bf16(p0, p1);
                }
              } else {
#pragma unroll
                for (int i = 0; i < 32; i += 2) {
                  const bool v0 = c * 32 + i < n_valid, v1 = c * 32 + i + 1 < n_valid;
                  const float s0 = v0 ? __uint_as_float(cur[i]) : -CUDART_INF_F, s1 = v1 ? __uint_as_float(cur[i + 1]) : -CUDART_INF_F;
                  mx = fmaxf(mx, fmaxf(s0, s1));
                  const float p0 = v0 ? ptx::ex2(fmaf(s0, p.scale_log2, -m_new)) : 0.f, p1 = v1 ? ptx::ex2(fmaf(s1, p.scale_log2, -m_new)) : 0.f;
                  rs += p0 + p1;
                  pk[c * 16 + (i >> 1)] = pack_bf16(p0, p1);
                }
              }
            }
            mx *= p.scale_log2;
            const bool grow = j > 0 && pass == 0 && mx > m_new + kTaRescaleThreshold;
            if (grow) { m_new = mx; need = true; }
            if (!__any_sync(0xffffffffu, grow)) break;       // warp-uniform: the second pass is rare
          }
        }
        ptx::tc_fence_before();
        ptx::mbar_arrive(s_empty(b));                 // the score buffer may take S_{j+2}
        // P buffer free and O quiescent: PV of the previous tile (of this or the previous item) has completed
        ptx::mbar_wait(pv_done, ((uint32_t)pc & 1u) ^ 1u);
        ptx::tc_fence_after();
        if (warp_live) {
          if (__any_sync(0xffffffffu, need)) {
            const float corr = need ? ptx::ex2(m_used - m_new) : 1.f;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              ptx::tmem_ld_32x32(tmem_o + lane_addr + c * 32, rg);
              ptx::tmem_ld_wait();
#pragma unroll
              for (int i = 0; i < 32; ++i) rg[i] = __float_as_uint(__uint_as_float(rg[i]) * corr);
              ptx::tmem_st_32x32(tmem_o + lane_addr + c * 32, rg);
            }
            ptx::tmem_st_wait();
            l *= corr;
          }
          m_used = m_new;
          l += rs;
          // kv columns [c*32, c*32+32) of this row: box c/2, 16-byte chunks (c%2)*4 .. +4, XOR-swizzled by row%8
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const uint32_t dst = p_row + (c >> 1) * 16384;
#pragma unroll
            for (int q4 = 0; q4 < 4; ++q4) {
              const uint32_t a = dst + ((((c & 1) * 4 + q4) ^ sw) << 4);
              asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(pk[c * 16 + 4 * q4]), "r"(pk[c * 16 + 4 * q4 + 1]),
                           "r"(pk[c * 16 + 4 * q4 + 2]), "r"(pk[c * 16 + 4 * q4 + 3]) : "memory");
            }
          }
        }
        ptx::tc_fence_before();
        if (n_valid < kTaTile) {
          // last tile of the request: zero the V rows past S (0 x garbage must not reach O)
          const int vs = pc % kTaVStages;
          ptx::mbar_wait(v_full(vs), (uint32_t)(pc / kTaVStages) & 1u);
          if (row >= n_valid) {
            const uint32_t vrow = sV + vs * kTaTileBytes + row * 128;
#pragma unroll
            for (int hb = 0; hb < 2; ++hb)
#pragma unroll
              for (int q8 = 0; q8 < 8; ++q8)
                asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(vrow + hb * 16384 + q8 * 16), "r"(0u) : "memory");
          }
        }
        ptx::fence_proxy_async();
        ptx::mbar_arrive(p_full);
        ++sc; ++pc;
      }
      // ---- epilogue: O of the item is complete when the PV of its last tile has been committed ----
      ptx::mbar_wait(pv_done, ((uint32_t)pc & 1u) ^ 1u);
      ptx::tc_fence_after();
      if (warp_live) {
        const float inv = 1.f / l;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          __syncwarp();
          ptx::tmem_ld_32x32(tmem_o + lane_addr + c * 32, rg);
          ptx::tmem_ld_wait();
          if (!row_ok) {
            // padding row of the tile: nothing to store
          } else if (p.splits == 1) {
            bf16* dst = p.out + orow * 128 + c * 32;
#pragma unroll
            for (int i = 0; i < 32; i += 8) {
              uint4 v;
              v.x = pack_bf16(__uint_as_float(rg[i]) * inv, __uint_as_float(rg[i + 1]) * inv);
              v.y = pack_bf16(__uint_as_float(rg[i + 2]) * inv, __uint_as_float(rg[i + 3]) * inv);
              v.z = pack_bf16(__uint_as_float(rg[i + 4]) * inv, __uint_as_float(rg[i + 5]) * inv);
              v.w = pack_bf16(__uint_as_float(rg[i + 6]) * inv, __uint_as_float(rg[i + 7]) * inv);
              *reinterpret_cast<uint4*>(dst + i) = v;
            }
          } else {
            float* dst = p.ws_o + ((long long)im.split * TH + orow) * 128 + c * 32;
#pragma unroll
            for (int i = 0; i < 32; i += 4)
              *reinterpret_cast<float4*>(dst + i) = make_float4(__uint_as_float(rg[i]), __uint_as_float(rg[i + 1]), __uint_as_float(rg[i + 2]), __uint_as_float(rg[i + 3]));
          }
        }
        if (p.splits > 1 && row_ok) {
          float* ml = p.ws_ml + ((long long)im.split * TH + orow) * 2;
          ml[0] = m_used; ml[1] = l;
        }
      }
      ptx::tc_fence_before();
      ptx::mbar_arrive(o_empty);
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) trace_end(p.tr);
  if (warp == 2) ptx::tmem_dealloc(tmem_base, 512);
}

}  // namespace dlm
