// a5  Transposed-score variant of the tcgen05 attention kernel for work items with at most 64 stacked query rows
// (cached steps of MHA models: 32 or 64 block rows per (request, head)).
//
// In attn_tc_kernel a thread owns a query row (= TMEM lane), so with 32 / 64 live rows only one / two of the four SM
// sub-partitions do the softmax -- and the softmax is MUFU-bound (one ex2 warp instruction per ~16 cycles per
// sub-partition).  Here the products are transposed:
//     S^T [128 kv, 64 q] = K_j Q^T          A = K tile (K-major), B = Q (N = 64)
//     O^T [128 d_h, 64 q] += V_j^T P_j^T    A = V tile read MN-major (no transpose), B = P^T (MN-major, 128 B per kv row)
// so a thread owns a K/V token, all four sub-partitions share the exponentials, and only the live query columns are
// exponentiated.  Softmax statistics live per COLUMN:
//   * reference m[c] = scaled score of the item's first K/V token (any real score works: the true maximum is then
//     >= the reference, so nothing underflows); a block-wide vote (bar.red.or) detects a score above m[c] + 2^16,
//     in which case exact column maxima are taken (warp shuffles + shared memory), O^T columns and the partial sums
//     are rescaled and the tile is redone;
//   * l[c] is accumulated per thread in registers over the whole item and reduced across the 128 K/V lanes once, in
//     the epilogue (62-shuffle transpose-reduce per warp + shared memory).
// Everything else (persistent items, TMA K/V rings from the paged store, split-KV partials, V rows past S zeroed)
// is as in attn_tc.cuh.
#pragma once
#include "attn_tc.cuh"

namespace dlm {

constexpr int kTtNQ = 64;                          // query columns of an item (stacked rows <= 64)
constexpr int kTtQBytes = 64 * 128 * 2;            // 16 KB: two [64 x 64] swizzled boxes
constexpr int kTtPBytes = 128 * 128;               // 16 KB: P^T, [128 kv][64 q] bf16, 128-byte rows
constexpr int kTtSmem = kTtQBytes + kTtPBytes + (kTaKStages + kTaVStages) * kTaTileBytes + 1024 + 256 + 3072;
constexpr float kTtGrowThreshold = 16.f;           // log2 units above the column reference before the exact pass

__global__ void __launch_bounds__(kTaThreads, 1) attn_tct_kernel(const __grid_constant__ CUtensorMap mapKV, const TaParams p) {
  extern __shared__ uint8_t ta_smem[];
  const uint32_t base = (ptx::smem_u32(ta_smem) + 1023u) & ~1023u;
  const uint32_t sQ = base, sP = base + kTtQBytes;
  const uint32_t sK = sP + kTtPBytes, sV = sK + kTaKStages * kTaTileBytes;
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
  // softmax scratch (generic pointers): m_ref[64], corr[64], l_fin[64], wred[4][64]
  float* scratch = reinterpret_cast<float*>(ta_smem + (bar + 256 - ptx::smem_u32(ta_smem)));
  float* m_ref = scratch; float* corr = scratch + 64; float* l_fin = scratch + 128; float* wred = scratch + 192;
  long long* orow_s = reinterpret_cast<long long*>(scratch + 448);      // [64] output row of each query column of the item

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
    ptx::tmem_alloc(tmem_ptr_addr, 256);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr));
  const uint32_t tmem_o = tmem_base + 128;          // S^T buffers at columns 0 and 64, O^T at 128
  pdl_wait();
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
    // ---------------- MMA issuer ----------------
    const uint32_t idesc_qk = ptx::umma_idesc_bf16(128, kTtNQ);                  // A = K tile, B = Q: both K-major
    const uint32_t idesc_pv = idesc_qk | (1u << 15) | (1u << 16);                // A = V^T and B = P^T: both MN-major
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
        for (int kk = 0; kk < 8; ++kk) {          // 16 K/V rows per step = two 8-row groups = 2048 bytes in both operands
          const uint32_t a_lo = (((v0 + kk * 2048) & 0x3FFFFu) >> 4) | ((16384u >> 4) << 16);   // d_h 64..127 at +16 KB
          const uint32_t b_lo = (((sP + kk * 2048) & 0x3FFFFu) >> 4) | (1u << 16);
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
            const uint32_t a_lo = ptx::umma_desc_lo(k0 + (kk >> 2) * 16384 + (kk & 3) * 32);
            const uint32_t b_lo = ptx::umma_desc_lo(sQ + (kk >> 2) * 8192 + (kk & 3) * 32);
            ptx::umma_bf16_desc2(tmem_base + b * kTtNQ, a_lo, hi, b_lo, hi, idesc_qk, kk ? 1u : 0u);
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
    // ---------------- Q loader: <= 64 stacked rows x 128 into two swizzled [64 x 64] boxes (rows past the end: zeros) ----------------
    int qc = 0;
    for (int k = 0, it; (it = ta_sched(k, p.n_items)) >= 0; ++k) {
      const TaItem im = ta_item(it, p);
      int t0, t1, n_rows, S;
      ta_range(im, p, &t0, &t1, &n_rows, &S);
      if (t1 - t0 <= 0) continue;
      ptx::mbar_wait(q_empty, ((uint32_t)qc & 1u) ^ 1u);
      const int q_off = p.b.q_off[im.bi];
      for (int i = lane; i < kTtNQ * 16; i += 32) {
        const int row = i >> 4, ch = i & 15;
        const bool ok = row < n_rows;
        const int tok = ok ? row / r : 0, hh = ok ? row % r : 0;
        const bf16* src = p.q + ((long long)(q_off + tok) * H + im.kvh * r + hh) * 128 + ch * 8;
        cp_async16(sQ + (ch >> 3) * 8192 + row * 128 + (((ch & 7) ^ (row & 7)) << 4), src, ok);
      }
      cp_async_commit();
      cp_async_wait<0>();
      ptx::fence_proxy_async();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(q_full);
      ++qc;
    }
  } else if (warp >= 4) {
    // ---------------- softmax + epilogue: thread = K/V token of the tile (S^T lane) = d_h index of O^T ----------------
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;
    const int tid = threadIdx.x - 128;                       // 0..127 among the softmax threads
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    const uint32_t pt_row = sP + row * 128;
    const int sw = row & 7;
    const float4* m4 = reinterpret_cast<const float4*>(m_ref);
    auto bar128 = [] { asm volatile("bar.sync 1, 128;" ::: "memory"); };
    auto vote_any = [](bool v) {
      uint32_t out;
      asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.u32 p, %1, 0;\n\tbar.red.or.pred q, 1, 128, p;\n\tselp.u32 %0, 1, 0, q;\n\t}" : "=r"(out) : "r"((uint32_t)v) : "memory");
      return out != 0;
    };
    int sc = 0, pc = 0;
    for (int k = 0, it; (it = ta_sched(k, p.n_items)) >= 0; ++k) {
      const TaItem im = ta_item(it, p);
      int t0, t1, n_rows, S;
      ta_range(im, p, &t0, &t1, &n_rows, &S);
      const int n = t1 - t0;
      const int nq = min(n_rows, kTtNQ);
      const int q_off = p.b.q_off[im.bi];
      const long long TH = (long long)p.b.T * H;
      auto orow_of = [&](int c) { return (long long)(q_off + c / r) * H + im.kvh * r + c % r; };
      if (n <= 0) {
        if (p.splits > 1 && tid < nq) {             // empty K/V range of a live row: a partial the combine pass ignores
          float* ml = p.ws_ml + ((long long)im.split * TH + orow_of(tid)) * 2;
          ml[0] = -CUDART_INF_F; ml[1] = 0.f;
        }
        continue;
      }
      float lsum[kTtNQ];
#pragma unroll
      for (int c = 0; c < kTtNQ; ++c) lsum[c] = 0.f;
      for (int j = 0; j < n; ++j) {
        const int b = sc & 1;
        const int n_valid = min(kTaTile, S - (t0 + j) * kTaTile);
        const bool valid = row < n_valid;
        const uint32_t s_addr = tmem_base + lane_addr + b * kTtNQ;
        ptx::mbar_wait(s_full(b), (uint32_t)(sc >> 1) & 1u);
        ptx::tc_fence_after();
        uint32_t sa[32], sb[32], pk[32];
        ptx::tmem_ld_32x32(s_addr, sa);
        if (nq > 32) ptx::tmem_ld_32x32(s_addr + 32, sb);
        ptx::tmem_ld_wait();
        if (j == 0) {                                // column references: the scores of the item's first K/V token
          if (row == 0) {
#pragma unroll
            for (int c = 0; c < 32; ++c) { m_ref[c] = __uint_as_float(sa[c]) * p.scale_log2; m_ref[32 + c] = (nq > 32) ? __uint_as_float(sb[c]) * p.scale_log2 : 0.f; }
          }
          bar128();
        }
        bool rescaled = false;
        for (int pass = 0; pass < 2; ++pass) {
          float xmax = -CUDART_INF_F;
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (h * 32 < nq) {
              const uint32_t(&sr)[32] = h ? sb : sa;
#pragma unroll
              for (int i = 0; i < 32; i += 4) {
                const float4 mm = m4[h * 8 + (i >> 2)];
                const float x0 = fmaf(__uint_as_float(sr[i]), p.scale_log2, -mm.x), x1 = fmaf(__uint_as_float(sr[i + 1]), p.scale_log2, -mm.y);
                const float x2 = fmaf(__uint_as_float(sr[i + 2]), p.scale_log2, -mm.z), x3 = fmaf(__uint_as_float(sr[i + 3]), p.scale_log2, -mm.w);
                xmax = fmaxf(fmaxf(xmax, fmaxf(x0, x1)), fmaxf(x2, x3));
                pk[h * 16 + (i >> 1)] = pack_bf16(ptx::ex2(x0), ptx::ex2(x1));
                pk[h * 16 + (i >> 1) + 1] = pack_bf16(ptx::ex2(x2), ptx::ex2(x3));
              }
            }
          }
          const bool grow = valid && pass == 0 && xmax > kTtGrowThreshold;
          if (pass == 1 || !vote_any(grow)) break;
          // ---- rare: some score outgrew its column reference: exact column maxima, rescale, redo the tile ----
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (h * 32 < nq) {
              const uint32_t(&sr)[32] = h ? sb : sa;
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                const float v = warp_max(valid ? __uint_as_float(sr[i]) * p.scale_log2 : -CUDART_INF_F);
                if (lane == 0) wred[quarter * 64 + h * 32 + i] = v;
              }
            }
          }
          bar128();
          if (tid < kTtNQ) {
            const float mo = m_ref[tid];
            float mn = mo;
            if (tid < ((nq + 31) & ~31)) mn = fmaxf(fmaxf(mo, fmaxf(wred[tid], wred[64 + tid])), fmaxf(wred[128 + tid], wred[192 + tid]));
            corr[tid] = ptx::ex2(mo - mn);
            m_ref[tid] = mn;
          }
          bar128();
#pragma unroll
          for (int c = 0; c < kTtNQ; ++c) lsum[c] *= corr[c];
          rescaled = true;
        }
        ptx::tc_fence_before();
        ptx::mbar_arrive(s_empty(b));                 // the score buffer may take S^T_{j+2}
        // P^T buffer free and O^T quiescent: PV of the previous tile (of this or the previous item) has completed
        ptx::mbar_wait(pv_done, ((uint32_t)pc & 1u) ^ 1u);
        ptx::tc_fence_after();
        if (rescaled && j > 0) {                      // block-uniform
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            uint32_t o[32];
            ptx::tmem_ld_32x32(tmem_o + lane_addr + h * 32, o);
            ptx::tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * corr[h * 32 + i]);
            ptx::tmem_st_32x32(tmem_o + lane_addr + h * 32, o);
          }
          ptx::tmem_st_wait();
        }
        // the row's weights: zero past S; partial sums taken from the bf16 values the MMA will see
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          if (h * 32 < nq) {
#pragma unroll
            for (int k = 0; k < 16; ++k) {
              const uint32_t w = valid ? pk[h * 16 + k] : 0u;
              pk[h * 16 + k] = w;
              lsum[h * 32 + 2 * k] += __uint_as_float(w << 16);
              lsum[h * 32 + 2 * k + 1] += __uint_as_float(w & 0xffff0000u);
            }
#pragma unroll
            for (int q4 = 0; q4 < 4; ++q4) {
              const uint32_t a = pt_row + (((h * 4 + q4) ^ sw) << 4);
              asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(pk[h * 16 + 4 * q4]), "r"(pk[h * 16 + 4 * q4 + 1]),
                           "r"(pk[h * 16 + 4 * q4 + 2]), "r"(pk[h * 16 + 4 * q4 + 3]) : "memory");
            }
          }
        }
        ptx::tc_fence_before();
        if (n_valid < kTaTile) {
          // last tile of the request: zero the V rows past S (0 x garbage must not reach O^T)
          const int vs = pc % kTaVStages;
          ptx::mbar_wait(v_full(vs), (uint32_t)(pc / kTaVStages) & 1u);
          if (!valid) {
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
      // ---- epilogue: O^T of the item is complete when the PV of its last tile has been committed ----
      // l[c] = sum over the 128 K/V lanes of the per-thread partial sums: transpose-reduce inside the warp (62 shuffles,
      // lane ends up with columns 2*lane and 2*lane+1), then across the four warps through shared memory
#pragma unroll
      for (int ofs = 16, cnt = kTtNQ; ofs >= 1; ofs >>= 1, cnt >>= 1) {
        const bool up = (lane & ofs) != 0;
#pragma unroll
        for (int i = 0; i < cnt / 2; ++i) {
          const float keep = up ? lsum[i + cnt / 2] : lsum[i];
          const float send = up ? lsum[i] : lsum[i + cnt / 2];
          lsum[i] = keep + __shfl_xor_sync(0xffffffffu, send, ofs);
        }
      }
      wred[quarter * 64 + 2 * lane] = lsum[0];
      wred[quarter * 64 + 2 * lane + 1] = lsum[1];
      bar128();
      if (tid < kTtNQ) {
        const float l = (wred[tid] + wred[64 + tid]) + (wred[128 + tid] + wred[192 + tid]);
        l_fin[tid] = l;
        corr[tid] = 1.f / l;                          // corr[] doubles as 1 / l in the epilogue
        orow_s[tid] = orow_of(min(tid, max(nq - 1, 0)));
      }
      bar128();
      ptx::mbar_wait(pv_done, ((uint32_t)pc & 1u) ^ 1u);
      ptx::tc_fence_after();
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (h * 32 < nq) {                             // warp-uniform
          uint32_t o[32];
          ptx::tmem_ld_32x32(tmem_o + lane_addr + h * 32, o);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const int c = h * 32 + i;
            if (c < nq) {
              const long long orow = orow_s[c];
              if (p.splits == 1) p.out[orow * 128 + row] = __float2bfloat16_rn(__uint_as_float(o[i]) * corr[c]);
              else p.ws_o[((long long)im.split * TH + orow) * 128 + row] = __uint_as_float(o[i]);
            }
          }
        }
      }
      if (p.splits > 1 && tid < nq) {
        float* ml = p.ws_ml + ((long long)im.split * TH + orow_s[tid]) * 2;
        ml[0] = m_ref[tid]; ml[1] = l_fin[tid];
      }
      ptx::tc_fence_before();
      ptx::mbar_arrive(o_empty);
      bar128();                                        // the scratch arrays are rewritten by the next item
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) trace_end(p.tr);
  if (warp == 2) ptx::tmem_dealloc(tmem_base, 256);
}

}  // namespace dlm
