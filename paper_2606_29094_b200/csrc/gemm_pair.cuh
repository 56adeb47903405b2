// Persistent CTA-pair tcgen05 GEMM for M > 128 tokens (refresh steps, large cached batches):
//   D[M, N] = A[M, K] . W[N, K]^T, bf16 in, fp32 accumulation in tensor memory.  Rows a3, a6, a8, a9, a11 of DESIGN.md.
//
// A cluster of two CTAs (one TPC) owns a 256 x BN output tile: tcgen05.mma.cta_group::2 with M = 256, N = BN.
// Each CTA stages its own 128 rows of A and its own BN/2 rows of W per 64-wide K block, so every operand byte is
// fetched once per CTA pair (half the L2 -> SM traffic of two independent 128 x BN tiles).  The accumulator is
// double buffered in TMEM (2 x 256 columns): the epilogue warps drain tile i while the MMAs of tile i+1 run.
//   warp 0      TMA producer (one lane): `stages`-deep ring, completion of BOTH CTAs' boxes counted on the leader's
//               full[stage] barrier (cp.async.bulk.tensor ... cta_group::2)
//   warp 1      TMEM allocation (both CTAs); in the leader one lane issues 4 x UMMA (256 x BN x 16) per K block,
//               tcgen05.commit multicast to both CTAs frees the stage / publishes the accumulator
//   warps 2..5  epilogue: tcgen05.ld (lane = row, 32 columns at a time) + the fused epilogue (fp32 | bf16 |
//               residual add | SwiGLU | LM-head split-vocab statistics), then a remote arrive on the leader's
//               tmem_empty barrier
// Tiles are walked persistently (grid = one pair per TPC) in panels of `panel` m-tiles so that a wave shares its A
// panel and a few W tiles through L2.  A launch may mix two tile widths (GemmPairParams::bn2): the leading column blocks
// are BN wide, the rest narrower, so that with few row tiles the pairs' last tiles form a full wave of cheap tiles.
// SwiGLU: the leader CTA stages gate rows, its peer the matching up rows, so accumulator columns [0, BN/2) are
// the gate and [BN/2, BN) the up projection of the same BN/2 features.
#pragma once
#include "attn_flash.cuh"
#include "common.cuh"
#include "gemm_tc.cuh"
#include "kernels_basic.cuh"
#include "ptx_sm100.cuh"

namespace dlm {

// EPI_ROPE (a3 + a4 fused): the QKV projection's epilogue rotates Q and K (half-split pairs, table lookup by absolute
// position), rounds to bf16 and writes Q to [T, H, 128] and K / V straight into the request's pages.
constexpr int EPI_ROPE = 5;
struct RopeEpi {
  bf16* q;
  bf16* kv_store;
  const float* rope_cos;   // [max_seq, 64]
  const float* rope_sin;
  const int* page_table;
  BatchDesc b;
  KvGeom g;
  int layer, n_heads;
};

struct GemmPairParams {
  int M, N, K;        // N = output features (SwiGLU: F; a tile covers bn/2 of them)
  int bn;             // MMA N of the pair tile: multiple of 32 (SwiGLU: 64) in [64, 256]
  int bn2, n_tiles_a; // mixed widths (bn2 > 0): the first n_tiles_a column blocks are bn wide, the rest bn2 < bn wide, so that the
                      // last wave of a launch with few row tiles is a wave of narrower, cheaper tiles instead of a partly filled one
  int stages;
  int up_row0;        // SwiGLU: first row of the up projection inside W (= F)
  int m_tiles, n_tiles_n, panel;
  int splits, kb_per_split;      // split-K (EPI_F32 only): unit = (tile, K range); split s writes slice out_f32 + s * split_stride
  long long split_stride;
  float* out_f32;     // EPI_F32 / EPI_RESID
  bf16* out_bf16;     // EPI_BF16 / EPI_SWIGLU
  long long ldc;
  RowPartial* part;   // EPI_LMHEAD: [M, n_tiles]
  int n_tiles;        // row pitch of `part`
  int mask_id;
  float scale;
  unsigned long long w_policy, a_policy;
  RopeEpi rope;       // EPI_ROPE
  TraceSlot tr;       // DLM_OPT_TRACE record of this launch (null: off)
};

constexpr int kPairThreads = 192;
constexpr int kPairAccCols = 256;       // TMEM columns per accumulator stage

// A ring stage holds kPairKbPerStage 64-wide K blocks: [A k0][A k1][W k0][W k1] (A 128 x 64, W (bn/2) x 64 per block).  Every
// stage hand-off (full-barrier wait, fence, election, commits in the issuing warp; empty-barrier wait and TMA issue in the
// producer) costs a few hundred cycles whatever the tile width (DESIGN.md section 6 (1)); with two K blocks per hand-off
// (eight straight-line MMAs) a 192- or 128-wide tile costs 0.78 / 0.61 of a 256-wide one instead of ~1.
constexpr int kPairKbPerStage = 2;
__host__ __device__ inline int gemm_pair_kb_bytes(int bn) { return kATileBytes + bn * 64; }
__host__ __device__ inline int gemm_pair_stage_bytes(int bn) { return kPairKbPerStage * gemm_pair_kb_bytes(bn); }
constexpr int kPairEpiStageBytes = 4 * 2 * 4096;      // per epilogue warp: two swizzled 32 x 32 fp32 tiles (coalescing stage)
__host__ inline int gemm_pair_smem_bytes(int bn, int stages) { return stages * gemm_pair_stage_bytes(bn) + 1024 + 1024 + kPairEpiStageBytes; }

namespace ptx {
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_id_x() { uint32_t r; asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t n_clusters_x() { uint32_t r; asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cta address -> shared::cluster address of the same offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// 2-D tile load into this CTA's shared memory; the bytes are counted on an mbarrier that may live in the peer CTA.
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst_smem, const void* tmap, int c0, int c1, uint32_t bar_cluster,
                                                 uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%3, %4}], [%2], %5;"
      ::"r"(dst_smem), "l"(tmap), "r"(bar_cluster), "r"(c0), "r"(c1), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tmem_alloc_pair(uint32_t dst_smem, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish_pair() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void umma_bf16_pair(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_bf16_pair_lo(uint32_t tmem_d, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "mov.b64 da, {%1, %5};\n\t"
      "mov.b64 db, {%2, %5};\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], da, db, %3, p;\n\t}"
      ::"r"(tmem_d), "r"(a_lo), "r"(b_lo), "r"(idesc), "r"(accumulate), "r"(kDescHiSw128)
      : "memory");
}
// Bulk tensor store / reduce-add of one shared-memory box to global memory (async proxy, bulk-group completion).
__device__ __forceinline__ void tma_store_3d(const void* tmap, uint32_t src_smem, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"(tmap), "r"(src_smem), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_reduce_add_3d(const void* tmap, uint32_t src_smem, int c0, int c1, int c2) {
  asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"(tmap), "r"(src_smem), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }
// arrive (once) on the barrier at this shared-memory offset in BOTH CTAs of the pair when the MMAs issued so far are done
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"((uint16_t)3)
               : "memory");
}
}  // namespace ptx

struct PairTile { int m_blk, n_blk; };
__device__ __forceinline__ PairTile pair_tile(int t, int m_tiles, int n_tiles, int panel) {
  const int pw = panel * n_tiles;
  const int pid = t / pw, rem = t - pid * pw;
  const int m_base = pid * panel;
  const int ph = min(panel, m_tiles - m_base);
  PairTile r;
  r.n_blk = rem / ph;
  r.m_blk = m_base + rem - r.n_blk * ph;
  return r;
}

// width and first output column (SwiGLU: first feature) of column block n_blk
struct PairCols { int bn, n0; };
template <int EPI>
__device__ __forceinline__ PairCols pair_cols(int n_blk, const GemmPairParams& p) {
  PairCols c;
  const int per1 = EPI == EPI_SWIGLU ? p.bn / 2 : p.bn;
  if (p.bn2 <= 0 || n_blk < p.n_tiles_a) { c.bn = p.bn; c.n0 = n_blk * per1; return c; }
  const int per2 = EPI == EPI_SWIGLU ? p.bn2 / 2 : p.bn2;
  c.bn = p.bn2; c.n0 = p.n_tiles_a * per1 + (n_blk - p.n_tiles_a) * per2;
  return c;
}

template <int EPI>
__global__ void __launch_bounds__(kPairThreads, 1)
gemm_pair_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const __grid_constant__ CUtensorMap mapC,
                 const GemmPairParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const int BN = p.bn;
  const int stages = p.stages;
  const uint32_t stage_bytes = gemm_pair_stage_bytes(BN);
  const uint32_t bar_base = base + stages * stage_bytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };                    // used in the leader
  auto empty_bar = [&](int s) { return bar_base + 8u * (stages + s); };        // per CTA (multicast commit)
  const uint32_t tmem_full_bar = bar_base + 16u * stages;                      // [2], per CTA (multicast commit)
  const uint32_t tmem_empty_bar = tmem_full_bar + 16u;                         // [2], used in the leader
  const uint32_t tmem_ptr_addr = tmem_empty_bar + 16u;
  const uint32_t epi_stage = bar_base + 1024u;                                 // kPairEpiStageBytes, 1024-byte aligned (TMA 128-byte swizzle)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank();
  const bool leader = rank == 0;
  const int cluster = (int)ptx::cluster_id_x(), n_clusters = (int)ptx::n_clusters_x();
  const int num_kb = (p.K + kBK - 1) / kBK;
  const int total_tiles = p.m_tiles * p.n_tiles_n;
  const int total_units = total_tiles * p.splits;      // unit u: tile u % total_tiles, K split u / total_tiles

  ptx::pdl_launch_dependents();
  if (threadIdx.x == 0) trace_begin(p.tr);
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&mapA);
    ptx::prefetch_tmap(&mapB);
    for (int s = 0; s < stages; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; ++a) { ptx::mbar_init(tmem_full_bar + 8u * a, 1); ptx::mbar_init(tmem_empty_bar + 8u * a, 8); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) {
    ptx::tmem_alloc_pair(tmem_ptr_addr, 512);
    ptx::tmem_relinquish_pair();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::cluster_sync();          // the peer's barriers exist before anything is signalled across the pair
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr));

  if (warp == 0) {
    if (ptx::elect_one()) {        // one elected lane of the converged warp: TMA issues compile straight-line
      // ---------------- TMA producer (both CTAs, one lane) ----------------
      const uint32_t half_rows = (uint32_t)BN / 2;
      const uint32_t w_bytes = half_rows * 128u;
      const uint32_t tx_kb = 2u * (kATileBytes + w_bytes);          // both CTAs' bytes of one K block
      // the box is always BN / 2 rows (one tensor map); a narrower tile uses the first bn_t / 2 of them
      auto w_row_of = [&](const PairTile& tl) {
        const PairCols pc = pair_cols<EPI>(tl.n_blk, p);
        if (EPI == EPI_SWIGLU) return pc.n0 + (leader ? 0 : p.up_row0);
        return pc.n0 + (int)rank * (pc.bn / 2);
      };
      auto load_w = [&](uint32_t sa, int kb_abs, int cnt, int w_row, uint32_t fb) {
        for (int h = 0; h < cnt; ++h)
          ptx::tma_load_2d_pair(sa + kPairKbPerStage * kATileBytes + h * w_bytes, &mapB, (kb_abs + h) * kBK, w_row, fb, p.w_policy);
      };
      auto load_a = [&](uint32_t sa, int kb_abs, int cnt, int m0, uint32_t fb) {
        for (int h = 0; h < cnt; ++h)
          ptx::tma_load_2d_pair(sa + h * kATileBytes, &mapA, (kb_abs + h) * kBK, m0, fb, p.a_policy);
      };
      // Ring fill of the first tile: weights do not depend on the upstream kernel, so their boxes are issued
      // before the programmatic-dependency wait; A follows once the producer of A has finished.
      int pre = 0;
      if (cluster < total_units) {
        const PairTile tl = pair_tile(cluster % total_tiles, p.m_tiles, p.n_tiles_n, p.panel);
        const int m0 = tl.m_blk * 256 + (int)rank * 128, w_row = w_row_of(tl);
        const int kb0 = (cluster / total_tiles) * p.kb_per_split;
        const int nkb = min(p.kb_per_split, num_kb - kb0);
        pre = min(stages, (nkb + kPairKbPerStage - 1) / kPairKbPerStage);
        for (int st = 0; st < pre; ++st) {
          const int cnt = min(kPairKbPerStage, nkb - st * kPairKbPerStage);
          if (leader) ptx::mbar_expect_tx(full_bar(st), tx_kb * cnt);
          load_w(base + st * stage_bytes, kb0 + st * kPairKbPerStage, cnt, w_row, ptx::mapa(full_bar(st), 0));
        }
        ptx::pdl_wait();
        trace_wait(p.tr);
        for (int st = 0; st < pre; ++st)
          load_a(base + st * stage_bytes, kb0 + st * kPairKbPerStage, min(kPairKbPerStage, nkb - st * kPairKbPerStage), m0, ptx::mapa(full_bar(st), 0));
      } else {
        ptx::pdl_wait();
        trace_wait(p.tr);
      }
      // ring position kept as running (stage, phase) counters: `it % stages` with a run-time divisor is a ~30-instruction
      // sequence with a MUFU in the middle, once per stage on the critical path of the pipeline
      int it = 0, s = 0;
      uint32_t ph = 0;
      for (int u = cluster; u < total_units; u += n_clusters) {
        const PairTile tl = pair_tile(u % total_tiles, p.m_tiles, p.n_tiles_n, p.panel);
        const int m0 = tl.m_blk * 256 + (int)rank * 128, w_row = w_row_of(tl);
        const int kb0 = (u / total_tiles) * p.kb_per_split;
        const int nkb = min(p.kb_per_split, num_kb - kb0);
        for (int kb = 0; kb < nkb; kb += kPairKbPerStage, ++it, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1u : 0u)) {
          if (it < pre) continue;                       // issued by the ring fill above
          const int cnt = min(kPairKbPerStage, nkb - kb);
          ptx::mbar_wait(empty_bar(s), ph ^ 1u);
          const uint32_t fb = ptx::mapa(full_bar(s), 0);
          if (leader) ptx::mbar_expect_tx(full_bar(s), tx_kb * cnt);
          const uint32_t sa = base + s * stage_bytes;
          load_w(sa, kb0 + kb, cnt, w_row, fb);
          load_a(sa, kb0 + kb, cnt, m0, fb);
        }
      }
    }
  } else if (warp == 1) {
    if (leader) {
      // ---------------- MMA issuer (leader CTA; the whole warp walks the loop, one elected lane issues) ----------------
      int i = 0, s = 0;
      uint32_t ph = 0;
      for (int u = cluster; u < total_units; u += n_clusters, ++i) {
        const uint32_t idesc = ptx::umma_idesc_bf16(256, pair_cols<EPI>(pair_tile(u % total_tiles, p.m_tiles, p.n_tiles_n, p.panel).n_blk, p).bn);
        const uint32_t as = (uint32_t)i & 1u, aph = ((uint32_t)i >> 1) & 1u;
        ptx::mbar_wait(tmem_empty_bar + 8u * as, aph ^ 1u);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * kPairAccCols;
        const int nkb = min(p.kb_per_split, num_kb - (u / total_tiles) * p.kb_per_split);
        const uint32_t w_bytes = (uint32_t)BN * 64u;
        for (int kb = 0; kb < nkb; kb += kPairKbPerStage, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1u : 0u)) {
          const int cnt = min(kPairKbPerStage, nkb - kb);
          ptx::mbar_wait(full_bar(s), ph);
          ptx::tc_fence_after();
          if (ptx::elect_one()) {
            const uint32_t sa = base + s * stage_bytes;
            const uint32_t a_lo = ptx::umma_desc_lo(sa), b_lo = ptx::umma_desc_lo(sa + kPairKbPerStage * kATileBytes);
            const uint32_t a_step = kATileBytes >> 4, b_step = w_bytes >> 4;      // next K block, in encoded (16-byte) units
            if (cnt == kPairKbPerStage) {                 // the common case, straight-line
#pragma unroll
              for (int h = 0; h < kPairKbPerStage; ++h)
#pragma unroll
                for (int k = 0; k < kBK / 16; ++k)    // +32 bytes along K inside the 128-byte swizzle row = +2 in the encoded address
                  ptx::umma_bf16_pair_lo(d_tmem, a_lo + h * a_step + 2 * k, b_lo + h * b_step + 2 * k, idesc, (kb | h | k) != 0 ? 1u : 0u);
            } else {
              for (int h = 0; h < cnt; ++h)
#pragma unroll
                for (int k = 0; k < kBK / 16; ++k)
                  ptx::umma_bf16_pair_lo(d_tmem, a_lo + h * a_step + 2 * k, b_lo + h * b_step + 2 * k, idesc, (kb | h | k) != 0 ? 1u : 0u);
            }
            ptx::umma_commit_pair(empty_bar(s));          // both CTAs' producers may refill the stage
            if (kb + cnt == nkb) ptx::umma_commit_pair(tmem_full_bar + 8u * as);   // accumulator complete in both CTAs' TMEM
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ---------------- epilogue (warps 2..5 of both CTAs; TMEM lane quarter = warp % 4) ----------------
    const int quarter = warp & 3;
    const uint32_t te_leader = ptx::mapa(tmem_empty_bar, 0);
    int i = 0;
    for (int u = cluster; u < total_units; u += n_clusters, ++i) {
      const PairTile tl = pair_tile(u % total_tiles, p.m_tiles, p.n_tiles_n, p.panel);
      const PairCols pc = pair_cols<EPI>(tl.n_blk, p);
      const int BNt = pc.bn;                              // this tile's width (== BN unless the launch mixes two widths)
      const uint32_t as = (uint32_t)i & 1u, aph = ((uint32_t)i >> 1) & 1u;
      const int row = tl.m_blk * 256 + (int)rank * 128 + quarter * 32 + lane;
      const bool row_ok = row < p.M;
      ptx::mbar_wait(tmem_full_bar + 8u * as, aph);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + as * kPairAccCols;
      uint32_t r[32];
      // Coalescing stage: a thread owns an accumulator ROW (TMEM lane), but a warp-wide global access should cover whole
      // 128-byte lines.  Each 32 x 32 fp32 chunk goes through a swizzled 4 KB shared-memory tile and comes back
      // transposed: in access i lane l holds 4 columns (l % 8) of row 4 i + l / 8, so one instruction touches 4 full lines
      // instead of 32 partial ones (measured: 1470 -> ~250 cycles per chunk, the exposed epilogue of a one-wave GEMM).
      const uint32_t stg = epi_stage + (uint32_t)(warp - 2) * 8192u;
      auto stg_write = [&](int buf, const uint32_t (&v)[32]) {
#pragma unroll
        for (int jq = 0; jq < 8; ++jq)
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(stg + buf * 4096 + lane * 128 + ((jq ^ (lane & 7)) << 4)), "r"(v[4 * jq]),
                       "r"(v[4 * jq + 1]), "r"(v[4 * jq + 2]), "r"(v[4 * jq + 3]) : "memory");
      };
      auto stg_read = [&](int buf, int i) {
        const int rr = 4 * i + (lane >> 3), jj = lane & 7;
        float4 v;
        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                     : "r"(stg + buf * 4096 + rr * 128 + ((jj ^ (rr & 7)) << 4)) : "memory");
        return v;
      };
      const int row_w0 = tl.m_blk * 256 + (int)rank * 128 + quarter * 32;       // first row of this warp's quarter
      const int t_rr = lane >> 3, t_c4 = (lane & 7) * 4;                         // transposed view: row 4 i + t_rr, columns t_c4 .. t_c4 + 3
      if (EPI == EPI_F32 || EPI == EPI_RESID) {
        // fp32 outputs leave through TMA: the chunk is staged (swizzled as the output map expects) and one lane issues a bulk
        // tensor store -- or, for the residual stream, a bulk REDUCE-ADD (x += acc happens in L2: no read of x by the SM, and
        // exactly one add per element, so the result is deterministic).  TMA clips rows >= M and columns >= N.
        const int n0 = pc.n0, nch = BNt / 32;
        for (int c = 0; c < nch; ++c) {
          const int b = c & 1;
          if (c >= 2) {                                                            // the bulk op that last read this buffer
            if (lane == 0) ptx::bulk_wait_read<1>();
          }
          __syncwarp();
          ptx::tmem_ld_32x32(taddr + c * 32, r);
          ptx::tmem_ld_wait();
          stg_write(b, r);
          ptx::fence_proxy_async();
          __syncwarp();
          if (lane == 0 && n0 + c * 32 < p.N && row_w0 < p.M) {
            if (EPI == EPI_RESID) ptx::tma_reduce_add_3d(&mapC, stg + b * 4096, n0 + c * 32, row_w0, 0);
            else ptx::tma_store_3d(&mapC, stg + b * 4096, n0 + c * 32, row_w0, u / total_tiles);
          }
          if (lane == 0) ptx::bulk_commit();
        }
        if (lane == 0) ptx::bulk_wait_read<0>();                                   // the stage is reused by the next tile
        __syncwarp();
      } else if (EPI == EPI_BF16) {
        const int n0 = pc.n0, nch = BNt / 32;
        const long long obase = (long long)(row_w0 + t_rr) * p.ldc + n0 + t_c4;   // transposed view, hoisted
        for (int c = 0; c < nch; ++c) {
          __syncwarp();
          ptx::tmem_ld_32x32(taddr + c * 32, r);
          ptx::tmem_ld_wait();
          stg_write(0, r);
          __syncwarp();
          const int col0 = n0 + c * 32;
          float4 v[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) v[i] = stg_read(0, i);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int grow = row_w0 + 4 * i + t_rr;
            if (grow >= p.M || col0 + t_c4 >= p.N) continue;
            bf16* o = p.out_bf16 + obase + (long long)i * 4 * p.ldc + c * 32;
            if (col0 + t_c4 + 4 <= p.N) {
              *reinterpret_cast<uint2*>(o) = make_uint2(pack_bf16(v[i].x, v[i].y), pack_bf16(v[i].z, v[i].w));
            } else {
              const float e[4] = {v[i].x, v[i].y, v[i].z, v[i].w};
              for (int q = 0; q < 4; ++q) if (col0 + t_c4 + q < p.N) o[q] = __float2bfloat16_rn(e[q]);
            }
          }
        }
      } else if (EPI == EPI_SWIGLU) {
        const int half = BNt / 2;
        const int f0 = pc.n0;
        uint32_t u2[32];
        for (int c = 0; c < half / 32; ++c) {
          __syncwarp();
          ptx::tmem_ld_32x32(taddr + c * 32, r);
          ptx::tmem_ld_32x32(taddr + half + c * 32, u2);
          ptx::tmem_ld_wait();
          stg_write(0, r);
          stg_write(1, u2);
          __syncwarp();
          const int fc = f0 + c * 32;
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int grow = row_w0 + 4 * i + t_rr;
            const float4 g = stg_read(0, i), w = stg_read(1, i);
            if (grow >= p.M || fc + t_c4 >= p.N) continue;
            const float e[4] = {silu_f(g.x) * w.x, silu_f(g.y) * w.y, silu_f(g.z) * w.z, silu_f(g.w) * w.w};
            bf16* o = p.out_bf16 + (long long)grow * p.ldc + fc + t_c4;
            if (fc + t_c4 + 4 <= p.N) {
              *reinterpret_cast<uint2*>(o) = make_uint2(pack_bf16(e[0], e[1]), pack_bf16(e[2], e[3]));
            } else {
              for (int q = 0; q < 4; ++q) if (fc + t_c4 + q < p.N) o[q] = __float2bfloat16_rn(e[q]);
            }
          }
        }
      } else if (EPI == EPI_ROPE) {
        // tile = BN / 128 whole heads of 128 columns (BN = 256 or 128); pairs (i, i + 64) live in chunks (a, a + 2) of a head
        const RopeEpi& e = p.rope;
        int pos = 0, page = 0, slot_in_page = 0;
        if (row_ok) {
          const int bi = e.b.tok_bi[row];
          pos = e.b.q_pos0[bi] + (row - e.b.q_off[bi]);
          page = e.page_table[(long long)e.b.slot[bi] * e.g.max_pages_per_req + pos / e.g.page_tokens];
          slot_in_page = pos % e.g.page_tokens;
        }
        uint32_t u2[32];
#pragma unroll 1
        for (int hh = 0; hh < (BNt >> 7); ++hh) {
          const int hg = (pc.n0 >> 7) + hh;             // global head index: Q heads, then K heads, then V heads
          const bool head_ok = hg < e.n_heads + 2 * e.g.n_kv_heads;
          const bool rotate = hg < e.n_heads + e.g.n_kv_heads;
          long long dst_own = 0;                                // element offset of this thread's row in its destination, -1: none
          int which = 0;                                        // 0: q, 1: kv_store
          if (row_ok && head_ok) {
            if (hg < e.n_heads) dst_own = ((long long)row * e.n_heads + hg) * 128;
            else if (rotate) { dst_own = e.g.offset(e.layer, page, 0, hg - e.n_heads, slot_in_page); which = 1; }
            else { dst_own = e.g.offset(e.layer, page, 1, hg - e.n_heads - e.g.n_kv_heads, slot_in_page); which = 1; }
          } else {
            dst_own = -1;
          }
          bf16* const dbase = (hg < e.n_heads) ? e.q : e.kv_store;
          (void)which;
#pragma unroll 1
          for (int a = 0; a < 2; ++a) {
            __syncwarp();
            ptx::tmem_ld_32x32(taddr + hh * 128 + a * 32, r);
            ptx::tmem_ld_32x32(taddr + hh * 128 + a * 32 + 64, u2);
            ptx::tmem_ld_wait();
            stg_write(0, r);
            stg_write(1, u2);
            __syncwarp();
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int rr = 4 * i + t_rr;
              const long long d_rr = __shfl_sync(0xffffffffu, dst_own, rr);
              const int pos_rr = __shfl_sync(0xffffffffu, pos, rr);
              float4 lo = stg_read(0, i), hi = stg_read(1, i);
              if (d_rr < 0) continue;
              if (rotate) {
                const float4 c = *reinterpret_cast<const float4*>(e.rope_cos + (long long)pos_rr * 64 + a * 32 + t_c4);
                const float4 s = *reinterpret_cast<const float4*>(e.rope_sin + (long long)pos_rr * 64 + a * 32 + t_c4);
                const float4 l2 = make_float4(lo.x * c.x - hi.x * s.x, lo.y * c.y - hi.y * s.y, lo.z * c.z - hi.z * s.z, lo.w * c.w - hi.w * s.w);
                hi = make_float4(hi.x * c.x + lo.x * s.x, hi.y * c.y + lo.y * s.y, hi.z * c.z + lo.z * s.z, hi.w * c.w + lo.w * s.w);
                lo = l2;
              }
              bf16* d = dbase + d_rr + a * 32 + t_c4;
              *reinterpret_cast<uint2*>(d) = make_uint2(pack_bf16(lo.x, lo.y), pack_bf16(lo.z, lo.w));
              *reinterpret_cast<uint2*>(d + 64) = make_uint2(pack_bf16(hi.x, hi.y), pack_bf16(hi.z, hi.w));
            }
          }
        }
      } else if (EPI == EPI_LMHEAD) {
        // a11: split-vocab online (max, sum exp(z - max), argmax); z = scale * acc; mask_id and columns >= V excluded.
        const int n0 = tl.n_blk * BN;
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
          *reinterpret_cast<int4*>(p.part + (long long)row * p.n_tiles + tl.n_blk) = *reinterpret_cast<int4*>(&o);
        }
      }
      // this warp's quarter of the accumulator stage has been read: let the leader's MMA issuer reuse it
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster(te_leader + 8u * as);
    }
  }
  if ((EPI == EPI_F32 || EPI == EPI_RESID) && warp >= 2 && lane == 0) ptx::bulk_wait<0>();   // bulk stores / reductions have landed
  ptx::tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) trace_end(p.tr);
  ptx::cluster_sync();          // no CTA of the pair frees TMEM / leaves while its peer may still signal it
  if (warp == 1) ptx::tmem_dealloc_pair(tmem_base, 512);
}

}  // namespace dlm
