// Persistent whole-stack kernel for small cached steps (T <= 64 tokens, the batch-1 "cache step" of P:347 that the
// headline workload spends 31 of every 32 steps in): ALL layers of the step in ONE launch, one CTA per SM.  An experiment that
// is kept because it is correct and instructive, not because it is faster (see Status below).
//
// Why.  With 32 tokens a layer is pure weight streaming (436 MB per layer at the LLaDA shape = 66.7 us at the measured
// HBM rate) and the in-kernel timeline of the multi-kernel path (DLM_OPT_TRACE) shows its GEMMs already AT that rate --
// the whole distance to the roofline (3.19 ms vs 2.34 ms per step) is the ~25 us per layer during which the small
// kernels between the GEMMs (RMSNorm x 2, RoPE + K/V write, attention, split merge) hold the stream while HBM idles:
// a kernel boundary costs ~3.5 us of dependency latency and only the next GEMM's shared-memory ring can be prefetched
// under it.  Here the weight stream never stops:
//
//   warp 0        W producer: walks the step's whole sequence of (layer, projection, tile, K block) work of THIS SM and
//                 issues the TMA loads of the weight tiles into a ring of `stages` x 16 KB as slots free up.  It depends on
//                 nothing but ring space, so it runs ahead across every phase boundary: while the SM waits for a grid-wide
//                 dependency, does attention or a norm, the ring fills with the NEXT projection's weights.
//   warp 1        X producer: TMA loads of the activation tiles (tpad rows x 64) of the same sequence; before the first load
//                 of a projection it waits for the grid-wide phase counter (the producer of that activation has finished).
//   warp 2        MMA issuer: tcgen05.mma 128 x tpad x 16, swap-AB (weights on the 128 TMEM lanes, tokens on N), accumulator
//                 double-buffered in TMEM.
//   warps 3..6    compute: GEMM epilogues (TMEM -> fp32 partial slices) and the phases between the projections: residual
//                 fold + RMSNorm, RoPE + K/V page write + attention (mma.sync flash loop over the paged K/V), SwiGLU.
//
// Work split (stream-K).  A projection with n_tiles x kbt (tile, K block) units is cut into gridDim.x equal contiguous runs,
// so every SM streams the same number of weight bytes in every phase (+-16 KB) whatever N / 128 is (32 tiles for O / down,
// 96 for QKV, 192 for gate/up on 148 SMs).  A tile cut by a run boundary leaves one fp32 partial slice per run (`seg`); the
// consumer phase sums the slices of a tile in slice order, so results are deterministic (no atomics).
//
// Phases per layer (each ends with one arrival per CTA on a global counter; waiting = polling that counter):
//   0 fold + norm   x += sum of the down-projection slices of the previous layer; u = bf16(RMSNorm(x))   (one row per CTA)
//   1 QKV GEMM      u -> partial slices; the CTA that completes a 128-column tile (= one head) finishes it: slice sum, RoPE,
//                   Q row / K,V page rows (qkv_finish.cuh)
//   2 attention     per (request, KV head, K/V range): mma.sync flash loop over the pages; the last range of a head to arrive
//                   merges the ranges
//   3 O GEMM        attn -> slices
//   4 fold + norm   -> u2
//   5 gate/up GEMM  u2 -> slices (64 gate + 64 up rows per tile); the completing CTA applies SwiGLU -> act
//   6 down GEMM     act -> slices
// and a final fold after the last layer.  Rounding points are those of the per-stage path.
//
// Status: correct (tests/test_gpu_engine.py::test_layer_kernel_option_*), but 3.95 ms per C2 cached step against 3.2 ms for the
// per-stage kernels: a grid-wide phase boundary is a chain of dependent L2 round trips (slice stores, fence, atomic, poll, TMA
// of X, first MMA) that costs what a kernel boundary costs under programmatic dependent launch, and the ring here is smaller.
// Off by default (DLM_OPT_LAYER_KERNEL); DESIGN.md section 8 has the phase timings.
#pragma once
#include <math_constants.h>

#include "attn_flash.cuh"
#include "common.cuh"
#include "kernels_basic.cuh"
#include "ptx_sm100.cuh"
#include "qkv_finish.cuh"

namespace dlm {

constexpr int kMgThreads = 224;
constexpr int kMgWBytes = 128 * 128;          // one weight tile: 128 rows x 64 bf16
constexpr int kMgMaxTpad = 64;
constexpr int kMgPhasesPerLayer = 7;          // fold+norm, QKV (+RoPE, K/V write), attention, O, fold+norm, gate/up (+SwiGLU), down
constexpr int kMgScratchOwn = 48 * 1024;      // attention scratch beyond the (idle) X ring: Q 16 KB + K 2 x 16 KB + V 2 x 16 KB = 80 KB in all
constexpr int kMgAttnBytes = 80 * 1024;
constexpr int kMgMaxSeg = 6;                  // most slices a tile of the O / down projection may be cut into
constexpr int kMgMaxSegQkv = 3, kMgMaxSegGu = 2;
constexpr int kMgMaxAttSplits = 4;            // K/V ranges per (request, KV head) in the attention phase
constexpr int kMgMaxTiles = 384;              // tiles per projection the slice-count tables hold
constexpr int kMgTailBytes = 512 + 4 * kMgMaxTiles * 4 + 64;      // barriers, slice-count tables, reduction scratch

struct MegaParams {
  int layer0, n_layers;            // layers [layer0, layer0 + n_layers) in this launch (debug-dump mode runs them one by one)
  int T, tpad, stages;
  int d, HQ, NQKV, F, Fp;          // Fp = first tiled row of the up projection (pad128(F))
  int n_heads;
  float eps, scale_log2;
  const CUtensorMap* wmaps;        // device array [n_layers][4]: tiled weight maps of Wqkv, Wo, Wgu (box 64), Wd
  float* x;                        // [T, d] fp32 residual stream (in: embeddings; out: the last layer's output)
  bf16* u;                         // [T, d] RMSNorm output feeding QKV
  bf16* u2;                        // [T, d] RMSNorm output feeding gate/up
  bf16* q;                         // [T, HQ] Q after RoPE (written by the QKV projection's finishing CTA of each head)
  float* xmid_dump;                // optional [T, d]: residual after the O projection (debug dump), or null
  bf16* attn;                      // [T, HQ]
  bf16* act;                       // [T, F]
  float* part_a;                   // slices of the QKV and gate/up projections: [seg][T][NQKV | 2F]
  float* part_x;                   // slices of the O and down projections:       [seg][T][d]
  const float* rope_cos;
  const float* rope_sin;
  bf16* kv_store;
  const int* page_table;
  BatchDesc b;
  KvGeom g;
  unsigned int* bar;               // phase counter, zero at launch
  unsigned int* tile_cnt;          // [kMgMaxTiles] arrivals per tile of the projection in flight (zero at launch, self-resetting)
  int att_splits;                  // K/V splits per (request, KV head) in the attention phase (1: no merge)
  float* ws_o;                     // [att_splits][T * H][128] unnormalised partial outputs
  float* ws_ml;                    // [att_splits][T * H][2]   (running max in log2 units, running sum)
  unsigned long long* phase_ts;    // optional [8 L + 2] %globaltimer at the end of each phase in CTA 0 (tuning aid), or null
  TraceSlot tr;
};

__host__ __device__ inline int mega_stage_bytes(int tpad) { return kMgWBytes + tpad * 128; }
__host__ inline int mega_stages(int tpad) { return (227 * 1024 - kMgScratchOwn - kMgTailBytes - 1024) / mega_stage_bytes(tpad); }
__host__ inline int mega_smem_bytes(int tpad, int stages) { return stages * mega_stage_bytes(tpad) + kMgScratchOwn + kMgTailBytes + 1024; }

// ---- stream-K geometry of a projection: U = n_tiles * kbt units over G CTAs ----
struct MgGemm { int n_tiles, kbt; };
__device__ __forceinline__ long long mg_u0(long long U, int G, int i) { return U * i / G; }
// CTA whose run contains `unit`: smallest i with U (i + 1) / G > unit
__device__ __forceinline__ int mg_owner(long long unit, long long U, int G) { return (int)(((unit + 1) * G + U - 1) / U) - 1; }
__device__ __forceinline__ int mg_nseg(int tile, const MgGemm& gm, int G) {
  const long long U = (long long)gm.n_tiles * gm.kbt;
  return mg_owner((long long)(tile + 1) * gm.kbt - 1, U, G) - mg_owner((long long)tile * gm.kbt, U, G) + 1;
}

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// poll the phase counter until `target` arrivals (bounded: a protocol bug traps instead of hanging the GPU)
__device__ __forceinline__ void mg_wait_count(const unsigned int* bar, unsigned int target) {
  if (ld_acquire_u32(bar) >= target) return;
  const long long t0 = clock64();
  while (ld_acquire_u32(bar) < target) {
    __nanosleep(32);
    if (clock64() - t0 > 4000000000LL) __trap();
  }
}
__device__ __forceinline__ void mg_bar128() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

__global__ void __launch_bounds__(kMgThreads, 1)
layer_mega_kernel(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapU2, const __grid_constant__ CUtensorMap mapAttn,
                  const __grid_constant__ CUtensorMap mapAct, const MegaParams p) {
  extern __shared__ uint8_t mg_smem[];
  const uint32_t base = (ptx::smem_u32(mg_smem) + 1023u) & ~1023u;
  uint8_t* const gen_base = mg_smem + (base - ptx::smem_u32(mg_smem));
  const int stages = p.stages;
  const uint32_t sW = base;                                          // [stages][16 KB]
  const uint32_t sX = sW + stages * kMgWBytes;                       // [stages][tpad x 128 B]   (attention scratch aliases it)
  const uint32_t x_stage = (uint32_t)p.tpad * 128u;
  const uint32_t sOwn = sX + stages * x_stage;                       // kMgScratchOwn
  const uint32_t bar_base = sOwn + kMgScratchOwn;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (stages + s); };
  const uint32_t tmem_full = bar_base + 16u * stages;                // [2]
  const uint32_t tmem_empty = tmem_full + 16u;                       // [2]
  const uint32_t tmem_ptr_addr = tmem_empty + 16u;
  int* const nseg_tab = reinterpret_cast<int*>(gen_base + (bar_base - base) + 512);     // [4][kMgMaxTiles]
  float* const red = reinterpret_cast<float*>(gen_base + (bar_base - base) + 512 + 4 * kMgMaxTiles * 4);   // [4]
  int* const red_i = reinterpret_cast<int*>(red + 8);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = (int)gridDim.x, cta = (int)blockIdx.x;
  const int L = p.n_layers, T = p.T, tpad = p.tpad;
  const MgGemm gm[4] = {{p.NQKV / 128, p.d / 64}, {p.d / 128, p.HQ / 64}, {p.F / 64, p.d / 64}, {p.d / 128, p.F / 64}};
  const uint32_t tmem_cols = 2 * tpad <= 64 ? 64u : 128u;

  if (threadIdx.x == 0) trace_begin(p.tr);
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&mapU); ptx::prefetch_tmap(&mapU2); ptx::prefetch_tmap(&mapAttn); ptx::prefetch_tmap(&mapAct);
    for (int s = 0; s < stages; ++s) { ptx::mbar_init(full_bar(s), 2); ptx::mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; ++a) { ptx::mbar_init(tmem_full + 8u * a, 1); ptx::mbar_init(tmem_empty + 8u * a, 4); }
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc(tmem_ptr_addr, tmem_cols);
    ptx::tmem_relinquish();
  }
  // slice counts per tile of the four projections (consumers sum that many slices)
  for (int i = threadIdx.x; i < 4 * kMgMaxTiles; i += kMgThreads) {
    const int gi = i / kMgMaxTiles, t = i % kMgMaxTiles;
    nseg_tab[i] = t < gm[gi].n_tiles ? mg_nseg(t, gm[gi], G) : 0;
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_ptr_addr));

  if (warp == 0) {
    // =============================== W producer ===============================
    if (ptx::elect_one()) {
      int s = 0;
      uint32_t ph = 0;
      for (int l = 0; l < L; ++l) {
        for (int gi = 0; gi < 4; ++gi) {
          const CUtensorMap* mw = p.wmaps + (p.layer0 + l) * 4 + gi;
          const long long U = (long long)gm[gi].n_tiles * gm[gi].kbt;
          const long long u0 = mg_u0(U, G, cta), u1 = mg_u0(U, G, cta + 1);
          for (long long un = u0; un < u1; ++un, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1u : 0u)) {
            const int tile = (int)(un / gm[gi].kbt), kb = (int)(un % gm[gi].kbt);
            ptx::mbar_wait(empty_bar(s), ph ^ 1u);
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)kMgWBytes);
            const uint32_t dst = sW + s * kMgWBytes;
            if (gi == 2) {          // 64 gate rows + the matching 64 up rows
              ptx::tma_load_w_tiled(dst, mw, kb, tile * 64, 64, 64, full_bar(s), DLM_L2_EVICT_FIRST);
              ptx::tma_load_w_tiled(dst + 64 * 128, mw, kb, p.Fp + tile * 64, 64, 64, full_bar(s), DLM_L2_EVICT_FIRST);
            } else {
              ptx::tma_load_w_tiled(dst, mw, kb, tile * 128, 128, 128, full_bar(s), DLM_L2_EVICT_FIRST);
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // =============================== X producer ===============================
    if (ptx::elect_one()) {
      pdl_wait();                    // x (embeddings) and the request state come from the kernels before this one
      int s = 0;
      uint32_t ph = 0;
      for (int l = 0; l < L; ++l) {
        for (int gi = 0; gi < 4; ++gi) {
          const CUtensorMap* mx = gi == 0 ? &mapU : (gi == 1 ? &mapAttn : (gi == 2 ? &mapU2 : &mapAct));
          const long long U = (long long)gm[gi].n_tiles * gm[gi].kbt;
          const long long u0 = mg_u0(U, G, cta), u1 = mg_u0(U, G, cta + 1);
          if (u0 < u1) {
            // the activation is complete when the phase before this projection has been arrived at by every CTA
            const int phase = l * kMgPhasesPerLayer + (gi == 3 ? 6 : 2 * gi + 1);      // phases completed before this projection may read X
            mg_wait_count(p.bar, (unsigned)G * (unsigned)phase);
            asm volatile("fence.proxy.async;" ::: "memory");      // generic-proxy writes of other CTAs -> TMA (async proxy) reads
          }
          for (long long un = u0; un < u1; ++un, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1u : 0u)) {
            const int kb = (int)(un % gm[gi].kbt);
            ptx::mbar_wait(empty_bar(s), ph ^ 1u);
            ptx::mbar_expect_tx(full_bar(s), x_stage);
            ptx::tma_load_2d(sX + s * x_stage, mx, kb * 64, 0, full_bar(s), DLM_L2_EVICT_LAST);
          }
        }
      }
    }
  } else if (warp == 2) {
    // =============================== MMA issuer ===============================
    const uint32_t idesc = ptx::umma_idesc_bf16(128, tpad);
    int s = 0, it = 0;
    uint32_t ph = 0;
    for (int l = 0; l < L; ++l) {
      for (int gi = 0; gi < 4; ++gi) {
        const long long U = (long long)gm[gi].n_tiles * gm[gi].kbt;
        const long long u0 = mg_u0(U, G, cta), u1 = mg_u0(U, G, cta + 1);
        for (long long un = u0; un < u1;) {
          const int k0 = (int)(un % gm[gi].kbt);
          const int n = (int)min((long long)(gm[gi].kbt - k0), u1 - un);      // K blocks of this segment
          const uint32_t acc = (uint32_t)it & 1u, aph = ((uint32_t)it >> 1) & 1u;
          ptx::mbar_wait(tmem_empty + 8u * acc, aph ^ 1u);
          ptx::tc_fence_after();
          const uint32_t d_tmem = tmem_base + acc * (uint32_t)tpad;
          for (int k = 0; k < n; ++k, s = (s + 1 == stages ? 0 : s + 1), ph ^= (s == 0 ? 1u : 0u)) {
            ptx::mbar_wait(full_bar(s), ph);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
              const uint32_t w_lo = ptx::umma_desc_lo(sW + s * kMgWBytes), x_lo = ptx::umma_desc_lo(sX + s * x_stage);
#pragma unroll
              for (int kk = 0; kk < 4; ++kk)
                ptx::umma_bf16_lo(d_tmem, w_lo + 2 * kk, x_lo + 2 * kk, idesc, (k | kk) != 0 ? 1u : 0u);
              ptx::umma_commit(empty_bar(s));
              if (k + 1 == n) ptx::umma_commit(tmem_full + 8u * acc);
            }
            __syncwarp();
          }
          un += n;
          ++it;
        }
      }
    }
  } else {
    // =============================== compute warps (3..6) ===============================
    const int tid = threadIdx.x - 96;                 // 0..127
    const int cw = warp - 3;                          // 0..3
    const int quarter = warp & 3;                     // TMEM lane quarter this warp may read
    int it = 0;                                       // accumulator use counter (mirrors the MMA warp)
    int phase = 0;                                    // phases completed by this CTA
    pdl_wait();
    if (tid == 0) trace_wait(p.tr);

    auto arrive = [&]() {                             // this CTA has finished the current phase
      mg_bar128();
      if (tid == 0) {
        __threadfence();
        asm volatile("fence.proxy.async;" ::: "memory");
        atomicAdd(p.bar, 1u);
        if (p.phase_ts && cta == 0) p.phase_ts[phase] = gtimer_ns();
      }
      ++phase;
    };
    auto wait_prev = [&]() {                          // every CTA has finished the phase before the current one
      if (tid == 0) mg_wait_count(p.bar, (unsigned)G * (unsigned)phase);
      mg_bar128();
    };

    // ---- finish one 128-column tile (= one head) of the QKV projection: qkv_finish.cuh ----
    QkvFinish qf_;
    qf_.part = p.part_a; qf_.slice_stride = (long long)T * p.NQKV; qf_.ld = p.NQKV; qf_.T = T; qf_.HQ = p.HQ; qf_.n_heads = p.n_heads;
    qf_.q = p.q; qf_.kv_store = p.kv_store; qf_.rope_cos = p.rope_cos; qf_.rope_sin = p.rope_sin; qf_.page_table = p.page_table;
    qf_.b = p.b; qf_.g = p.g; qf_.tile_cnt = p.tile_cnt;
    auto finish_qkv = [&](int tile, int ns, int layer) { qkv_finish_tile<kMgMaxSegQkv>(qf_, tile, ns, layer, tid); };

    // ---- finish one gate/up tile (64 features): act[t, f] = bf16(silu(sum gate slices) * sum up slices) ----
    auto finish_gu = [&](int tile, int ns) {
      const int ld = 2 * p.F;
      const long long st = (long long)T * ld;
      for (int i0 = tid; i0 < T * 16; i0 += 4 * 128) {        // item = (token, features j .. j + 3 of the tile's 64)
        float4 ga[4][kMgMaxSegGu], ua[4][kMgMaxSegGu];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
          const int i = i0 + m * 128;
          const bool ok = i < T * 16;
          const int t = ok ? i >> 4 : 0, j = (i & 15) * 4;
          const float* gp = p.part_a + (long long)t * ld + tile * 128 + j;
#pragma unroll
          for (int s = 0; s < kMgMaxSegGu; ++s) {
            ga[m][s] = (ok && s < ns) ? __ldcg(reinterpret_cast<const float4*>(gp + s * st)) : make_float4(0.f, 0.f, 0.f, 0.f);
            ua[m][s] = (ok && s < ns) ? __ldcg(reinterpret_cast<const float4*>(gp + s * st + 64)) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
        }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
          const int i = i0 + m * 128;
          if (i >= T * 16) continue;
          const int t = i >> 4, j = (i & 15) * 4;
          float4 g = ga[m][0], w = ua[m][0];
#pragma unroll
          for (int s = 1; s < kMgMaxSegGu; ++s) {
            g.x += ga[m][s].x; g.y += ga[m][s].y; g.z += ga[m][s].z; g.w += ga[m][s].w;
            w.x += ua[m][s].x; w.y += ua[m][s].y; w.z += ua[m][s].z; w.w += ua[m][s].w;
          }
          uint2 o;
          o.x = pack_bf16(silu_f(g.x) * w.x, silu_f(g.y) * w.y); o.y = pack_bf16(silu_f(g.z) * w.z, silu_f(g.w) * w.w);
          __stcg(reinterpret_cast<uint2*>(p.act + (long long)t * p.F + tile * 64 + j), o);
        }
      }
    };

    // ---- GEMM epilogue: this CTA's segments of projection gi -> fp32 slices ----
    auto gemm_epilogue = [&](int gi, float* part, int ld, const int* nseg, int layer) {
      const long long U = (long long)gm[gi].n_tiles * gm[gi].kbt;
      const long long u0 = mg_u0(U, G, cta), u1 = mg_u0(U, G, cta + 1);
      for (long long un = u0; un < u1;) {
        const int tile = (int)(un / gm[gi].kbt), k0 = (int)(un % gm[gi].kbt);
        const int n = (int)min((long long)(gm[gi].kbt - k0), u1 - un);
        const int seg = cta - mg_owner((long long)tile * gm[gi].kbt, U, G);
        const uint32_t acc = (uint32_t)it & 1u, aph = ((uint32_t)it >> 1) & 1u;
        ptx::mbar_wait(tmem_full + 8u * acc, aph);
        ptx::tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + acc * (uint32_t)tpad;
        float* o = part + ((long long)seg * T) * ld + (long long)tile * 128 + quarter * 32 + lane;
        uint32_t r[32];
        for (int c = 0; c < tpad / 32; ++c) {
          __syncwarp();
          ptx::tmem_ld_32x32(taddr + c * 32, r);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const int tok = c * 32 + j;
            if (tok < T) __stcg(o + (long long)tok * ld, __uint_as_float(r[j]));
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(tmem_empty + 8u * acc);
        if (gi == 0 || gi == 2) {
          // the CTA that completes a tile (the last of its <= 3 runs to arrive) finishes it: sums the slices in slice order and
          // applies RoPE + the Q / K/V-page write (QKV) or SwiGLU (gate/up).  This runs under the other CTAs' streaming
          // instead of in a phase of its own.
          __threadfence();
          mg_bar128();
          if (tid == 0) red_i[0] = (int)atomicAdd(p.tile_cnt + tile, 1u);
          mg_bar128();
          if (red_i[0] == nseg[tile] - 1) {
            if (tid == 0) p.tile_cnt[tile] = 0;           // every run of the tile has arrived: ready for the next layer
            __threadfence();
            if (gi == 0) finish_qkv(tile, nseg[tile], layer); else finish_gu(tile, nseg[tile]);
          }
        }
        un += n;
        ++it;
      }
      arrive();
    };

    // ---- fold + RMSNorm: x[t] += slices of the previous O / down projection (tile slice counts nseg), u = bf16(x rs) ----
    auto fold_norm = [&](const int* nseg, bool have_part, bf16* uo, float* copy_to) {
      wait_prev();
      const int nvec = p.d >> 2;
      for (int t = cta; t < T; t += G) {
        float4* xr = reinterpret_cast<float4*>(p.x + (long long)t * p.d);
        float4 v[8];                                   // d <= 4096 (8 x 128 threads x 4)
        float ss = 0.f;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int i = tid + k * 128;
          v[k] = i < nvec ? __ldcg(xr + i) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        if (have_part) {
          // every slice load of four chunks is issued before the first add (independent loads: one L2 round trip per half
          // instead of one per slice); slices past a tile's count are not read and add an exact zero, order = slice order
          const float4* pr = reinterpret_cast<const float4*>(p.part_x + (long long)t * p.d);
          const long long st4 = ((long long)T * p.d) >> 2;
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            float4 q[4][kMgMaxSeg];
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              const int i = tid + (h * 4 + kk) * 128;
              const int ns = i < nvec ? nseg[i >> 5] : 0;
#pragma unroll
              for (int s = 0; s < kMgMaxSeg; ++s) q[kk][s] = s < ns ? __ldcg(pr + s * st4 + i) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              float4& a = v[h * 4 + kk];
#pragma unroll
              for (int s = 0; s < kMgMaxSeg; ++s) { a.x += q[kk][s].x; a.y += q[kk][s].y; a.z += q[kk][s].z; a.w += q[kk][s].w; }
            }
          }
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const int i = tid + k * 128;
            if (i < nvec) __stcg(xr + i, v[k]);
          }
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int i = tid + k * 128;
          if (i < nvec) {
            if (copy_to) reinterpret_cast<float4*>(copy_to + (long long)t * p.d)[i] = v[k];
            ss += v[k].x * v[k].x + v[k].y * v[k].y + v[k].z * v[k].z + v[k].w * v[k].w;
          }
        }
        if (!uo) continue;                             // final fold: only x is wanted
        ss = warp_sum(ss);
        if (lane == 0) red[cw] = ss;
        mg_bar128();
        const float rs = rsqrtf(((red[0] + red[1]) + (red[2] + red[3])) / (float)p.d + p.eps);
        bf16* ur = uo + (long long)t * p.d;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int i = tid + k * 128;
          if (i < nvec) {
            uint2 w;
            w.x = pack_bf16(v[k].x * rs, v[k].y * rs); w.y = pack_bf16(v[k].z * rs, v[k].w * rs);
            __stcg(reinterpret_cast<uint2*>(ur + 4 * i), w);
          }
        }
        mg_bar128();                                   // red[] is reused by the next row
      }
      arrive();
    };

    // ---- attention phase of layer l: units (request, KV head) ----
    auto attention = [&](int l) {
      wait_prev();
      const int H = p.n_heads, Hkv = p.g.n_kv_heads, r = H / Hkv;
      // scratch = the X ring (idle during this phase: this CTA's X producer cannot pass the phase counter before the CTA
      // arrives) followed by the own scratch, contiguous: Q [64 rows][256 B] 16 KB, K 2 x 16 KB, V 2 x 16 KB
      const uint32_t sQ = sX, bK = sX + 16384, bV = sX + 16384 + 32768;
      const int nsp = p.att_splits;
      const long long TH = (long long)T * H;
      for (int unit = cta; unit < p.b.n * Hkv * nsp; unit += G) {
        const int sp = unit % nsp, bi = (unit / nsp) / Hkv, kvh = (unit / nsp) % Hkv;
        const int q_len = p.b.q_len[bi];
        if (q_len <= 0) continue;
        const int n_rows = q_len * r, S = p.b.kv_len[bi], q_off = p.b.q_off[bi];
        const int* pt = p.page_table + (long long)p.b.slot[bi] * p.g.max_pages_per_req;
        // -- Q tile: the rows the QKV projection's finishing CTAs wrote (bf16, rotated); rows past n_rows: zeros
        for (int i = tid; i < 64 * 16; i += 128) {
          const int rho = i >> 4, ch = i & 15;
          const bool ok = rho < n_rows;
          const int tok = ok ? rho / r : 0, hh = ok ? rho % r : 0;
          cp_async16(sQ + tile_off(rho, ch), p.q + ((long long)(q_off + tok) * H + kvh * r + hh) * 128 + ch * 8, ok);
        }
        // -- (c) flash loop over the request's K/V pages (64-token tiles, double-buffered cp.async); warp w owns rows 16 w .. 16 w + 15
        auto load_kv = [&](int tile, int buf) {
          const int j0 = tile * kFaBN;
          const int page = pt[j0 / p.g.page_tokens];
          const int in_page = j0 % p.g.page_tokens;
          const bf16* kb = p.kv_store + p.g.offset(l, page, 0, kvh, in_page);
          const bf16* vb = p.kv_store + p.g.offset(l, page, 1, kvh, in_page);
          for (int i = tid; i < kFaBN * 16; i += 128) {
            const int row = i >> 4, ch = i & 15;
            const bool ok = j0 + row < S;
            cp_async16(bK + buf * kFaBN * 256 + tile_off(row, ch), kb + row * kFaDh + ch * 8, ok);
            cp_async16(bV + buf * kFaBN * 256 + tile_off(row, ch), vb + row * kFaDh + ch * 8, ok);
          }
        };
        const int n_tiles_all = (S + kFaBN - 1) / kFaBN;
        const int per_sp = (n_tiles_all + nsp - 1) / nsp;
        const int t_begin = sp * per_sp, t_end = min(n_tiles_all, t_begin + per_sp);     // this unit's K/V tiles (may be empty)
        if (t_begin < t_end) load_kv(t_begin, 0);
        cp_async_commit();
        float o[16][4];
#pragma unroll
        for (int i = 0; i < 16; ++i) { o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f; }
        float m0 = -CUDART_INF_F, m1 = -CUDART_INF_F, l0 = 0.f, l1 = 0.f;
        uint32_t qf[8][4];
        const int wrow = cw * 16;
        const bool live = wrow < n_rows;                    // warp-uniform: this warp has query rows
        for (int t = t_begin; t < t_end; ++t) {
          const int buf = (t - t_begin) & 1;
          if (t + 1 < t_end) load_kv(t + 1, buf ^ 1);
          cp_async_commit();
          cp_async_wait<1>();
          mg_bar128();
          if (live) {
            if (t == t_begin) {
#pragma unroll
              for (int ks = 0; ks < 8; ++ks)
                ldsm_x4(sQ + tile_off(wrow + (lane & 7) + ((lane >> 3) & 1) * 8, ks * 2 + (lane >> 4)), qf[ks][0], qf[ks][1], qf[ks][2], qf[ks][3]);
            }
            const uint32_t kbase = bK + buf * kFaBN * 256, vbase = bV + buf * kFaBN * 256;
            float sc[8][4];
#pragma unroll
            for (int j = 0; j < 8; ++j) { sc[j][0] = sc[j][1] = sc[j][2] = sc[j][3] = 0.f; }
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
#pragma unroll
              for (int jp = 0; jp < 4; ++jp) {
                uint32_t b0, b1, b2, b3;
                ldsm_x4(kbase + tile_off(jp * 16 + (lane & 7) + (lane >> 4) * 8, ks * 2 + ((lane >> 3) & 1)), b0, b1, b2, b3);
                mma_bf16_16816(sc[2 * jp], qf[ks], b0, b1);
                mma_bf16_16816(sc[2 * jp + 1], qf[ks], b2, b3);
              }
            }
            const int j0 = t * kFaBN;
            float tm0 = -CUDART_INF_F, tm1 = -CUDART_INF_F;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const int col = j0 + j * 8 + (lane & 3) * 2;
              sc[j][0] = (col < S) ? sc[j][0] * p.scale_log2 : -CUDART_INF_F;
              sc[j][1] = (col + 1 < S) ? sc[j][1] * p.scale_log2 : -CUDART_INF_F;
              sc[j][2] = (col < S) ? sc[j][2] * p.scale_log2 : -CUDART_INF_F;
              sc[j][3] = (col + 1 < S) ? sc[j][3] * p.scale_log2 : -CUDART_INF_F;
              tm0 = fmaxf(tm0, fmaxf(sc[j][0], sc[j][1]));
              tm1 = fmaxf(tm1, fmaxf(sc[j][2], sc[j][3]));
            }
            tm0 = fmaxf(tm0, __shfl_xor_sync(0xffffffffu, tm0, 1)); tm0 = fmaxf(tm0, __shfl_xor_sync(0xffffffffu, tm0, 2));
            tm1 = fmaxf(tm1, __shfl_xor_sync(0xffffffffu, tm1, 1)); tm1 = fmaxf(tm1, __shfl_xor_sync(0xffffffffu, tm1, 2));
            const float nm0 = fmaxf(m0, tm0), nm1 = fmaxf(m1, tm1);
            const float c0 = exp2f(m0 - nm0), c1 = exp2f(m1 - nm1);
            m0 = nm0; m1 = nm1;
            float rs0 = 0.f, rs1 = 0.f;
            uint32_t pf[4][4];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const float p0 = exp2f(sc[j][0] - nm0), p1 = exp2f(sc[j][1] - nm0);
              const float p2 = exp2f(sc[j][2] - nm1), p3 = exp2f(sc[j][3] - nm1);
              rs0 += p0 + p1; rs1 += p2 + p3;
              pf[j >> 1][(j & 1) * 2 + 0] = pack_bf16(p0, p1);
              pf[j >> 1][(j & 1) * 2 + 1] = pack_bf16(p2, p3);
            }
            l0 = l0 * c0 + rs0; l1 = l1 * c1 + rs1;
#pragma unroll
            for (int i = 0; i < 16; ++i) { o[i][0] *= c0; o[i][1] *= c0; o[i][2] *= c1; o[i][3] *= c1; }
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
#pragma unroll
              for (int np = 0; np < 8; ++np) {
                uint32_t b0, b1, b2, b3;
                ldsm_x4_t(vbase + tile_off(kk * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, np * 2 + (lane >> 4)), b0, b1, b2, b3);
                mma_bf16_16816(o[2 * np], pf[kk], b0, b1);
                mma_bf16_16816(o[2 * np + 1], pf[kk], b2, b3);
              }
            }
          }
          mg_bar128();                                      // everyone is done with `buf` before the next prefetch overwrites it
        }
        cp_async_wait<0>();
        if (live) {
          l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
          l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
          const int gq = lane >> 2, tq = lane & 3;
#pragma unroll
          for (int hr = 0; hr < 2; ++hr) {
            const int rho = wrow + gq + hr * 8;
            if (rho >= n_rows) continue;
            const int tok = rho / r, hh = rho % r;
            const long long orow = (long long)(q_off + tok) * H + kvh * r + hh;
            if (nsp == 1) {
              const float inv = 1.f / (hr ? l1 : l0);
              bf16* dst = p.attn + orow * kFaDh;
#pragma unroll
              for (int i = 0; i < 16; ++i)
                __stcg(reinterpret_cast<unsigned int*>(dst + i * 8 + tq * 2), pack_bf16(o[i][hr * 2] * inv, o[i][hr * 2 + 1] * inv));
            } else {                                          // unnormalised partial of this K/V range
              float* dst = p.ws_o + ((long long)sp * TH + orow) * kFaDh;
#pragma unroll
              for (int i = 0; i < 16; ++i)
                __stcg(reinterpret_cast<float2*>(dst + i * 8 + tq * 2), make_float2(o[i][hr * 2], o[i][hr * 2 + 1]));
              if (tq == 0) {
                const bool any = t_begin < t_end;
                __stcg(reinterpret_cast<float2*>(p.ws_ml + ((long long)sp * TH + orow) * 2), make_float2(any ? (hr ? m1 : m0) : -CUDART_INF_F, any ? (hr ? l1 : l0) : 0.f));
              }
            }
          }
        }
        if (nsp > 1) {
          // the last of the (request, KV head)'s K/V ranges to arrive merges them: out = sum_s o_s 2^(m_s - m) / sum_s l_s 2^(m_s - m),
          // ranges in index order (deterministic)
          unsigned int* cnt = p.tile_cnt + kMgMaxTiles + (bi * Hkv + kvh);
          mg_bar128();
          if (tid == 0) { __threadfence(); red_i[0] = (int)atomicAdd(cnt, 1u); }
          mg_bar128();
          if (red_i[0] == nsp - 1) {
            if (tid == 0) *cnt = 0;
            __threadfence();
            for (int i0 = tid; i0 < n_rows * 32; i0 += 2 * 128) {       // item = (stacked row, 4 output dims); 2 items per pass
              float4 po[2][kMgMaxAttSplits];
              float2 ml[2][kMgMaxAttSplits];
#pragma unroll
              for (int mm = 0; mm < 2; ++mm) {
                const int i = i0 + mm * 128;
                const bool ok = i < n_rows * 32;
                const int rho = ok ? i >> 5 : 0, e = (i & 31) * 4;
                const long long orow = (long long)(q_off + rho / r) * H + kvh * r + rho % r;
#pragma unroll
                for (int s2 = 0; s2 < kMgMaxAttSplits; ++s2) {
                  const bool ld = ok && s2 < nsp;
                  ml[mm][s2] = ld ? __ldcg(reinterpret_cast<const float2*>(p.ws_ml + ((long long)s2 * TH + orow) * 2)) : make_float2(-CUDART_INF_F, 0.f);
                  po[mm][s2] = ld ? __ldcg(reinterpret_cast<const float4*>(p.ws_o + ((long long)s2 * TH + orow) * kFaDh + e)) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
              }
#pragma unroll
              for (int mm = 0; mm < 2; ++mm) {
                const int i = i0 + mm * 128;
                if (i >= n_rows * 32) continue;
                const int rho = i >> 5, e = (i & 31) * 4;
                const long long orow = (long long)(q_off + rho / r) * H + kvh * r + rho % r;
                float mx = -CUDART_INF_F;
#pragma unroll
                for (int s2 = 0; s2 < kMgMaxAttSplits; ++s2) mx = fmaxf(mx, ml[mm][s2].x);
                float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
                float lsum = 0.f;
#pragma unroll
                for (int s2 = 0; s2 < kMgMaxAttSplits; ++s2) {
                  if (ml[mm][s2].x == -CUDART_INF_F) continue;
                  const float w = exp2f(ml[mm][s2].x - mx);
                  lsum += ml[mm][s2].y * w;
                  acc.x += po[mm][s2].x * w; acc.y += po[mm][s2].y * w; acc.z += po[mm][s2].z * w; acc.w += po[mm][s2].w * w;
                }
                const float inv = 1.f / lsum;
                __stcg(reinterpret_cast<uint2*>(p.attn + orow * kFaDh + e), make_uint2(pack_bf16(acc.x * inv, acc.y * inv), pack_bf16(acc.z * inv, acc.w * inv)));
              }
            }
          }
        }
        mg_bar128();                                        // sQ / K / V buffers are rewritten by the next unit
      }
      arrive();
    };

    const int* ns_qkv = nseg_tab, *ns_o = nseg_tab + kMgMaxTiles, *ns_gu = nseg_tab + 2 * kMgMaxTiles, *ns_dn = nseg_tab + 3 * kMgMaxTiles;
    for (int l = 0; l < L; ++l) {
      fold_norm(ns_dn, l > 0, p.u, nullptr);                // phase 7 l + 0 (the launch's first layer finds x complete)
      gemm_epilogue(0, p.part_a, p.NQKV, ns_qkv, p.layer0 + l);   //   1  (+ RoPE, Q and K/V page write by each tile's last CTA)
      attention(p.layer0 + l);                              //             2
      gemm_epilogue(1, p.part_x, p.d, ns_o, 0);             //             3
      fold_norm(ns_o, true, p.u2, p.xmid_dump);             //             4
      gemm_epilogue(2, p.part_a, 2 * p.F, ns_gu, 0);        //             5  (+ SwiGLU by each tile's last CTA)
      gemm_epilogue(3, p.part_x, p.d, ns_dn, 0);            //             6
    }
    fold_norm(ns_dn, true, nullptr, nullptr);               // the last layer's down slices into x (the head normalises its own rows)
  }
  pdl_launch_dependents();
  ptx::tc_fence_before();
  __syncthreads();
  if (threadIdx.x == 0) trace_end(p.tr);
  if (warp == 2) ptx::tmem_dealloc(tmem_base, tmem_cols);
}

}  // namespace dlm
