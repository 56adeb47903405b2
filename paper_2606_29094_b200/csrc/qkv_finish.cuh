// a4 fused behind the weight-streaming QKV projection (T <= 128 tokens): the CTA that completes a 128-column tile -- one
// head of Q, K or V -- sums the tile's fp32 split-K slices in slice order, rotates Q / K by the token's absolute position
// (half-split pairs (e, e + 64), table lookup; reading G12), rounds to bf16 and writes Q [T, H, 128] or the K / V rows of
// the request's pages.  Used by gemm_skinny_kernel (per-stage path) and layer_mega_kernel: both leave one slice
// [split][T][ld] per K range, and a per-tile arrival counter tells which CTA is the last.
#pragma once
#include "attn_flash.cuh"
#include "common.cuh"

namespace dlm {

struct QkvFinish {
  const float* part;          // slices [n][T][ld]
  long long slice_stride;     // T * ld
  int ld, T, HQ, n_heads;
  bf16* q;                    // [T, H, 128]
  bf16* kv_store;
  const float* rope_cos;      // [max_seq, 64]
  const float* rope_sin;
  const int* page_table;
  BatchDesc b;
  KvGeom g;
  unsigned int* tile_cnt;     // arrivals per tile, zero when the projection starts, reset by the finishing CTA
};

// 128 threads (tid 0..127) of one CTA; MS = most slices a tile can have
template <int MS>
__device__ __forceinline__ void qkv_finish_tile(const QkvFinish& f, int tile, int ns, int layer, int tid) {
  const int col0 = tile * 128, Hkv = f.g.n_kv_heads, H = f.n_heads, T = f.T;
  const int kind = col0 < f.HQ ? 0 : (col0 < f.HQ + Hkv * 128 ? 1 : 2);          // Q head | K head | V head
  const int head = kind == 0 ? tile : (kind == 1 ? tile - H : tile - H - Hkv);
  for (int i0 = tid; i0 < T * 16; i0 += 4 * 128) {        // item = (token, pair indices e .. e + 3 of [0, 64)); 4 items per pass
    float4 lo[4][MS], hi[4][MS], cs[4], sn[4];
    int pos[4], bi_[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) {                         // every load of the pass is issued before the first use
      const int i = i0 + m * 128;
      const bool ok = i < T * 16;
      const int t = ok ? i >> 4 : 0, e = (i & 15) * 4;
      const float* src = f.part + (long long)t * f.ld + col0 + e;
#pragma unroll
      for (int s = 0; s < MS; ++s) {
        lo[m][s] = (ok && s < ns) ? __ldcg(reinterpret_cast<const float4*>(src + s * f.slice_stride)) : make_float4(0.f, 0.f, 0.f, 0.f);
        hi[m][s] = (ok && s < ns) ? __ldcg(reinterpret_cast<const float4*>(src + s * f.slice_stride + 64)) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
      const int bi = f.b.tok_bi[t];
      bi_[m] = bi;
      pos[m] = f.b.q_pos0[bi] + (t - f.b.q_off[bi]);
      cs[m] = *reinterpret_cast<const float4*>(f.rope_cos + (long long)pos[m] * 64 + e);
      sn[m] = *reinterpret_cast<const float4*>(f.rope_sin + (long long)pos[m] * 64 + e);
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      const int i = i0 + m * 128;
      if (i >= T * 16) continue;
      const int t = i >> 4, e = (i & 15) * 4;
      float4 a = lo[m][0], c = hi[m][0];
#pragma unroll
      for (int s = 1; s < MS; ++s) {
        a.x += lo[m][s].x; a.y += lo[m][s].y; a.z += lo[m][s].z; a.w += lo[m][s].w;
        c.x += hi[m][s].x; c.y += hi[m][s].y; c.z += hi[m][s].z; c.w += hi[m][s].w;
      }
      if (kind < 2) {
        const float4 a2 = make_float4(a.x * cs[m].x - c.x * sn[m].x, a.y * cs[m].y - c.y * sn[m].y, a.z * cs[m].z - c.z * sn[m].z, a.w * cs[m].w - c.w * sn[m].w);
        c = make_float4(c.x * cs[m].x + a.x * sn[m].x, c.y * cs[m].y + a.y * sn[m].y, c.z * cs[m].z + a.z * sn[m].z, c.w * cs[m].w + a.w * sn[m].w);
        a = a2;
      }
      bf16* dst;
      if (kind == 0) {
        dst = f.q + ((long long)t * H + head) * 128 + e;
      } else {
        const int page = f.page_table[(long long)f.b.slot[bi_[m]] * f.g.max_pages_per_req + pos[m] / f.g.page_tokens];
        dst = f.kv_store + f.g.offset(layer, page, kind - 1, head, pos[m] % f.g.page_tokens) + e;
      }
      __stcg(reinterpret_cast<uint2*>(dst), make_uint2(pack_bf16(a.x, a.y), pack_bf16(a.z, a.w)));
      __stcg(reinterpret_cast<uint2*>(dst + 64), make_uint2(pack_bf16(c.x, c.y), pack_bf16(c.z, c.w)));
    }
  }
}

}  // namespace dlm
