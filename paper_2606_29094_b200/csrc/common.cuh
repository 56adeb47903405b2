// Shared declarations of the denoising-step engine (device helpers, launch bookkeeping).
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

namespace dlm {

typedef __nv_bfloat16 bf16;

__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(bf16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ bf16 from_f32<bf16>(float v) { return __float2bfloat16_rn(v); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Programmatic dependent launch (PDL): every kernel of a step lets its successor start early and waits for its
// predecessor's results right before it first touches them.  Both are no-ops for a plain launch.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Per-step ragged batch descriptor, built on the host, copied once per step (a0 in DESIGN.md).
// Request i of the batch computes q_len[i] consecutive positions starting at absolute position q_pos0[i];
// its rows live at [q_off[i], q_off[i]+q_len[i]) of every [T, *] activation buffer.
struct BatchDesc {
  int n;             // requests
  int T;             // computed tokens (sum q_len)
  int R;             // rows that need logits (sum blk_len)
  int max_q_len;     // max over requests (attention grid sizing)
  int max_kv_len;
  int min_q_len;     // min over requests that compute anything (mixed steps: block rows of the cached requests)
  int n_big;         // requests with more than 64 stacked query rows per KV head: they come first in `order`
  int qt_big, qt_total; // 128-row query tiles of the first n_big / of all requests of `order` (qt_off[n_big], qt_off[n])
  const int* slot;   // [n] request slot (row of tokens / page table)
  const int* q_off;  // [n]
  const int* q_len;  // [n]
  const int* q_pos0; // [n]
  const int* kv_len; // [n] S_r
  const int* blk_lo; // [n] absolute position of the current block's first token
  const int* blk_len;// [n] B_r (0 for a finished request)
  const int* row_off;// [n] offset of the request's block rows in the [R, *] buffers
  const float* tau;  // [n]
  const int* tok_bi; // [T] batch index of each computed token
  const int* qt_off; // [n + 1] prefix sums, over `order`, of the requests' 128-row query tiles (nullptr: q_tiles_max each)
  const int* order;  // [n] batch indices: the n_big requests first, each group by decreasing K/V length (work order of the attention kernels)
};

// Paged K/V store geometry: [layer][page][K|V][H_kv][page_tokens][d_h]
struct KvGeom {
  int n_kv_heads, head_dim, page_tokens, max_pages_per_req;
  long long n_pages;
  __host__ __device__ long long page_elems() const { return 2LL * n_kv_heads * page_tokens * head_dim; }
  __host__ __device__ long long offset(int layer, int page, int kv, int head, int tok_in_page) const {
    return ((((long long)layer * n_pages + page) * 2 + kv) * n_kv_heads + head) * (long long)page_tokens * head_dim +
           (long long)tok_in_page * head_dim;
  }
};

// Per-thread launch bookkeeping: a ctx is used from one thread at a time, so the entry points (DevGuard in engine.cu) bind
// the thread to the context's device and credit the kernels launched in between to that context (dlm_launch_count).
extern thread_local long long g_launches;   // kernels launched by this thread
extern thread_local int g_num_sms;          // SM count of the device the thread is bound to
extern thread_local int g_dev;              // that device's ordinal (index of the per-device one-time kernel configuration)
constexpr int kMaxDevices = 64;

#define DLM_LAUNCH_CHECK() do { ::dlm::g_launches++; } while (0)

// In-kernel timeline (DLM_OPT_TRACE): every launch of a step owns one record of three 64-bit words in global memory,
//   [0] min over CTAs of %globaltimer at kernel entry, [1] min of the time griddepcontrol.wait returned (= the upstream
//   kernel has completed), [2] min of ~%globaltimer at exit (i.e. the complement of the latest exit).
// A null pointer (tracing off, the default) costs one predicated branch per CTA.  Works under CUDA-graph replay and
// programmatic dependent launch, where host-side events cannot separate overlapping kernels.
struct TraceSlot { unsigned long long* p; };
__device__ __forceinline__ unsigned long long gtimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ void trace_begin(const TraceSlot& tr) { if (tr.p) atomicMin(tr.p, gtimer_ns()); }
__device__ __forceinline__ void trace_wait(const TraceSlot& tr) { if (tr.p) atomicMin(tr.p + 1, gtimer_ns()); }
__device__ __forceinline__ void trace_end(const TraceSlot& tr) { if (tr.p) atomicMin(tr.p + 2, ~gtimer_ns()); }
// prologue of the small kernels: let the successor start, stamp, wait for the predecessor, stamp
#define DLM_PROLOGUE(tr) do { pdl_launch_dependents(); if (threadIdx.x == 0) trace_begin(tr); pdl_wait(); if (threadIdx.x == 0) trace_wait(tr); } while (0)
#define DLM_EPILOGUE(tr) do { if (threadIdx.x == 0) trace_end(tr); } while (0)

}  // namespace dlm
