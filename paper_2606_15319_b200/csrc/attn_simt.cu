// attn_simt.cu — A3, validation / fp32 path: the definition in include/slack.h evaluated with CUDA cores and fp32
// accumulation, for any page size and both storage dtypes.  It serves fp32 pools (BASELINE.json config 1) and is the
// on-GPU cross-check of the tensor-core kernel (slack_plan_opts.force_simt).  One warp per (query row, head); the 32
// lanes split head_dim, keys are visited in position order through the page table, softmax is the
// streaming (running max / running sum) form of softmax_t(scale * <q, k_t>).
#include <cuda_bf16.h>

#include "kernels.h"

namespace slack {
namespace {

constexpr int kSimtThreads = 128;

template <typename T> __device__ __forceinline__ float to_f32(T x);
template <> __device__ __forceinline__ float to_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f32(float x);
template <> __device__ __forceinline__ float from_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

template <typename T, int D>
__global__ void __launch_bounds__(kSimtThreads)
attn_simt_kernel(const T *__restrict__ q, const T *__restrict__ k_pool, const T *__restrict__ v_pool, T *__restrict__ out,
                 float *__restrict__ lse, const DevStream *__restrict__ streams, int n_streams, int total_q,
                 const int32_t *__restrict__ page_tables, int n_heads, int page_log2, float scale,
                 const uint32_t *__restrict__ mask, int mask_words) {
  constexpr int E = D / 32; // elements per lane
  const int lane = threadIdx.x & 31;
  const long long unit = (long long)blockIdx.x * (kSimtThreads / 32) + (threadIdx.x >> 5);
  if (unit >= (long long)total_q * n_heads) return;
  const int row = (int)(unit / n_heads);
  const int h = (int)(unit % n_heads);
  // stream of this row (streams are in row order; empty streams have q_len 0)
  int lo_i = 0, hi_i = n_streams - 1;
  while (lo_i < hi_i) {
    const int mid = (lo_i + hi_i + 1) >> 1;
    if (streams[mid].q_row0 <= row) lo_i = mid; else hi_i = mid - 1;
  }
  while (streams[lo_i].q_len == 0 || row >= streams[lo_i].q_row0 + streams[lo_i].q_len) --lo_i; // skip empty successors sharing q_row0
  const DevStream s = streams[lo_i];
  const int32_t *pt = page_tables + s.pt_off;
  const int page_mask = (1 << page_log2) - 1;

  float qv[E], acc[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    qv[e] = to_f32<T>(q[((long long)row * n_heads + h) * D + lane * E + e]);
    acc[e] = 0.f;
  }
  // block-sparse variant (P:88 knob (2)): bit t of this (256-row query block, head)'s mask row = key block t selected
  const uint32_t *mrow = mask ? mask + ((size_t)(s.qblock0 + (row - s.q_row0) / kItemRows) * n_heads + h) * mask_words : nullptr;
  float m = -INFINITY, l = 0.f;
  // visible positions: the sink [base, sink_hi) (empty unless the window has left it behind), then [pos_lo, pos_hi)
  const int n_sink = s.sink_hi - s.base;
  const int n_vis = n_sink + (s.pos_hi - s.pos_lo);
  for (int t = 0; t < n_vis; ++t) {
    const int pos = t < n_sink ? s.base + t : s.pos_lo + (t - n_sink);
    if (mrow != nullptr && !((__ldg(mrow + (pos / kTileN >> 5)) >> ((pos / kTileN) & 31)) & 1u)) continue;
    const long long page = pt[pos >> page_log2];
    const long long off = ((((page * n_heads + h) << page_log2) + (pos & page_mask)) * D) + lane * E;
    float dot = 0.f;
#pragma unroll
    for (int e = 0; e < E; ++e) dot = fmaf(qv[e], to_f32<T>(k_pool[off + e]), dot);
#pragma unroll
    for (int sh = 16; sh > 0; sh >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, sh);
    const float sc = dot * scale;
    const float m_new = fmaxf(m, sc);
    const float alpha = expf(m - m_new); // exp(-inf) = 0 on the first key
    const float pr = expf(sc - m_new);
    l = l * alpha + pr;
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = fmaf(pr, to_f32<T>(v_pool[off + e]), acc[e] * alpha);
    m = m_new;
  }
  const float inv = l > 0.f ? 1.0f / l : 0.f; // no selected key (block-sparse only): out = 0, lse = -inf
#pragma unroll
  for (int e = 0; e < E; ++e) out[((long long)row * n_heads + h) * D + lane * E + e] = from_f32<T>(acc[e] * inv);
  if (lse != nullptr && lane == 0) lse[(long long)h * total_q + row] = m + logf(l);
}

int ilog2(int x) {
  int l = 0;
  while ((1 << l) < x) ++l;
  return l;
}

} // namespace

cudaError_t launch_attn_simt(int dtype, const void *q, const void *k_pool, const void *v_pool, void *out, float *lse,
                             const DevStream *d_streams, int n_streams, int total_q, const int32_t *d_page_tables,
                             int n_heads, int head_dim, int page_size, float scale, const uint32_t *mask, int mask_words,
                             cudaStream_t st, int *n_launched) {
  if (total_q == 0) return cudaSuccess;
  const long long units = (long long)total_q * n_heads;
  const int wpb = kSimtThreads / 32;
  const unsigned grid = (unsigned)((units + wpb - 1) / wpb);
  const int pl = ilog2(page_size);
#define SLACK_SIMT_LAUNCH(T, D)                                                                                          \
  attn_simt_kernel<T, D><<<grid, kSimtThreads, 0, st>>>(reinterpret_cast<const T *>(q), reinterpret_cast<const T *>(k_pool), \
                                                        reinterpret_cast<const T *>(v_pool), reinterpret_cast<T *>(out), lse, \
                                                        d_streams, n_streams, total_q, d_page_tables, n_heads, pl, scale, mask, mask_words)
  if (dtype == SLACK_F32 && head_dim == 64) SLACK_SIMT_LAUNCH(float, 64);
  else if (dtype == SLACK_F32 && head_dim == 128) SLACK_SIMT_LAUNCH(float, 128);
  else if (dtype == SLACK_BF16 && head_dim == 64) SLACK_SIMT_LAUNCH(__nv_bfloat16, 64);
  else if (dtype == SLACK_BF16 && head_dim == 128) SLACK_SIMT_LAUNCH(__nv_bfloat16, 128);
  else return cudaErrorInvalidValue;
#undef SLACK_SIMT_LAUNCH
  if (n_launched) *n_launched += 1;
  return cudaGetLastError();
}

} // namespace slack
