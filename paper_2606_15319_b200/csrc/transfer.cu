// transfer.cu — NEXT-4: state-plane page transfer, "transfer(stream, src, dst, page_range)" (§4.4), the one
// primitive behind credit-aware eviction, re-homing and elastic SP; issued layer-major so that the destination can start
// layer k as soon as layer k's pages have arrived, and head-partition-aware (only the donor worker's
// head partition of the KV pages moves).
//
// One launch per layer: page src_ids[i] of the source pool becomes page dst_ids[i] of the destination pool, heads
// [h0, h1) only.  In the pool layout [n_pages][H][P][D] the head slice [h0, h1) of one page is ONE contiguous run of
// (h1 - h0) * P * D elements, so the copy is a plain 16-byte-vector stream per page (blockIdx.y = page, grid-stride in x),
// HBM-bound: 2 (K, V) x 2 (read + write) x pages x (h1 - h0) x P x D x elem bytes per layer.  Source and destination are
// addressed through unified virtual addresses, so either pool may live in this GPU's HBM, in pinned host memory
// (eviction / offload) or in a peer GPU's HBM with peer access enabled (re-homing, elastic SP over NVLink); only the
// first two can be exercised on a one-GPU box.
#include "kernels.h"

namespace slack {
namespace {

constexpr int kXferThreads = 256;
constexpr int kXferUnroll = 4;

__global__ void __launch_bounds__(kXferThreads)
kv_transfer_kernel(const uint4 *__restrict__ src_k, const uint4 *__restrict__ src_v, uint4 *__restrict__ dst_k,
                   uint4 *__restrict__ dst_v, const int32_t *__restrict__ src_ids, const int32_t *__restrict__ dst_ids,
                   long long page_vecs /* 16-byte vectors per whole page (all heads) */,
                   long long slice_off /* vectors from the page start to head h0 */,
                   long long slice_vecs /* vectors in heads [h0, h1) */) {
  const long long s0 = (long long)src_ids[blockIdx.y] * page_vecs + slice_off;
  const long long d0 = (long long)dst_ids[blockIdx.y] * page_vecs + slice_off;
  const long long stride = (long long)gridDim.x * kXferThreads;
  for (long long u0 = (long long)blockIdx.x * kXferThreads + threadIdx.x; u0 < slice_vecs; u0 += stride * kXferUnroll) {
    uint4 kk[kXferUnroll], vv[kXferUnroll];
#pragma unroll
    for (int j = 0; j < kXferUnroll; ++j) {
      const long long u = u0 + j * stride;
      if (u < slice_vecs) {
        kk[j] = __ldcs(src_k + s0 + u);
        vv[j] = __ldcs(src_v + s0 + u);
      }
    }
#pragma unroll
    for (int j = 0; j < kXferUnroll; ++j) {
      const long long u = u0 + j * stride;
      if (u < slice_vecs) {
        __stcs(dst_k + d0 + u, kk[j]);
        __stcs(dst_v + d0 + u, vv[j]);
      }
    }
  }
}

// FP8 pools (include/slack.h slack_dtype): the scales of the moved (page, head) slices travel with the codes.  Scales are
// fp32 [n_pages][H][P / 128]; one thread per (page, head in [h0, h1), block).
__global__ void __launch_bounds__(kXferThreads)
kv_scale_transfer_kernel(const float *__restrict__ src_k, const float *__restrict__ src_v, float *__restrict__ dst_k,
                         float *__restrict__ dst_v, const int32_t *__restrict__ src_ids, const int32_t *__restrict__ dst_ids,
                         int n_pages, int n_heads, int blocks_per_page, int h0, int h1) {
  const int per_page = (h1 - h0) * blocks_per_page;
  const long long n = (long long)n_pages * per_page;
  for (long long u = (long long)blockIdx.x * kXferThreads + threadIdx.x; u < n; u += (long long)gridDim.x * kXferThreads) {
    const int pg = (int)(u / per_page), r = (int)(u % per_page);
    const long long off = (long long)h0 * blocks_per_page + r;
    const long long s = (long long)src_ids[pg] * n_heads * blocks_per_page + off;
    const long long d = (long long)dst_ids[pg] * n_heads * blocks_per_page + off;
    dst_k[d] = src_k[s];
    dst_v[d] = src_v[s];
  }
}

} // namespace

cudaError_t launch_kv_scale_transfer(const float *src_k, const float *src_v, float *dst_k, float *dst_v, const int32_t *d_src_ids,
                                     const int32_t *d_dst_ids, int n_pages, int n_heads, int page_size, int head_begin,
                                     int head_end, cudaStream_t st, int *n_launched) {
  if (n_pages == 0 || head_end <= head_begin) return cudaSuccess;
  const int bpp = page_size / 128;
  const long long n = (long long)n_pages * (head_end - head_begin) * bpp;
  const int grid = (int)((n + kXferThreads - 1) / kXferThreads < 1024 ? (n + kXferThreads - 1) / kXferThreads : 1024);
  kv_scale_transfer_kernel<<<grid, kXferThreads, 0, st>>>(src_k, src_v, dst_k, dst_v, d_src_ids, d_dst_ids, n_pages, n_heads, bpp,
                                                           head_begin, head_end);
  if (n_launched) *n_launched += 1;
  return cudaGetLastError();
}

cudaError_t launch_kv_transfer(const void *src_k, const void *src_v, void *dst_k, void *dst_v, const int32_t *d_src_ids,
                               const int32_t *d_dst_ids, int n_pages, int n_heads, int head_dim, int page_size,
                               int elem_bytes, int head_begin, int head_end, int sm_count, cudaStream_t st,
                               int *n_launched) {
  if (n_pages == 0 || head_end <= head_begin) return cudaSuccess;
  const long long head_vecs = (long long)page_size * head_dim * elem_bytes / 16;
  const long long slice_vecs = head_vecs * (head_end - head_begin);
  long long want = (slice_vecs + (long long)kXferThreads * kXferUnroll - 1) / ((long long)kXferThreads * kXferUnroll);
  long long cap = ((long long)sm_count * 8 + n_pages - 1) / n_pages; // ~8 CTAs per SM over the whole grid
  if (cap < 1) cap = 1;
  const int gx = (int)(want < cap ? want : cap);
  constexpr int kMaxGridY = 65535; // gridDim.y limit: longer page lists go out in several launches (same stream, in order)
  for (int p0 = 0; p0 < n_pages; p0 += kMaxGridY) {
    const int np = n_pages - p0 < kMaxGridY ? n_pages - p0 : kMaxGridY;
    kv_transfer_kernel<<<dim3(gx > 0 ? gx : 1, np), kXferThreads, 0, st>>>(
        reinterpret_cast<const uint4 *>(src_k), reinterpret_cast<const uint4 *>(src_v), reinterpret_cast<uint4 *>(dst_k),
        reinterpret_cast<uint4 *>(dst_v), d_src_ids + p0, d_dst_ids + p0, head_vecs * n_heads, head_vecs * head_begin, slice_vecs);
    if (n_launched) *n_launched += 1;
  }
  return cudaGetLastError();
}

} // namespace slack
