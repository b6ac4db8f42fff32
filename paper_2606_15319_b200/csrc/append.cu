// append.cu — A1: KV append, "appended to a rolling KV cache for subsequent chunks" (§2.1), into the
// paged pool of P:251 §4.4.  Pure 16-byte-vector scatter copy, HBM-bound: 8*Lq*H*D*elem bytes moved per call
// (read + write, K and V).  Source rows are token-major [row][h][d] and therefore contiguous in the unit index;
// destination of (token, head) is the contiguous head_dim run at ((page*H + h)*P + slot)*D of the token->slot rule
// in include/slack.h.  blockIdx.y = stream, grid-stride over the stream's 16-byte units in x.
#include "kernels.h"

namespace slack {
namespace {

constexpr int kAppendThreads = 256;
constexpr int kUnroll = 4;

__global__ void __launch_bounds__(kAppendThreads)
kv_append_kernel(const uint4 *__restrict__ k_new, const uint4 *__restrict__ v_new, uint4 *__restrict__ k_pool,
                 uint4 *__restrict__ v_pool, const DevStream *__restrict__ streams,
                 const int32_t *__restrict__ page_tables, int n_heads, int page_log2, int vec_log2 /* log2(16-byte vectors per (token, head) row) */) {
  pdl_wait(); // K_new / V_new may come from the kernel before; the pool may still be read by the previous layer's attention
  pdl_launch_dependents();
  const DevStream s = streams[blockIdx.y];
  if (s.q_len == 0) return;
  const int vecs = 1 << vec_log2;
  const int page_mask = (1 << page_log2) - 1;
  const long long row_units = (long long)n_heads << vec_log2;            // units per token
  const long long units = (long long)s.q_len * row_units;
  const long long src0 = (long long)s.q_row0 * row_units;
  const long long stride = (long long)gridDim.x * kAppendThreads;
  const int32_t *pt = page_tables + s.pt_off;
  for (long long u0 = (long long)blockIdx.x * kAppendThreads + threadIdx.x; u0 < units; u0 += stride * kUnroll) {
    uint4 kk[kUnroll], vv[kUnroll];
    long long dst[kUnroll];
#pragma unroll
    for (int j = 0; j < kUnroll; ++j) {
      const long long u = u0 + j * stride;
      dst[j] = -1;
      if (u < units) {
        kk[j] = __ldcs(k_new + src0 + u);
        vv[j] = __ldcs(v_new + src0 + u);
        const int tok = (int)(u / row_units);
        const int rem = (int)(u - (long long)tok * row_units);
        const int h = rem >> vec_log2;
        const int c = rem & (vecs - 1);
        const int pos = s.app_pos0 + tok;
        const long long page = pt[pos >> page_log2];
        const int slot = pos & page_mask;
        dst[j] = ((((page * n_heads + h) << page_log2) + slot) << vec_log2) + c;
      }
    }
#pragma unroll
    for (int j = 0; j < kUnroll; ++j) {
      if (dst[j] >= 0) {
        k_pool[dst[j]] = kk[j];
        v_pool[dst[j]] = vv[j];
      }
    }
  }
}

int ilog2(int x) {
  int l = 0;
  while ((1 << l) < x) ++l;
  return l;
}

} // namespace

cudaError_t launch_kv_append(const void *k_new, const void *v_new, void *k_pool, void *v_pool, const DevStream *d_streams,
                             int n_streams, int max_q_len, const int32_t *d_page_tables, int n_heads, int head_dim,
                             int page_size, int elem_bytes, int sm_count, cudaStream_t st, int *n_launched) {
  if (n_streams == 0 || max_q_len == 0) return cudaSuccess;
  const int vecs = head_dim * elem_bytes / 16;
  const long long units_max = (long long)max_q_len * n_heads * vecs;
  long long want = (units_max + (long long)kAppendThreads * kUnroll - 1) / ((long long)kAppendThreads * kUnroll);
  // enough CTAs in flight to cover HBM latency (about 8 per SM over the whole grid), never more than the work needs
  long long cap = ((long long)sm_count * 8 + n_streams - 1) / n_streams;
  if (cap < 1) cap = 1;
  const int gx = (int)(want < cap ? want : cap);
  constexpr int kMaxGridY = 65535; // gridDim.y limit: larger batches go out in several launches (same stream, in order)
  cudaError_t e = cudaSuccess;
  for (int s0 = 0; s0 < n_streams && e == cudaSuccess; s0 += kMaxGridY) {
    const int ns = n_streams - s0 < kMaxGridY ? n_streams - s0 : kMaxGridY;
    e = launch_pdl(kv_append_kernel, dim3(gx > 0 ? gx : 1, ns), dim3(kAppendThreads), 0, st, reinterpret_cast<const uint4 *>(k_new),
                   reinterpret_cast<const uint4 *>(v_new), reinterpret_cast<uint4 *>(k_pool), reinterpret_cast<uint4 *>(v_pool),
                   d_streams + s0, d_page_tables, n_heads, ilog2(page_size), ilog2(vecs));
    if (n_launched) *n_launched += 1;
  }
  return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace slack
