// combine.cu — A4: split-KV combine.  For a row whose key range was cut into parts p, each part wrote a normalised
// partial output O_p and lse_p = ln sum_{t in part} exp(scale*<q,k_t>); since softmax over the union is the
// lse-weighted mean of the parts,
//     m = max_p lse_p ;  out = sum_p e^{lse_p - m} O_p / sum_p e^{lse_p - m} ;  lse = m + ln sum_p e^{lse_p - m}.
// (Not in the paper: BASELINE.json north_star "split-KV with a combine pass for long caches"; the formula is pinned
// against the unsplit definition in tests/test_oracle_pins.py.)  HBM-bound: (4*D + 4)*parts bytes read and 2*D written
// per row.  One CTA per (row block, head); a warp owns a row at a time, its 32 lanes split head_dim as float4.
#include <cuda_bf16.h>

#include "kernels.h"

namespace slack {
namespace {

constexpr int kCombineThreads = 256;

template <int D>
__global__ void __launch_bounds__(kCombineThreads)
combine_kernel(const DevCombine *__restrict__ combines, const float *__restrict__ ws_o, const float *__restrict__ ws_lse,
               __nv_bfloat16 *__restrict__ out, float *__restrict__ lse, int n_heads, int total_q) {
  constexpr int E = D / 32;
  const DevCombine cb = combines[blockIdx.x];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int r = warp; r < cb.q_rows; r += kCombineThreads / 32) {
    float m = -INFINITY;
    for (int p = 0; p < cb.n_parts; ++p) m = fmaxf(m, ws_lse[(size_t)(cb.slot_begin + p) * kItemRows + r]);
    float den = 0.f, acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.f;
    for (int p = 0; p < cb.n_parts; ++p) {
      const size_t slot = (size_t)(cb.slot_begin + p);
      const float w = expf(ws_lse[slot * kItemRows + r] - m);
      den += w;
      const float *src = ws_o + (slot * kItemRows + r) * D + lane * E;
#pragma unroll
      for (int e = 0; e < E; ++e) acc[e] = fmaf(w, src[e], acc[e]);
    }
    const float inv = 1.0f / den;
    __nv_bfloat16 *dst = out + ((size_t)(cb.q_row0 + r) * n_heads + cb.head) * D + lane * E;
#pragma unroll
    for (int e = 0; e < E; e += 2) {
      __nv_bfloat162 v = __floats2bfloat162_rn(acc[e] * inv, acc[e + 1] * inv);
      *reinterpret_cast<__nv_bfloat162 *>(dst + e) = v;
    }
    if (lse != nullptr && lane == 0) lse[(size_t)cb.head * total_q + cb.q_row0 + r] = m + logf(den);
  }
}

} // namespace

cudaError_t launch_combine(const DevCombine *d_combines, int n_combines, const float *ws_o, const float *ws_lse, void *out,
                           float *lse, int n_heads, int head_dim, int total_q, cudaStream_t st, int *n_launched) {
  if (n_combines == 0) return cudaSuccess;
  if (head_dim != 128) return cudaErrorInvalidValue;
  combine_kernel<128><<<n_combines, kCombineThreads, 0, st>>>(d_combines, ws_o, ws_lse,
                                                              reinterpret_cast<__nv_bfloat16 *>(out), lse, n_heads, total_q);
  if (n_launched) *n_launched += 1;
  return cudaGetLastError();
}

} // namespace slack
