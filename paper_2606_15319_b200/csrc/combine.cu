// combine.cu — A4: split-KV combine.  For a row whose key range was cut into parts p, each part wrote a normalised
// partial output O_p and lse_p = ln sum_{t in part} exp(scale*<q,k_t>); since softmax over the union is the
// lse-weighted mean of the parts,
//     m = max_p lse_p ;  out = sum_p e^{lse_p - m} O_p / sum_p e^{lse_p - m} ;  lse = m + ln sum_p e^{lse_p - m}.
// (Not in the paper: BASELINE.json north_star "split-KV with a combine pass for long caches"; the formula is pinned
// against the unsplit definition in tests/test_oracle_pins.py.)  HBM-bound: (4*D + 4)*parts bytes read and 2*D written
// per row.  Grid = (combine entries, 256 / kRowsPerCta); a warp owns one row, its 32 lanes split head_dim (float4 each at 128, float2 at 64), and
// the loads of all parts of a row are independent (the partials were just written and mostly still sit in L2).
#include <cuda_bf16.h>

#include <type_traits>

#include "kernels.h"

namespace slack {
namespace {

constexpr int kCombineThreads = 256;
constexpr int kRowsPerCta = kCombineThreads / 32; // one row per warp
constexpr int kMaxPartsUnrolled = 4;

template <int D>
__global__ void __launch_bounds__(kCombineThreads)
combine_kernel(const DevCombine *__restrict__ combines, const float *__restrict__ ws_o, const float *__restrict__ ws_lse,
               __nv_bfloat16 *__restrict__ out, float *__restrict__ lse, int n_heads, int total_q) {
  static_assert(D == 128 || D == 64, "one float4 / float2 per lane");
  constexpr int kV = D / 32;                                          // fp32 values per lane
  using Vec = typename std::conditional<kV == 4, float4, float2>::type;
  auto ld = [](const Vec *q, float (&v)[kV]) {
    const Vec t = __ldg(q);
    v[0] = t.x, v[1] = t.y;
    if constexpr (kV == 4) v[2] = t.z, v[3] = t.w;
  };
  pdl_wait(); // the partials are written by the attention kernel right before
  pdl_launch_dependents();
  const DevCombine cb = combines[blockIdx.x];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r = blockIdx.y * kRowsPerCta + warp;
  if (r >= cb.q_rows) return;
  const float *lse_p = ws_lse + (size_t)cb.slot_begin * kItemRows + r;
  const Vec *o_p = reinterpret_cast<const Vec *>(ws_o + ((size_t)cb.slot_begin * kItemRows + r) * D) + lane;
  constexpr size_t kSlotStride4 = (size_t)kItemRows * D / kV;
  float m = -INFINITY;
  for (int p = 0; p < cb.n_parts; ++p) m = fmaxf(m, __ldg(lse_p + (size_t)p * kItemRows));
  if (m == -INFINITY) { // block-sparse: no part of this row had a selected key -> out = 0, lse = -inf
    __nv_bfloat16 *z = out + ((size_t)(cb.q_row0 + r) * n_heads + cb.head) * D + lane * kV;
    if constexpr (kV == 4) *reinterpret_cast<uint2 *>(z) = make_uint2(0u, 0u);
    else *reinterpret_cast<uint32_t *>(z) = 0u;
    if (lse != nullptr && lane == 0) lse[(size_t)cb.head * total_q + cb.q_row0 + r] = -INFINITY;
    return;
  }
  float den = 0.f;
  float acc[kV] = {};
  int p = 0;
  for (; p + kMaxPartsUnrolled <= cb.n_parts; p += kMaxPartsUnrolled) { // batches of independent loads
    float v[kMaxPartsUnrolled][kV];
    float w[kMaxPartsUnrolled];
#pragma unroll
    for (int u = 0; u < kMaxPartsUnrolled; ++u) {
      ld(o_p + (size_t)(p + u) * kSlotStride4, v[u]);
      w[u] = __ldg(lse_p + (size_t)(p + u) * kItemRows);
    }
#pragma unroll
    for (int u = 0; u < kMaxPartsUnrolled; ++u) {
      const float e = expf(w[u] - m);
      den += e;
#pragma unroll
      for (int c = 0; c < kV; ++c) acc[c] = fmaf(e, v[u][c], acc[c]);
    }
  }
  for (; p < cb.n_parts; ++p) {
    float v[kV];
    ld(o_p + (size_t)p * kSlotStride4, v);
    const float e = expf(__ldg(lse_p + (size_t)p * kItemRows) - m);
    den += e;
#pragma unroll
    for (int c = 0; c < kV; ++c) acc[c] = fmaf(e, v[c], acc[c]);
  }
  const float inv = 1.0f / den;
  __nv_bfloat16 *dst = out + ((size_t)(cb.q_row0 + r) * n_heads + cb.head) * D + lane * kV;
  const __nv_bfloat162 lo = __floats2bfloat162_rn(acc[0] * inv, acc[1] * inv);
  if constexpr (kV == 4) {
    const __nv_bfloat162 hi = __floats2bfloat162_rn(acc[2] * inv, acc[3] * inv);
    uint2 o;
    o.x = *reinterpret_cast<const uint32_t *>(&lo);
    o.y = *reinterpret_cast<const uint32_t *>(&hi);
    *reinterpret_cast<uint2 *>(dst) = o;
  } else {
    *reinterpret_cast<uint32_t *>(dst) = *reinterpret_cast<const uint32_t *>(&lo);
  }
  if (lse != nullptr && lane == 0) lse[(size_t)cb.head * total_q + cb.q_row0 + r] = m + logf(den);
}

} // namespace

cudaError_t launch_combine(const DevCombine *d_combines, int n_combines, const float *ws_o, const float *ws_lse, void *out,
                           float *lse, int n_heads, int head_dim, int total_q, cudaStream_t st, int *n_launched) {
  if (n_combines == 0) return cudaSuccess;
  if (head_dim != 128 && head_dim != 64) return cudaErrorInvalidValue;
  const dim3 grid((unsigned)n_combines, kItemRows / kRowsPerCta);
  cudaError_t e = head_dim == 128 ? launch_pdl(combine_kernel<128>, grid, dim3(kCombineThreads), 0, st, d_combines, ws_o, ws_lse,
                                               reinterpret_cast<__nv_bfloat16 *>(out), lse, n_heads, total_q)
                                  : launch_pdl(combine_kernel<64>, grid, dim3(kCombineThreads), 0, st, d_combines, ws_o, ws_lse,
                                               reinterpret_cast<__nv_bfloat16 *>(out), lse, n_heads, total_q);
  if (n_launched) *n_launched += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace slack
