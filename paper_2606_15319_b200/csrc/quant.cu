// quant.cu — NEXT-3 (PAPER.md P:88 knob (4) "quantization mode Q", "online FP8 attention
// quantization"): the two quantisers of the FP8 path.  The rule is include/slack.h's (slack_dtype) and DESIGN.md A19:
// OCP e4m3, round to nearest even, saturating; code = e4m3(fp32(x) / scale) with scale = amax / 448 (amax = 0 -> 1), both
// divisions IEEE fp32 (__fdiv_rn), so that codes and scales are bit-exact against the oracle.
//
//   kv_append_fp8_kernel  A1 for FP8 pools: one CTA per (key block of 128 slots, head, stream x {K, V}); a block whose
//                         first held token this append writes gets its scale from the tokens written, any other
//                         block keeps the stored scale.  The block's rows (<= 128 x 256 B) stay in registers between
//                         the amax and the conversion: HBM-bound, 2 * Lq * H * D * 2 B read once, half of that written.
//   q_quant_kernel        Q of an attention call -> codes [sum Lq][H][128] + scales [H][sum Lq] in the workspace;
//                         one warp per (row, head).
#include <cuda_bf16.h>

#include "kernels.h"

namespace slack {
namespace {

constexpr int kQuantThreads = 256;
constexpr float kE4m3Max = 448.0f;

__device__ __forceinline__ uint32_t e4m3x2(float lo, float hi) { // lo in bits [0,8), hi in bits [8,16)
  uint16_t d;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// one lane's 4 consecutive head_dim elements (8 bytes of bf16) -> 4 codes, and their largest magnitude
__device__ __forceinline__ float amax4(uint2 v) {
  return fmaxf(fmaxf(fabsf(bf16_lo(v.x)), fabsf(bf16_hi(v.x))), fmaxf(fabsf(bf16_lo(v.y)), fabsf(bf16_hi(v.y))));
}
__device__ __forceinline__ uint32_t quant4(uint2 v, float scale) {
  const uint32_t a = e4m3x2(__fdiv_rn(bf16_lo(v.x), scale), __fdiv_rn(bf16_hi(v.x), scale));
  const uint32_t b = e4m3x2(__fdiv_rn(bf16_lo(v.y), scale), __fdiv_rn(bf16_hi(v.y), scale));
  return a | (b << 16);
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

__global__ void __launch_bounds__(kQuantThreads)
kv_append_fp8_kernel(const uint2 *__restrict__ k_new, const uint2 *__restrict__ v_new, uint32_t *__restrict__ k_pool,
                     uint32_t *__restrict__ v_pool, float *__restrict__ k_scale, float *__restrict__ v_scale,
                     const DevStream *__restrict__ streams, const int32_t *__restrict__ page_tables, int n_heads, int page_log2) {
  pdl_wait();
  pdl_launch_dependents();
  const DevStream s = streams[blockIdx.z >> 1];
  if (s.q_len == 0) return;
  const bool is_v = blockIdx.z & 1;
  const int h = blockIdx.y;
  const int kb = (s.app_pos0 >> 7) + blockIdx.x; // key block in the stream's position space
  const int p_first = max(kb << 7, s.app_pos0), p_last = min((kb << 7) + 128, s.app_pos0 + s.q_len); // positions written here
  if (p_first >= p_last) return;
  const uint2 *src = is_v ? v_new : k_new;
  uint32_t *pool = is_v ? v_pool : k_pool;
  float *scales = is_v ? v_scale : k_scale;
  const int page = page_tables[s.pt_off + ((kb << 7) >> page_log2)];
  const int blocks_per_page = 1 << (page_log2 - 7);
  float *scale_ptr = scales + ((size_t)page * n_heads + h) * blocks_per_page + (((kb << 7) & ((1 << page_log2) - 1)) >> 7);
  // none of the stream's earlier tokens lies in this block -> this append starts it and sets its scale
  const int b_lo = kb << 7, b_hi = b_lo + 128;
  const bool has_old = (s.base < b_hi && s.old_hi0 > b_lo && s.old_hi0 > s.base) || (s.old_lo1 < b_hi && s.app_pos0 > b_lo && s.app_pos0 > s.old_lo1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_tok = p_last - p_first;
  const int tok0 = p_first - s.app_pos0; // chunk-local index of the first token written here
  // source row of (token, head): 128 bf16 = 32 lanes x 8 bytes
  auto src_of = [&](int t) { return src + ((size_t)(s.q_row0 + tok0 + t) * n_heads + h) * 32 + lane; };
  // every warp keeps its (at most 16) token rows in registers: the source is read from HBM once
  constexpr int kWarps = kQuantThreads / 32, kRowsPerWarp = 128 / kWarps;
  uint2 rows[kRowsPerWarp];
  float am = 0.f;
#pragma unroll
  for (int r = 0; r < kRowsPerWarp; ++r) {
    const int t = warp + r * kWarps;
    rows[r] = t < n_tok ? __ldcs(src_of(t)) : make_uint2(0u, 0u);
    am = fmaxf(am, amax4(rows[r]));
  }
  __shared__ float red[kWarps];
  __shared__ float scale_sh;
  if (!has_old) {
    am = warp_max(am);
    if (lane == 0) red[warp] = am;
    __syncthreads();
    if (threadIdx.x == 0) {
      float a = red[0];
#pragma unroll
      for (int w = 1; w < kWarps; ++w) a = fmaxf(a, red[w]);
      const float sc = a > 0.f ? __fdiv_rn(a, kE4m3Max) : 1.0f;
      scale_sh = sc;
      *scale_ptr = sc;
    }
  } else if (threadIdx.x == 0) {
    scale_sh = *scale_ptr;
  }
  __syncthreads();
  const float sc = scale_sh;
  // destination row of position p, head h: 128 codes = 32 lanes x 4 bytes
  const int page_mask = (1 << page_log2) - 1;
#pragma unroll
  for (int r = 0; r < kRowsPerWarp; ++r) {
    const int t = warp + r * kWarps;
    if (t < n_tok) {
      const int slot = (p_first + t) & page_mask;
      pool[((((size_t)page * n_heads + h) << page_log2) + slot) * 32 + lane] = quant4(rows[r], sc);
    }
  }
}

__global__ void __launch_bounds__(kQuantThreads)
q_quant_kernel(const uint2 *__restrict__ q, uint32_t *__restrict__ q8, float *__restrict__ sq, int total_q, int n_heads) {
  pdl_wait();
  pdl_launch_dependents();
  const long long rh = (long long)blockIdx.x * (kQuantThreads / 32) + (threadIdx.x >> 5); // (row, head) index, row-major
  const int lane = threadIdx.x & 31;
  if (rh >= (long long)total_q * n_heads) return;
  const uint2 v = __ldg(q + rh * 32 + lane);
  const float am = warp_max(amax4(v));
  const float sc = am > 0.f ? __fdiv_rn(am, kE4m3Max) : 1.0f;
  q8[rh * 32 + lane] = quant4(v, sc);
  if (lane == 0) {
    const int row = (int)(rh / n_heads), h = (int)(rh % n_heads);
    sq[(size_t)h * total_q + row] = sc;
  }
}

} // namespace

cudaError_t launch_kv_append_fp8(const void *k_new, const void *v_new, void *k_pool, void *v_pool, float *k_scale, float *v_scale,
                                 const DevStream *d_streams, int n_streams, int max_q_len, const int32_t *d_page_tables,
                                 int n_heads, int page_size, cudaStream_t st, int *n_launched) {
  if (n_streams == 0 || max_q_len == 0) return cudaSuccess;
  int pl2 = 0;
  while ((1 << pl2) < page_size) ++pl2;
  const int max_blocks = (max_q_len + 127) / 128 + 1; // a chunk of L tokens touches at most ceil(L / 128) + 1 blocks
  constexpr int kMaxZ = 65534;
  cudaError_t e = cudaSuccess;
  for (int s0 = 0; s0 < n_streams && e == cudaSuccess; s0 += kMaxZ / 2) {
    const int ns = n_streams - s0 < kMaxZ / 2 ? n_streams - s0 : kMaxZ / 2;
    e = launch_pdl(kv_append_fp8_kernel, dim3(max_blocks, n_heads, 2 * ns), dim3(kQuantThreads), 0, st,
                   reinterpret_cast<const uint2 *>(k_new), reinterpret_cast<const uint2 *>(v_new), reinterpret_cast<uint32_t *>(k_pool),
                   reinterpret_cast<uint32_t *>(v_pool), k_scale, v_scale, d_streams + s0, d_page_tables, n_heads, pl2);
    if (n_launched) *n_launched += 1;
  }
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_q_quant(const void *q, void *q8, float *sq, int total_q, int n_heads, cudaStream_t st, int *n_launched) {
  if (total_q == 0) return cudaSuccess;
  const long long rows = (long long)total_q * n_heads;
  const int wpb = kQuantThreads / 32;
  cudaError_t e = launch_pdl(q_quant_kernel, dim3((unsigned)((rows + wpb - 1) / wpb)), dim3(kQuantThreads), 0, st,
                             reinterpret_cast<const uint2 *>(q), reinterpret_cast<uint32_t *>(q8), sq, total_q, n_heads);
  if (n_launched) *n_launched += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace slack
