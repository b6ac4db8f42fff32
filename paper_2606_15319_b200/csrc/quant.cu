// quant.cu — NEXT-3 (PAPER.md P:88 knob (4) "quantization mode Q", "online FP8 attention
// quantization"): the two quantisers of the FP8 path.  The rule is include/slack.h's (slack_dtype) and DESIGN.md A19:
// OCP e4m3, round to nearest even, saturating; code = e4m3(fp32(x) / scale) with scale = amax / 448 (amax = 0 -> 1), both
// divisions IEEE fp32 (__fdiv_rn), so that codes and scales are bit-exact against the oracle.
//
//   kv_append_fp8_kernel  A1 for FP8 pools: one CTA per (key block of 128 slots, head, stream x {K, V}); a block whose
//                         first held token this append writes gets its scale from the tokens written, any other
//                         block keeps the stored scale.  The block's rows (<= 128 x 256 B) are staged in shared memory by
//                         one TMA box load (cp.async.bulk.tensor) and read from there for the amax and for the conversion:
//                         HBM-bound, 2 * Lq * H * D * 2 B read once, half of that written.
//                         The per-element division shares one reciprocal per thread (Divider: same bits as __fdiv_rn).
//   q_quant_kernel        Q of an attention call -> codes [sum Lq][H][128] + scales [H][sum Lq] in the workspace;
//                         one warp per (row, head).
#include <cuda_bf16.h>

#include "kernels.h"
#include "ptx_sm100.cuh"

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

// x / scale, correctly rounded (== __fdiv_rn(x, scale), the oracle's IEEE division) with ONE reciprocal per thread instead of
// one per element, on packed pairs and on the FMA pipe only: r = RN(1 / scale), q0 = RN(x r), rem = x - q0 scale (exact in
// the FMA), q = RN(q0 + rem r) is the correctly rounded quotient whenever q0 is within an ulp of it (Markstein's theorem).
// rem is formed rounding toward -inf: it is exact, so only the sign of an exact zero changes (-0), which is what makes the
// quotient of x = -0 come out as -0 (x = +0: +0) without a copysign.  Where the theorem's argument or the exactness of rem
// fails, q0's own accuracy already decides the code: tiny quotients round to the zero code of x's sign either way, and a
// q0 that overflowed (Inf; x r can exceed fp32 only against a STORED scale, kGuard) or is NaN makes q NaN -> q0 is taken
// (Inf saturates to 448).  A scale outside [2^-60, 2^60] (a block of denormals / of huge values) takes the plain division.
template <bool kFast, bool kGuard>
struct Divider {
  float scale, r;
  __device__ __forceinline__ explicit Divider(float sc) {
    scale = sc;
    r = kFast ? __frcp_rn(sc) : 0.f;
  }
  __device__ __forceinline__ void operator()(float x0, float x1, float &o0, float &o1) const {
    if constexpr (!kFast) {
      o0 = __fdiv_rn(x0, scale), o1 = __fdiv_rn(x1, scale);
    } else {
      const uint64_t x2 = ptx::pack2(x0, x1), r2 = ptx::pack2(r, r);
      const uint64_t q0 = ptx::fmul2(x2, r2);
      const uint64_t q1 = ptx::ffma2(ptx::ffma2_rm(q0, ptx::pack2(-scale, -scale), x2), r2, q0);
      ptx::unpack2(q1, o0, o1);
      if constexpr (kGuard) {
        float b0, b1;
        ptx::unpack2(q0, b0, b1);
        o0 = (o0 == o0) ? o0 : b0;
        o1 = (o1 == o1) ? o1 : b1;
      }
    }
  }
};
__device__ __forceinline__ bool divider_fast(float sc) { return sc >= 0x1p-60f && sc <= 0x1p60f; }

// one lane's 8 consecutive head_dim elements (16 bytes of bf16): their largest magnitude, and their 8 codes
__device__ __forceinline__ float amax2(uint32_t u) { return fmaxf(fabsf(bf16_lo(u)), fabsf(bf16_hi(u))); }
// running |.| maximum of packed bf16 pairs, one LOP3 + one HMNMX2 per two elements (a NaN operand is ignored, as by fmaxf)
__device__ __forceinline__ uint32_t amax_acc(uint32_t acc, uint32_t u) {
  uint32_t d;
  asm("max.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(acc), "r"(u & 0x7fff7fffu));
  return d;
}
__device__ __forceinline__ uint32_t amax_acc(uint32_t acc, uint4 v) { return amax_acc(amax_acc(amax_acc(amax_acc(acc, v.x), v.y), v.z), v.w); }
template <class Div>
__device__ __forceinline__ uint32_t quant4(uint32_t a, uint32_t b, const Div &dv) {
  float q0, q1, q2, q3;
  dv(bf16_lo(a), bf16_hi(a), q0, q1);
  dv(bf16_lo(b), bf16_hi(b), q2, q3);
  return e4m3x2(q0, q1) | (e4m3x2(q2, q3) << 16);
}
template <class Div>
__device__ __forceinline__ uint2 quant8(uint4 v, const Div &dv) { return make_uint2(quant4(v.x, v.y, dv), quant4(v.z, v.w, dv)); }
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

__global__ void __launch_bounds__(kQuantThreads, 6)
kv_append_fp8_kernel(const __grid_constant__ CUtensorMap tm_k_new, const __grid_constant__ CUtensorMap tm_v_new, uint2 *__restrict__ k_pool,
                     uint2 *__restrict__ v_pool, float *__restrict__ k_scale, float *__restrict__ v_scale,
                     const DevStream *__restrict__ streams, const int32_t *__restrict__ page_tables, int n_heads, int page_log2,
                     unsigned long long *dbg) {
  // the block's token rows (<= 128 x 256 B), staged by ONE TMA box load: no registers are tied up while they are in
  // flight, so six CTAs per SM keep ~190 KB of loads outstanding
  __shared__ alignas(128) uint4 tile[128 * 16];
  __shared__ alignas(8) unsigned long long mbar;
  __shared__ float red[kQuantThreads / 32];
  const uint32_t bar = ptx::smem_u32(&mbar);
  if (threadIdx.x == 0) {
    ptx::mbar_init(bar, 1);
    ptx::fence_barrier_init();
  }
  __syncthreads();
  pdl_wait();
  pdl_launch_dependents();
  const DevStream s = streams[blockIdx.z >> 1];
  if (s.q_len == 0) return;
  const bool is_v = blockIdx.z & 1;
  const int h = blockIdx.y;
  const int kb = (s.app_pos0 >> 7) + blockIdx.x; // key block in the stream's position space
  const int p_first = max(kb << 7, s.app_pos0), p_last = min((kb << 7) + 128, s.app_pos0 + s.q_len); // positions written here
  if (p_first >= p_last) return;
  uint2 *pool = is_v ? v_pool : k_pool;
  float *scales = is_v ? v_scale : k_scale;
  const int n_tok = p_last - p_first;
  const int tok0 = p_first - s.app_pos0; // chunk-local index of the first token written here
  // A token row of one head is 128 bf16 = 256 contiguous bytes of the source, H rows apart from the next token's: a box of
  // 128 rows x 128 elements at (column h * 128, row = first token).  Rows past the tokens this CTA writes (the next
  // stream's, or zero fill past the end of the array) land in the tile and are not used.
  if (threadIdx.x == 0) {
    ptx::mbar_expect_tx(bar, 128u * 256u);
    ptx::tma_load_2d(ptx::smem_u32(tile), is_v ? &tm_v_new : &tm_k_new, bar, h * 128, s.q_row0 + tok0);
  }
  const int page = page_tables[s.pt_off + ((kb << 7) >> page_log2)];
  const int blocks_per_page = 1 << (page_log2 - 7);
  float *scale_ptr = scales + ((size_t)page * n_heads + h) * blocks_per_page + (((kb << 7) & ((1 << page_log2) - 1)) >> 7);
  // none of the stream's earlier tokens lies in this block -> this append starts it and sets its scale
  const int b_lo = kb << 7, b_hi = b_lo + 128;
  const bool has_old = (s.base < b_hi && s.old_hi0 > b_lo && s.old_hi0 > s.base) || (s.old_lo1 < b_hi && s.app_pos0 > b_lo && s.app_pos0 > s.old_lo1);
  float sc = has_old ? __ldg(scale_ptr) : 0.f; // written by the append that started the block (an earlier launch)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // 16 lanes x 16 bytes per row: a warp instruction handles two consecutive tokens, a warp owns 16 consecutive tokens
  // (2 KB of contiguous destination: consecutive slots of one (page, head) are adjacent rows of the pool)
  constexpr int kWarps = kQuantThreads / 32, kRowsPerWarp = 128 / kWarps, kIters = kRowsPerWarp / 2;
  const int sub = lane >> 4, l16 = lane & 15;
  auto tok_of = [&](int r) { return warp * kRowsPerWarp + 2 * r + sub; };
  ptx::mbar_wait(bar, 0u, 900, dbg);
  if (!has_old) { // one CTA barrier: every thread folds the 8 warp maxima itself
    uint32_t acc = 0u;
#pragma unroll
    for (int r = 0; r < kIters; ++r) {
      const int t = tok_of(r);
      if (t < n_tok) acc = amax_acc(acc, tile[t * 16 + l16]);
    }
    const float am = warp_max(amax2(acc));
    if (lane == 0) red[warp] = am;
    __syncthreads();
    float a = red[0];
#pragma unroll
    for (int w = 1; w < kWarps; ++w) a = fmaxf(a, red[w]);
    sc = a > 0.f ? __fdiv_rn(a, kE4m3Max) : 1.0f;
    if (threadIdx.x == 0) *scale_ptr = sc;
  }
  // destination row of position p, head h: 128 codes = 16 lanes x 8 bytes; consecutive slots are adjacent rows
  uint2 *dst = pool + ((((size_t)page * n_heads + h) << page_log2) + (size_t)(p_first & ((1 << page_log2) - 1))) * 16 + l16;
  auto convert = [&](auto dv) {
#pragma unroll
    for (int r = 0; r < kIters; ++r) {
      const int t = tok_of(r);
      if (t < n_tok) dst[(size_t)t * 16] = quant8(tile[t * 16 + l16], dv);
    }
  };
  // quotients against a scale this append has just set are bounded by 448: no overflow guard (kGuard) needed
  if (!divider_fast(sc)) convert(Divider<false, false>(sc));
  else if (has_old) convert(Divider<true, true>(sc));
  else convert(Divider<true, false>(sc));
}

__global__ void __launch_bounds__(kQuantThreads)
q_quant_kernel(const uint2 *__restrict__ q, uint32_t *__restrict__ q8, float *__restrict__ sq, int total_q, int n_heads) {
  pdl_wait();
  pdl_launch_dependents();
  const long long rh = (long long)blockIdx.x * (kQuantThreads / 32) + (threadIdx.x >> 5); // (row, head) index, row-major
  const int lane = threadIdx.x & 31;
  if (rh >= (long long)total_q * n_heads) return;
  const uint2 v = __ldg(q + rh * 32 + lane);
  const float am = warp_max(fmaxf(amax2(v.x), amax2(v.y)));
  const float sc = am > 0.f ? __fdiv_rn(am, kE4m3Max) : 1.0f;
  q8[rh * 32 + lane] = divider_fast(sc) ? quant4(v.x, v.y, Divider<true, false>(sc)) : quant4(v.x, v.y, Divider<false, false>(sc));
  if (lane == 0) {
    const int row = (int)(rh / n_heads), h = (int)(rh % n_heads);
    sq[(size_t)h * total_q + row] = sc;
  }
}

} // namespace

cudaError_t launch_kv_append_fp8(const CUtensorMap &tm_k_new, const CUtensorMap &tm_v_new, void *k_pool, void *v_pool, float *k_scale, float *v_scale,
                                 const DevStream *d_streams, int n_streams, int max_q_len, const int32_t *d_page_tables,
                                 int n_heads, int page_size, unsigned long long *dbg, cudaStream_t st, int *n_launched) {
  if (n_streams == 0 || max_q_len == 0) return cudaSuccess;
  int pl2 = 0;
  while ((1 << pl2) < page_size) ++pl2;
  const int max_blocks = (max_q_len + 127) / 128 + 1; // a chunk of L tokens touches at most ceil(L / 128) + 1 blocks
  constexpr int kMaxZ = 65534;
  cudaError_t e = cudaSuccess;
  for (int s0 = 0; s0 < n_streams && e == cudaSuccess; s0 += kMaxZ / 2) {
    const int ns = n_streams - s0 < kMaxZ / 2 ? n_streams - s0 : kMaxZ / 2;
    e = launch_pdl(kv_append_fp8_kernel, dim3(max_blocks, n_heads, 2 * ns), dim3(kQuantThreads), 0, st,
                   tm_k_new, tm_v_new, reinterpret_cast<uint2 *>(k_pool),
                   reinterpret_cast<uint2 *>(v_pool), k_scale, v_scale, d_streams + s0, d_page_tables, n_heads, pl2, dbg);
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
