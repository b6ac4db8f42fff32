// kernels.h — launch functions of the CUDA kernels (defined in append.cu, attn_simt.cu, attn_tc.cu, combine.cu).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "slack_internal.h"

namespace slack {

// Programmatic dependent launch (PDL): kernels of the per-layer hot loop (append -> attention -> combine, layer after
// layer on one stream) are launched with cudaLaunchAttributeProgrammaticStreamSerialization so that a kernel's launch
// overlaps the drain of its predecessor (~5-7 us per boundary, 3 boundaries per layer).  Every such kernel calls
// pdl_wait() before it touches memory a predecessor may still be writing (it returns once all prerequisite grids have
// completed and flushed), and pdl_launch_dependents() right after so that its own successor can be staged early.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
#ifdef SLACK_NO_PDL
  cfg.numAttrs = 0; // A/B switch: plain stream-ordered launches
#else
  cfg.numAttrs = 1;
#endif
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

// A1: paged scatter copy. elem_bytes = 2 (bf16) or 4 (f32). Launches 1 kernel (0 if nothing to copy).
cudaError_t launch_kv_append(const void *k_new, const void *v_new, void *k_pool, void *v_pool, const DevStream *d_streams,
                             int n_streams, int max_q_len, const int32_t *d_page_tables, int n_heads, int head_dim,
                             int page_size, int elem_bytes, int sm_count, cudaStream_t st, int *n_launched);

// A3 (validation / fp32 path): one warp per (query row, head), fp32 accumulation, any page size.
cudaError_t launch_attn_simt(int dtype, const void *q, const void *k_pool, const void *v_pool, void *out, float *lse,
                             const DevStream *d_streams, int n_streams, int total_q, const int32_t *d_page_tables,
                             int n_heads, int head_dim, int page_size, float scale, const uint32_t *mask, int mask_words,
                             cudaStream_t st, int *n_launched);

// A3 (tensor-core path: bf16 with head_dim 64 or 128, FP8 with head_dim 128; page_size >= 128).
struct TcParams {
  const DevItem *items;
  const int32_t *cta_begin;
  const int32_t *page_tables;
  void *out;            // bf16 [total_q][H][head_dim]
  float *lse;           // [H][total_q] or null
  float *ws_o;          // partial outputs [slot][256][head_dim] fp32
  float *ws_lse;        // partial lse [slot][256]
  float *dbg_s;         // SLACK_DIAGNOSTICS builds: dump of the first S tiles of CTA 0 ([2][128][128] fp32), else null
  uint32_t *dbg_t;      // SLACK_DIAGNOSTICS builds: time-stamp trace (selects the kTrace instantiation), else null
  unsigned long long *dbg_flag; // 4-word host-mapped record a timed-out barrier wait fills before it traps
  const uint16_t *steps;        // block-sparse: compacted step lists (sparse_steps.cu), else null = dense
  const int32_t *item_steps;    // block-sparse: selected steps per item
  const float *k_scale;         // FP8 pools: [n_pages][H][P / 128] scales of the K / V codes, else null
  const float *v_scale;
  const float *q_scale;         // FP8 pools: [H][total_q] scales of the quantised Q (q_quant_kernel)
  int32_t n_heads;
  int32_t head_dim;     // 128, or 64 (bf16 only: the kD = 64 instantiations)
  int32_t page_log2;
  int32_t total_q;
  int32_t has_dual;     // the plan holds dual items (DevItem::dual): launch the instantiation that serves them
  float scale;          // logits = scale * q.k
};
size_t attn_tc_smem_bytes();
cudaError_t attn_tc_configure(); // cudaFuncSetAttribute(max dynamic smem); once per process/device
cudaError_t launch_attn_tc(const TcParams &p, const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                           int n_cta, cudaStream_t st, int *n_launched);

// NEXT-3 (quant.cu): quantising append into an FP8 pool, and the Q quantiser of the FP8 attention call.
// tm_k_new / tm_v_new: unswizzled bf16 maps over K_new / V_new [sum Lq][H * 128] with 128 x 128 boxes (api.cu make_rows_map)
cudaError_t launch_kv_append_fp8(const CUtensorMap &tm_k_new, const CUtensorMap &tm_v_new, void *k_pool, void *v_pool, float *k_scale, float *v_scale,
                                 const DevStream *d_streams, int n_streams, int max_q_len, const int32_t *d_page_tables,
                                 int n_heads, int page_size, unsigned long long *dbg /* record of a timed-out wait, may be null */,
                                 cudaStream_t st, int *n_launched);
cudaError_t launch_q_quant(const void *q, void *q8, float *sq, int total_q, int n_heads, cudaStream_t st, int *n_launched);

// A3 on CTA pairs (attn_tc2.cu, tcgen05 cta_group::2): needs a pair plan (HostPlan::kernel_kind 2, even n_cta) and a K
// tensor map with 64-row boxes (each CTA loads half of a key tile's keys).
cudaError_t attn_tc2_configure();
cudaError_t launch_attn_tc2(const TcParams &p, const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                            int n_cta, cudaStream_t st, int *n_launched);

// Block-sparse A3: per item, the selected key-tile steps under a device block mask (see sparse_steps.cu).
cudaError_t launch_sparse_steps(const DevItem *d_items, int n_items, const uint32_t *mask, int n_heads, int mask_words,
                                uint16_t *steps, int32_t *count, cudaStream_t st, int *n_launched);

// NEXT-4: one layer of the state-plane page transfer (see transfer.cu).
cudaError_t launch_kv_transfer(const void *src_k, const void *src_v, void *dst_k, void *dst_v, const int32_t *d_src_ids,
                               const int32_t *d_dst_ids, int n_pages, int n_heads, int head_dim, int page_size,
                               int elem_bytes, int head_begin, int head_end, int sm_count, cudaStream_t st,
                               int *n_launched);

// NEXT-4 for FP8 pools: the scales of the moved (page, head) slices.
cudaError_t launch_kv_scale_transfer(const float *src_k, const float *src_v, float *dst_k, float *dst_v, const int32_t *d_src_ids,
                                     const int32_t *d_dst_ids, int n_pages, int n_heads, int page_size, int head_begin,
                                     int head_end, cudaStream_t st, int *n_launched);

// A4: merge split-KV partials into `out` (bf16) and `lse`.
cudaError_t launch_combine(const DevCombine *d_combines, int n_combines, const float *ws_o, const float *ws_lse, void *out,
                           float *lse, int n_heads, int head_dim, int total_q, cudaStream_t st, int *n_launched);

} // namespace slack
