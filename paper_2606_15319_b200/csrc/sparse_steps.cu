// sparse_steps.cu — block-sparse variant of A3 (PAPER.md P:88 knob (2): "skips nonselected attention
// blocks with sparse masks", sparsity rho in {0,.6,.7,.8,.9} P:568).  The block mask is a DEVICE input that may change
// with every layer and denoising step, so the host plan stays mask-independent (dense geometry) and this kernel turns
// the mask into what the attention kernel's roles walk: per planned item, the list of its SELECTED key-tile steps.
//
//   mask   uint32 [mask_rows][n_heads][mask_words]: bit (t % 32) of word t / 32 = key block t (positions
//          [128 t, 128 t + 128) of the stream's page-table space) is selected for that (256-row query block, head)
//   steps  uint16 [total dense steps]: item k's selected dense step indices j, ascending, at steps[items[k].step_off ..]
//   count  int32  [n_items]: how many (0 is legal: the item's rows have no key in this piece)
//
// One warp per item; 32 dense steps per iteration, compacted with a ballot.  Integer work, a few microseconds.
#include "kernels.h"

namespace slack {
namespace {

constexpr int kStepsThreads = 128;

__global__ void __launch_bounds__(kStepsThreads)
sparse_steps_kernel(const DevItem *__restrict__ items, int n_items, const uint32_t *__restrict__ mask, int n_heads,
                    int mask_words, uint16_t *__restrict__ steps, int32_t *__restrict__ count) {
  pdl_wait(); // the mask may be produced by the kernel before; the step lists may still be read by the previous attention
  pdl_launch_dependents();
  const int k = blockIdx.x * (kStepsThreads / 32) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (k >= n_items) return;
  const DevItem it = items[k];
  const uint32_t *row = mask + ((size_t)it.mask_row * n_heads + it.head) * mask_words;
  const int T = it.sink_tiles + (it.kv_tile_end - it.kv_tile_begin);
  uint16_t *dst = steps + it.step_off;
  int n = 0;
  for (int j0 = 0; j0 < T; j0 += 32) {
    const int j = j0 + lane;
    bool sel = false;
    if (j < T) {
      const int tile = j < it.sink_tiles ? it.sink_tile0 + j : it.kv_tile_begin + (j - it.sink_tiles);
      sel = (__ldg(row + (tile >> 5)) >> (tile & 31)) & 1u;
    }
    const uint32_t b = __ballot_sync(0xffffffffu, sel);
    if (sel) dst[n + __popc(b & ((1u << lane) - 1u))] = (uint16_t)j;
    n += __popc(b);
  }
  if (lane == 0) count[k] = n;
}

} // namespace

cudaError_t launch_sparse_steps(const DevItem *d_items, int n_items, const uint32_t *mask, int n_heads, int mask_words,
                                uint16_t *steps, int32_t *count, cudaStream_t st, int *n_launched) {
  if (n_items == 0) return cudaSuccess;
  const int wpb = kStepsThreads / 32;
  cudaError_t e = launch_pdl(sparse_steps_kernel, dim3((unsigned)((n_items + wpb - 1) / wpb)), dim3(kStepsThreads), 0, st, d_items,
                             n_items, mask, n_heads, mask_words, steps, count);
  if (n_launched) *n_launched += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace slack
