/* slack_diag.h — diagnostics of the attention kernel; exported only by a library built with -DSLACK_DIAGNOSTICS
 * (SLACK_DIAGNOSTICS=1 python -m paper_2606_15319_b200.build --force).  Never on the data path of the default build:
 * the default libslack.so exports none of this and does not contain the traced kernel instantiation.
 *
 * slack_debug_set(ctx, key, value):
 *   key 0: `value` = DEVICE pointer to a [2][128][128] fp32 buffer that receives the first two S = QK^T tiles computed by
 *          CTA 0 of the next dense tensor-core launches (NULL switches the dump off).
 *   key 1: `value` = DEVICE pointer to a uint32 buffer of 2048 + 4 * (number of SMs) words; while set, dense tensor-core
 *          launches store clock64() time stamps of CTA 0's first item (rows 0/1 = softmax of query tile 0/1, row 2 = MMA
 *          issuer, row 3 = per-warp arrivals; [row][kv step < 64][8 slots], slots documented in csrc/attn_tc.cu) and, from
 *          word 2048 on, {clock start, clock end, globaltimer start, end} of every CTA.  NULL switches it off.
 */
#ifndef SLACK_DIAG_H_
#define SLACK_DIAG_H_
#include "slack.h"
#ifdef __cplusplus
extern "C" {
#endif
slack_status slack_debug_set(slack_ctx *ctx, int32_t key, void *value);
#ifdef __cplusplus
}
#endif
#endif /* SLACK_DIAG_H_ */
