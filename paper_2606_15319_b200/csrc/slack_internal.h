// slack_internal.h — structures shared by the host planner (plan.cpp), the entry points (api.cu) and the kernels.
// Nothing here is part of the ABI (include/slack.h is).
#pragma once
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/slack.h"

namespace slack {

// Geometry of the tensor-core path (fixed at compile time).
constexpr int kTileM = 128;    // query rows per MMA tile (UMMA M)
constexpr int kTileN = 128;    // keys per KV tile (UMMA N of QK^T, K extent of PV); anchored to page slots
constexpr int kItemRows = 256; // an item carries two query tiles that ping-pong on the tensor pipe

// One planned unit of work as the kernels read it (device copy of slack_work_item plus table offsets). 80 bytes.
// Key tiles are visited in the order: sink tiles [sink_tile0, sink_tile0 + sink_tiles) with visible positions
// [sink_lo, sink_hi) ("sink + local"; only the first piece of a row carries them), then the window tiles
// [kv_tile_begin, kv_tile_end) with visible positions [pos_lo, pos_hi).
struct DevItem {
  int32_t q_row0;        // global row (ragged concat) of the item's first query row
  int32_t q_rows;        // valid rows, 1..256
  int32_t head;
  int32_t pt_off;        // offset of the stream's page table inside the concatenated device table
  int32_t kv_tile_begin; // position-tile range [begin, end), tile T = positions [128T, 128T+128)
  int32_t kv_tile_end;
  int32_t pos_lo;        // visible positions [pos_lo, pos_hi)
  int32_t pos_hi;
  int32_t partial_slot;  // -1 = final output, else workspace slot
  int32_t stream;
  int32_t sink_lo;       // = base
  int32_t sink_hi;       // = base + sink (== sink_lo when the item has no sink tiles)
  int32_t sink_tile0;
  int32_t sink_tiles;
  int32_t mask_row;      // block-sparse: global 256-row query block of the item = row of the block mask (P:88 knob (2))
  int32_t step_off;      // block-sparse: offset of the item's compacted step list (uint16 units) in the sparse workspace
  int32_t dual;          // 1: this item (<= 128 rows) and the NEXT one of the queue (<= 128 rows, same number of key steps,
                         // any stream / head) share a CTA: this one takes query-tile slot 0, the next one slot 1, each with
                         // its own K/V tiles (decode-like chunks; the 72-row tails of long chunks).  Kernels that do not
                         // implement it (block-sparse, FP8, SIMT) just walk the two items one after the other
  int32_t pad[3];
};
static_assert(sizeof(DevItem) == 80, "DevItem layout");

// One output row-block whose key range was cut: the combine kernel merges its partial slots (A4).
struct DevCombine {
  int32_t q_row0;     // global first row
  int32_t q_rows;     // valid rows (<= 256)
  int32_t head;
  int32_t slot_begin; // partial slots [slot_begin, slot_begin + n_parts)
  int32_t n_parts;
  int32_t pad[3];
};
static_assert(sizeof(DevCombine) == 32, "DevCombine layout");

// Per-stream record used by the append kernel and the SIMT kernel.
struct DevStream {
  int32_t q_row0;   // first row of the stream in the ragged concat
  int32_t q_len;
  int32_t cache_len;
  int32_t base;
  int32_t pos_lo;   // base + lo
  int32_t pos_hi;   // base + n
  int32_t pt_off;
  int32_t n_table_pages;
  int32_t sink_hi;  // visible sink positions [base, sink_hi) in front of [pos_lo, pos_hi); == base when there are none
  int32_t qblock0;  // global index of the stream's first 256-row query block (row of the block mask)
  int32_t app_pos0; // position of the first token the append writes: pos(cache_len) (slack.h token -> slot rule)
  int32_t old_hi0;  // positions of the stream's EARLIER tokens [0, cache_len): [base, old_hi0) and [old_lo1, app_pos0)
  int32_t old_lo1;  //   (the second range is empty unless a hole sits behind the sink; FP8 append: who owns a scale block)
  int32_t pad[3];
};
static_assert(sizeof(DevStream) == 64, "DevStream layout");

// Workspace layout for split-KV partials: slot s holds kItemRows rows of head_dim fp32 (normalised partial output)
// followed, in a second region, by kItemRows fp32 lse values.
struct WorkspaceLayout {
  size_t o_bytes = 0;   // n_slots * 256 * D * 4
  size_t lse_off = 0;   // = o_bytes
  size_t total = 0;
};

struct HostPlan {
  // shape the plan was made for
  int32_t n_pages = 0, n_heads = 0, head_dim = 0, page_size = 0, dtype = 0;
  int32_t n_streams = 0, total_q = 0;
  int32_t n_cta = 0;
  int32_t n_queues = 0;    // item queues: n_cta, or n_cta / 2 for pair plans
  int32_t kernel_kind = 0; // 0 tensor-core (one CTA per queue), 1 SIMT, 2 tensor-core CTA pairs (n_cta / 2 queues, cta_group::2)
  std::vector<DevStream> streams;
  std::vector<int32_t> page_tables;  // concatenated
  std::vector<DevItem> items;        // in queue order: CTA c owns items [cta_begin[c], cta_begin[c+1])
  std::vector<int32_t> cta_begin;    // queues + 1 (queues = n_cta, or n_cta / 2 for pair plans)
  std::vector<int32_t> item_cta;     // per item
  std::vector<DevCombine> combines;
  int32_t n_partial_slots = 0;
  bool has_dual = false;   // some item carries DevItem::dual
  WorkspaceLayout ws;
  // FP8 pools: the attention call quantises Q into the workspace first: codes [total_q][H][128] u8, scales [H][total_q] f32
  size_t q8_off = 0, q8_scale_off = 0;
  // block-sparse variant (slack_chunk_attention_sparse): mask geometry and the extra workspace behind ws.total
  int32_t mask_rows = 0;        // sum over streams of ceil(q_len / 256)
  int32_t mask_words_min = 1;   // 32-bit words a mask row needs: ceil(max_s ceil(pos_hi / 128) / 32)
  int64_t total_steps = 0;      // sum over items of their dense key-tile steps (entries of the step lists)
  int32_t max_item_steps = 0;   // longest item (the step lists hold 16-bit step indices)
  size_t sparse_steps_off = 0;  // byte offset of uint16 steps[total_steps] (16-byte aligned, >= ws.total)
  size_t sparse_count_off = 0;  // byte offset of int32 item_steps[n_items]
  size_t sparse_total = 0;      // workspace bytes slack_chunk_attention_sparse needs
  double makespan = 0, ideal = 0;    // in cost units (for tests / tuning)
};

// Validates and plans. Returns SLACK_OK or an error with `err` filled in.
slack_status build_plan(const slack_pool &shape, int32_t n_streams, const slack_stream *streams,
                        const slack_plan_opts &opts, int32_t default_sm_count, HostPlan &out, std::string &err);

} // namespace slack
