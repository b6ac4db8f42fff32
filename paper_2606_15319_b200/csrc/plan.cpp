// plan.cpp — A2: host-side ragged batch planner (integer work only; no CUDA).
//
// Not in the paper: the paper's Execution Plane dispatches one stream at a time per worker (§3.2,
// P:638 App. C.1); co-batching streams of different cache lengths in one launch is BASELINE.json north_star's
// extension.  The planner turns the batch into work items (stream, head, 256-row query block, range of 128-key
// tiles), decides where key ranges are cut (split-KV), and list-schedules the items onto one queue per SM.
//
// Item order = locality order: streams by descending key-tile count, then head, then query block (then key chunk
// when split-KV is forced).  Co-running CTAs sweep the same K/V tiles at the same time, so each tile is fetched from
// HBM once and then hit in L2.  See make_balanced() for the default plan.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <functional>
#include <numeric>
#include <queue>

#include "slack_internal.h"

namespace slack {
namespace {

struct StreamGeom {
  int32_t idx;
  int32_t tile0, tiles;   // position-tile range of the window part [pos_lo, pos_hi)
  int32_t q_blocks;       // ceil(q_len / 256)
  int32_t sink_tile0, sink_tiles; // tiles holding the visible sink positions [base, sink_hi) (0 tiles: no sink)
};

// the sink part of a row rides with the row's first piece
void set_sink(DevItem &it, const StreamGeom &g, const DevStream &s, bool first_piece) {
  it.sink_lo = s.base;
  it.sink_hi = first_piece ? s.sink_hi : s.base;
  it.sink_tile0 = g.sink_tile0;
  it.sink_tiles = first_piece ? g.sink_tiles : 0;
}

constexpr double kTileCost = 2.0;      // one 128-key tile against a 256-row item (two MMA tile pairs)
constexpr double kItemOverhead = 7.75; // pipeline fill/drain + epilogue: 12.6k cycles = 3.9 steps of 3250 (least-squares fit of per-CTA
                                       // spans on BASELINE configs 2, 4, 5: cycles = 3250 x two-tile steps + 2755 x one-tile steps + 12.6k x items)
constexpr double kTileCost1 = 1.70; // one 128-key tile against a single query tile: 2755 vs 3250 cycles (same fit; the chain bounds it)
constexpr double kPartialCost = 3.0;   // extra epilogue traffic + combine work per partial slot

struct Candidate {
  std::vector<DevItem> items;
  std::vector<int32_t> item_cta;
  std::vector<DevCombine> combines;
  int32_t n_slots = 0;
  double makespan = 0, ideal = 0, objective = 0;
};

int32_t ceil_div(int64_t a, int64_t b) { return (int32_t)((a + b - 1) / b); }

// parts[s] = number of key chunks for stream s
void make_candidate(const std::vector<StreamGeom> &order, const std::vector<int32_t> &parts,
                    const std::vector<DevStream> &ds, int32_t n_heads, int32_t n_cta, bool pairs, Candidate &c) {
  c = Candidate();
  for (size_t oi = 0; oi < order.size(); ++oi) {
    const StreamGeom &g = order[oi];
    const DevStream &s = ds[g.idx];
    const int32_t np = parts[oi];
    for (int32_t h = 0; h < n_heads; ++h) {
      int32_t slot0 = -1;
      if (np > 1) {
        slot0 = c.n_slots;
        c.n_slots += np * g.q_blocks;
        for (int32_t qb = 0; qb < g.q_blocks; ++qb) {
          DevCombine cb{};
          cb.q_row0 = s.q_row0 + qb * kItemRows;
          cb.q_rows = std::min(kItemRows, s.q_len - qb * kItemRows);
          cb.head = h;
          cb.slot_begin = slot0 + qb * np;
          cb.n_parts = np;
          c.combines.push_back(cb);
        }
      }
      for (int32_t p = 0; p < np; ++p) {
        const int32_t tb = g.tile0 + (int32_t)(((int64_t)p * g.tiles) / np);
        const int32_t te = g.tile0 + (int32_t)(((int64_t)(p + 1) * g.tiles) / np);
        for (int32_t qb = 0; qb < g.q_blocks; ++qb) {
          DevItem it{};
          it.q_row0 = s.q_row0 + qb * kItemRows;
          it.q_rows = std::min(kItemRows, s.q_len - qb * kItemRows);
          it.head = h;
          it.pt_off = s.pt_off;
          it.kv_tile_begin = tb;
          it.kv_tile_end = te;
          it.pos_lo = s.pos_lo;
          it.pos_hi = s.pos_hi;
          it.partial_slot = (np > 1) ? slot0 + qb * np + p : -1;
          it.stream = g.idx;
          set_sink(it, g, s, p == 0);
          c.items.push_back(it);
        }
      }
    }
  }
  // greedy list scheduling in item order: each item goes to the queue that frees up first
  using Slot = std::pair<double, int32_t>;
  std::priority_queue<Slot, std::vector<Slot>, std::greater<Slot>> heap;
  for (int32_t i = 0; i < n_cta; ++i) heap.push({0.0, i});
  c.item_cta.resize(c.items.size());
  double total = 0;
  for (size_t i = 0; i < c.items.size(); ++i) {
    const double tc = (pairs || c.items[i].q_rows > kTileM) ? kTileCost : kTileCost1;
    const double cost = tc * (c.items[i].kv_tile_end - c.items[i].kv_tile_begin + c.items[i].sink_tiles) + kItemOverhead;
    Slot s = heap.top();
    heap.pop();
    c.item_cta[i] = s.second;
    s.first += cost;
    total += cost;
    c.makespan = std::max(c.makespan, s.first);
    heap.push(s);
  }
  c.ideal = total / n_cta;
  c.objective = c.makespan + kPartialCost * c.n_slots / n_cta;
}

// Balanced candidate ("whole rows in lock step, then a cut tail").  A row is one (stream, head, 256-row query block)
// over the stream's whole key range.  Rows are taken in locality order and handed whole to the queue that frees up
// first, as long as that queue stays within the target (total cost / queues): with equal rows this is round-robin,
// so the queues of a wave sweep the same (stream, head) K/V tiles at the same time and each tile is read from HBM
// once.  Rows that no longer fit whole form the tail: their key ranges are laid end to end and dealt out in pieces
// that fill every queue up to the target (no piece shorter than kMinPiece tiles), so all queues end together and only
// tail rows produce split-KV partials.  (Cutting every queue's share out of one line - plain stream-K - balances as
// well but de-synchronises the sweeps: measured 17 % slower on BASELINE config 5, its K/V working set leaving L2.)
constexpr int32_t kMinPiece = 4;
constexpr bool kAutoPairs = false; // automatic plans use CTA pairs where they pay (see build_plan)

// A row of the balanced plan: one (stream, head, 256-row query block) over the stream's key range, or a DUAL row: two
// single-tile rows (<= 128 queries each) of the same stream that share a CTA, one per query-tile slot (DevItem::dual).
struct Row {
  int32_t oi, head, qb, q_rows, tile0, tiles, sink_tiles;
  int32_t head2 = -1, qb2 = 0, q_rows2 = 0; // companion of a dual row
  double tc;
};

void make_balanced(const std::vector<StreamGeom> &order, const std::vector<DevStream> &ds, int32_t n_heads, int32_t n_cta,
                   bool pairs, bool allow_dual, double target_scale, Candidate &c) {
  c = Candidate();
  std::vector<Row> rows;
  double total = 0;
  for (size_t oi = 0; oi < order.size(); ++oi) {
    const StreamGeom &g = order[oi];
    const DevStream &s = ds[g.idx];
    for (int32_t h = 0; h < n_heads; ++h)
      for (int32_t qb = 0; qb < g.q_blocks; ++qb) {
        Row r;
        r.oi = (int32_t)oi;
        r.head = h;
        r.qb = qb;
        r.q_rows = std::min(kItemRows, s.q_len - qb * kItemRows);
        r.tile0 = g.tile0;
        r.tiles = g.tiles;
        r.sink_tiles = g.sink_tiles;
        r.tc = (pairs || r.q_rows > kTileM) ? kTileCost : kTileCost1; // a CTA pair moves at one pace whatever the odd CTA holds
        rows.push_back(r);
      }
  }
  if (allow_dual) { // only where single-tile rows dominate (decode-like batches): the kernel instantiation that serves dual
                    // items runs ordinary two-tile steps ~5 % slower, so a few 72-row tails among long chunks do not pay
    size_t singles = 0;
    for (const Row &r : rows) singles += r.q_rows <= kTileM;
    allow_dual = 2 * singles >= rows.size();
  }
  if (allow_dual) { // single-tile rows of one stream (same key tiles, same step count) pair up, in row order
    std::vector<Row> merged;
    std::vector<int32_t> pending(order.size(), -1); // index in `merged` of a single still waiting for a companion
    for (const Row &r : rows) {
      if (r.q_rows > kTileM) {
        merged.push_back(r);
      } else if (pending[r.oi] >= 0) {
        Row &a = merged[(size_t)pending[r.oi]];
        a.head2 = r.head;
        a.qb2 = r.qb;
        a.q_rows2 = r.q_rows;
        a.tc = kTileCost; // two tiles in flight: the pace of a full item
        pending[r.oi] = -1;
      } else {
        pending[r.oi] = (int32_t)merged.size();
        merged.push_back(r);
      }
    }
    rows.swap(merged);
  }
  for (const Row &r : rows) total += r.tc * (r.tiles + r.sink_tiles) + kItemOverhead;
  const double target = target_scale * (total / n_cta) + kItemOverhead;
  std::vector<double> load((size_t)n_cta, 0.0);
  auto emit = [&](const Row &r, int32_t tb, int32_t take, int32_t cta) {
    const DevStream &s = ds[order[r.oi].idx];
    const bool first_piece = tb == r.tile0;
    for (int32_t m = 0; m < (r.head2 >= 0 ? 2 : 1); ++m) { // a dual row emits its two items back to back
      DevItem it{};
      it.q_row0 = s.q_row0 + (m == 0 ? r.qb : r.qb2) * kItemRows;
      it.q_rows = m == 0 ? r.q_rows : r.q_rows2;
      it.head = m == 0 ? r.head : r.head2;
      it.pt_off = s.pt_off;
      it.kv_tile_begin = tb;
      it.kv_tile_end = tb + take;
      it.pos_lo = s.pos_lo;
      it.pos_hi = s.pos_hi;
      it.partial_slot = -1;
      it.stream = order[r.oi].idx;
      it.dual = (m == 0 && r.head2 >= 0) ? 1 : 0;
      set_sink(it, order[r.oi], s, first_piece);
      c.items.push_back(it);
      c.item_cta.push_back(cta);
    }
    load[cta] += r.tc * (take + (first_piece ? r.sink_tiles : 0)) + kItemOverhead;
  };
  // ---- whole rows, earliest-free queue first --------------------------------------------------------------------
  using Slot = std::pair<double, int32_t>;
  std::priority_queue<Slot, std::vector<Slot>, std::greater<Slot>> heap;
  for (int32_t i = 0; i < n_cta; ++i) heap.push({0.0, i});
  std::vector<Row> tail;
  for (const Row &r : rows) {
    const Slot top = heap.top();
    if (top.first + r.tc * (r.tiles + r.sink_tiles) + kItemOverhead <= target + 1e-9) {
      heap.pop();
      emit(r, r.tile0, r.tiles, top.second);
      heap.push({load[top.second], top.second});
    } else {
      tail.push_back(r);
    }
  }
  // ---- the tail, cut to fill the queues -------------------------------------------------------------------------
  std::vector<int32_t> by_load((size_t)n_cta);
  std::iota(by_load.begin(), by_load.end(), 0);
  std::stable_sort(by_load.begin(), by_load.end(), [&](int32_t a, int32_t b) { return load[a] < load[b]; });
  size_t ti = 0;       // current tail row
  int32_t tb = 0, rem = 0;
  size_t first_piece = 0;
  auto open_row = [&]() {
    tb = tail[ti].tile0;
    rem = tail[ti].tiles;
    first_piece = c.items.size();
  };
  auto close_row = [&]() {
    const Row &r = tail[ti];
    const int32_t span = r.head2 >= 0 ? 2 : 1; // items per piece
    const int32_t np = (int32_t)(c.items.size() - first_piece) / span;
    if (np > 1) {
      for (int32_t m = 0; m < span; ++m) {
        const DevItem &i0 = c.items[first_piece + (size_t)m];
        DevCombine cb{};
        cb.q_row0 = i0.q_row0;
        cb.q_rows = i0.q_rows;
        cb.head = i0.head;
        cb.slot_begin = c.n_slots;
        cb.n_parts = np;
        c.combines.push_back(cb);
        for (int32_t q = 0; q < np; ++q) c.items[first_piece + (size_t)(q * span + m)].partial_slot = c.n_slots + q;
        c.n_slots += np;
      }
    }
    ++ti;
    if (ti < tail.size()) open_row();
  };
  if (!tail.empty()) open_row();
  for (int32_t qi = 0; qi < n_cta && ti < tail.size(); ++qi) {
    const int32_t cta = by_load[qi];
    while (ti < tail.size()) {
      const Row &r = tail[ti];
      const int32_t fit = (int32_t)std::floor((target - load[cta] - kItemOverhead) / r.tc + 1e-9) - (tb == r.tile0 ? r.sink_tiles : 0);
      if (fit >= rem) {
        emit(r, tb, rem, cta);
        close_row();
      } else if (fit >= kMinPiece && rem - fit >= kMinPiece) {
        emit(r, tb, fit, cta);
        tb += fit;
        rem -= fit;
        break;
      } else {
        break;
      }
    }
  }
  // What rounding and the minimum piece length left over: dealt out in pieces to the least loaded queues, each topped up to
  // the level all queues would reach if the leftovers were spread evenly (never a whole row on one queue unless it fits).
  if (ti < tail.size()) {
    double left = tail[ti].tc * rem + kItemOverhead;
    for (size_t t2 = ti + 1; t2 < tail.size(); ++t2) left += tail[t2].tc * (tail[t2].tiles + tail[t2].sink_tiles) + kItemOverhead;
    double have = 0;
    for (double v : load) have += v;
    const double level = (have + left) / n_cta + 2 * kItemOverhead;
    while (ti < tail.size()) {
      const int32_t cta = (int32_t)(std::min_element(load.begin(), load.end()) - load.begin());
      const Row &r = tail[ti];
      int32_t take = (int32_t)std::floor((level - load[cta] - kItemOverhead) / r.tc) - (tb == r.tile0 ? r.sink_tiles : 0);
      take = std::max(take, kMinPiece);
      if (take >= rem || rem - take < kMinPiece) {
        emit(r, tb, rem, cta);
        close_row();
      } else {
        emit(r, tb, take, cta);
        tb += take;
        rem -= take;
      }
    }
  }
  c.ideal = total / n_cta;
  for (double v : load) c.makespan = std::max(c.makespan, v);
  c.objective = c.makespan + kPartialCost * c.n_slots / n_cta;
}

bool is_pow2(int32_t x) { return x > 0 && (x & (x - 1)) == 0; }

} // namespace

slack_status build_plan(const slack_pool &shape, int32_t n_streams, const slack_stream *streams,
                        const slack_plan_opts &opts, int32_t default_sm_count, HostPlan &out, std::string &err) {
  char buf[256];
  auto fail = [&](slack_status st, const char *msg) {
    err = msg;
    return st;
  };
  if (n_streams < 0 || (n_streams > 0 && !streams)) return fail(SLACK_EINVAL, "n_streams < 0 or streams == NULL");
  if (shape.n_pages <= 0 || shape.n_heads <= 0) return fail(SLACK_EINVAL, "pool: n_pages and n_heads must be > 0");
  if (shape.dtype != SLACK_BF16 && shape.dtype != SLACK_F32 && shape.dtype != SLACK_FP8_E4M3)
    return fail(SLACK_EINVAL, "pool: unknown dtype");
  if (shape.head_dim != 64 && shape.head_dim != 128) return fail(SLACK_EUNSUPPORTED, "head_dim must be 64 or 128");
  if (!is_pow2(shape.page_size) || shape.page_size < 16)
    return fail(SLACK_EUNSUPPORTED, "page_size must be a power of two >= 16");
  if (opts.sm_count < 0 || opts.force_splits < 0) return fail(SLACK_EINVAL, "plan opts: negative sm_count/force_splits");

  out = HostPlan();
  out.n_pages = shape.n_pages;
  out.n_heads = shape.n_heads;
  out.head_dim = shape.head_dim;
  out.page_size = shape.page_size;
  out.dtype = shape.dtype;
  out.n_streams = n_streams;
  out.n_cta = opts.sm_count > 0 ? opts.sm_count : default_sm_count;
  const bool fp8 = shape.dtype == SLACK_FP8_E4M3;
  if (fp8 && (shape.head_dim != 128 || shape.page_size < kTileN || opts.force_simt))
    return fail(SLACK_EUNSUPPORTED, "FP8 pools need head_dim 128, page_size >= 128 and the tensor-core kernel");
  // tensor-core kernel: bf16 with head_dim 64 or 128, FP8 with head_dim 128 (checked above); fp32 pools and pages shorter
  // than a key tile go to the SIMT kernel
  const bool tc_ok = (shape.dtype == SLACK_BF16 || fp8) && shape.page_size >= kTileN;
  if (opts.cta_pairs < 0 || opts.cta_pairs > 2) return fail(SLACK_EINVAL, "plan opts: cta_pairs must be 0, 1 or 2");
  out.kernel_kind = (tc_ok && !opts.force_simt) ? 0 : 1;

  // ---- validate streams, build device stream records and the concatenated page table ------------------------
  std::vector<uint8_t> owned((size_t)shape.n_pages, 0);
  int64_t row = 0;
  const int32_t P = shape.page_size;
  for (int32_t i = 0; i < n_streams; ++i) {
    const slack_stream &s = streams[i];
    if (s.q_len < 0 || s.cache_len < 0 || s.window < 0 || s.n_table_pages < 0) {
      snprintf(buf, sizeof buf, "stream %d: negative q_len/cache_len/window/n_table_pages", i);
      return fail(SLACK_EINVAL, buf);
    }
    if (s.base < 0 || s.base >= P) {
      snprintf(buf, sizeof buf, "stream %d: base %d outside [0, page_size)", i, s.base);
      return fail(SLACK_EINVAL, buf);
    }
    if (s.sink_len < 0 || s.gap_slots < 0) {
      snprintf(buf, sizeof buf, "stream %d: negative sink_len / gap_slots", i);
      return fail(SLACK_EINVAL, buf);
    }
    if (s.gap_slots > 0 && (s.sink_len == 0 || s.cache_len < s.sink_len)) {
      snprintf(buf, sizeof buf, "stream %d: gap_slots needs sink_len > 0 and cache_len >= sink_len", i);
      return fail(SLACK_EINVAL, buf);
    }
    const int64_t n = (int64_t)s.cache_len + s.q_len;
    const int64_t end_pos = (int64_t)s.base + s.gap_slots + n; // one past the position of token n - 1
    if (end_pos > (int64_t)INT32_MAX / 2 || row + s.q_len > (int64_t)INT32_MAX / 2)
      return fail(SLACK_EINVAL, "batch too large for 32-bit token positions");
    const int32_t need = n > 0 ? ceil_div(end_pos, P) : 0;
    if (s.n_table_pages < need) {
      snprintf(buf, sizeof buf, "stream %d: page table has %d pages, needs %d", i, s.n_table_pages, need);
      return fail(SLACK_EINVAL, buf);
    }
    if (need > 0 && !s.page_table) {
      snprintf(buf, sizeof buf, "stream %d: page_table == NULL", i);
      return fail(SLACK_EINVAL, buf);
    }
    DevStream d{};
    d.q_row0 = (int32_t)row;
    d.qblock0 = out.mask_rows;
    out.mask_rows += ceil_div(s.q_len, kItemRows);
    out.mask_words_min = std::max<int32_t>(out.mask_words_min, ceil_div(ceil_div(end_pos, kTileN), 32));
    d.q_len = s.q_len;
    d.cache_len = s.cache_len;
    d.base = s.base;
    // visible tokens = [0, sink) U [max(sink, lo), n) ("sink + local"); token t sits at position base + t, plus
    // gap_slots behind the sink (slack.h).  One position range when the two touch and no slot is skipped between them.
    int64_t lo = (s.window > 0) ? std::max<int64_t>(0, n - s.window) : 0;
    const int64_t sink = std::min<int64_t>(s.sink_len, n);
    const bool one_range = lo <= sink && s.gap_slots == 0;
    if (one_range) lo = 0;
    else lo = std::max(lo, sink);
    d.pos_lo = (int32_t)(s.base + (one_range ? 0 : s.gap_slots) + lo);
    d.pos_hi = (int32_t)end_pos;
    d.sink_hi = (int32_t)(s.base + (one_range ? 0 : sink));
    d.app_pos0 = (int32_t)(s.base + s.cache_len + (s.cache_len >= s.sink_len ? s.gap_slots : 0));
    if (s.gap_slots > 0) { // earlier tokens: the sink [base, base + sink) and, behind the hole, [base + gap + sink, app_pos0)
      d.old_hi0 = s.base + s.sink_len;
      d.old_lo1 = s.base + s.gap_slots + s.sink_len;
    } else {
      d.old_hi0 = s.base + s.cache_len;
      d.old_lo1 = d.app_pos0;
    }
    d.pt_off = (int32_t)out.page_tables.size();
    d.n_table_pages = need;
    for (int32_t p = 0; p < need; ++p) {
      const int32_t id = s.page_table[p];
      if (id < 0 || id >= shape.n_pages) {
        snprintf(buf, sizeof buf, "stream %d: page_table[%d] = %d outside [0, %d)", i, p, id, shape.n_pages);
        return fail(SLACK_EINVAL, buf);
      }
      if (owned[id]) {
        snprintf(buf, sizeof buf, "stream %d: physical page %d is owned twice in the batch", i, id);
        return fail(SLACK_EINVAL, buf);
      }
      owned[id] = 1;
      out.page_tables.push_back(id);
    }
    out.streams.push_back(d);
    row += s.q_len;
  }
  out.total_q = (int32_t)row;
  if (out.page_tables.empty()) out.page_tables.push_back(0); // keep device arrays non-empty

  out.n_queues = out.n_cta;
  out.cta_begin.assign((size_t)out.n_cta + 1, 0);
  if (out.kernel_kind == 1) return SLACK_OK; // the SIMT kernel walks DevStream records directly: no items

  // ---- tensor-core path: geometry per stream ------------------------------------------------------------------
  std::vector<StreamGeom> order;
  for (int32_t i = 0; i < n_streams; ++i) {
    const DevStream &d = out.streams[i];
    if (d.q_len == 0) continue;
    StreamGeom g;
    g.idx = i;
    g.tile0 = d.pos_lo / kTileN;
    g.tiles = ceil_div(d.pos_hi, kTileN) - g.tile0;
    g.q_blocks = ceil_div(d.q_len, kItemRows);
    g.sink_tile0 = d.base / kTileN;
    g.sink_tiles = d.sink_hi > d.base ? ceil_div(d.sink_hi, kTileN) - g.sink_tile0 : 0;
    order.push_back(g);
  }
  std::stable_sort(order.begin(), order.end(),
                   [](const StreamGeom &a, const StreamGeom &b) { return a.tiles + a.sink_tiles > b.tiles + b.sink_tiles; });
  if (order.empty()) return SLACK_OK;

  // CTA pairs (attn_tc2.cu, tcgen05 cta_group::2): two SMs walk ONE queue together, each item's first 128 query rows on
  // the even CTA and the rest on the odd one, and share every K/V tile.  The plan is then made for n_cta / 2 queues.
  // Pays when most items have more than 128 rows; short chunks (decode-like) keep one CTA per item.
  // cta_pairs: 0 = automatic, 1 = never, 2 = always (needs an even CTA count).
  if (out.n_cta >= 2 && out.n_cta % 2 == 0 && !fp8 && shape.head_dim == 128) {
    bool pairs = opts.cta_pairs == 2;
    if (opts.cta_pairs == 0 && kAutoPairs) {
      int64_t rows = 0, padded = 0;
      for (const StreamGeom &g : order) {
        rows += out.streams[g.idx].q_len;
        padded += (int64_t)g.q_blocks * kItemRows;
      }
      pairs = rows * 100 >= padded * 85; // at least 85 % of the items' 256 query slots are real queries
    }
    if (pairs) out.kernel_kind = 2;
  }
  const int32_t n_queues = out.kernel_kind == 2 ? out.n_cta / 2 : out.n_cta;
  out.n_queues = n_queues;
  out.cta_begin.assign((size_t)n_queues + 1, 0);

  const int32_t t_max = order.front().tiles;
  Candidate best;
  bool have = false;
  std::vector<int32_t> parts(order.size());
  auto consider = [&](int32_t k, bool exact) {
    for (size_t i = 0; i < order.size(); ++i) {
      if (exact) {
        parts[i] = std::min(k, order[i].tiles);
      } else {
        const int32_t target = ceil_div(t_max, k); // chunk length the longest stream gets
        parts[i] = std::max(1, std::min(order[i].tiles, (int32_t)((order[i].tiles + target / 2) / target)));
      }
    }
    Candidate c;
    make_candidate(order, parts, out.streams, shape.n_heads, n_queues, out.kernel_kind == 2, c);
    if (!have || c.objective < best.objective - 1e-9) {
      best = std::move(c);
      have = true;
    }
  };
  if (opts.force_splits > 0) {
    consider(opts.force_splits, true);
  } else {
    consider(1, false); // no split at all: best when the rows already fill the queues evenly
    // rounding and the minimum piece length leave queues a little short or long of the target: try a few, keep the best
    const double scales[] = {1.0, 0.99, 1.01, 0.98, 1.02, 0.97, 1.03, 1.045, 1.06};
    for (double sc : scales) {
      Candidate c;
      make_balanced(order, out.streams, shape.n_heads, n_queues, out.kernel_kind == 2, out.kernel_kind == 0 && shape.head_dim == 128, sc, c);
      if (c.objective < best.objective - 1e-9) best = std::move(c);
    }
  }

  // ---- emit per-CTA queues (stable: queue order = item order) ------------------------------------------------
  const size_t n_items = best.items.size();
  std::vector<int32_t> count((size_t)n_queues, 0);
  for (size_t i = 0; i < n_items; ++i) count[best.item_cta[i]]++;
  for (int32_t c = 0; c < n_queues; ++c) out.cta_begin[c + 1] = out.cta_begin[c] + count[c];
  std::vector<int32_t> cursor(out.cta_begin.begin(), out.cta_begin.end() - 1);
  out.items.resize(n_items);
  out.item_cta.resize(n_items);
  for (size_t i = 0; i < n_items; ++i) {
    const int32_t c = best.item_cta[i];
    out.items[cursor[c]] = best.items[i];
    out.item_cta[cursor[c]] = c;
    cursor[c]++;
  }
  out.combines = std::move(best.combines);
  out.n_partial_slots = best.n_slots;
  out.makespan = best.makespan;
  out.ideal = best.ideal;
  out.ws.o_bytes = (size_t)out.n_partial_slots * kItemRows * shape.head_dim * sizeof(float);
  out.ws.lse_off = out.ws.o_bytes;
  out.ws.total = out.ws.o_bytes + (size_t)out.n_partial_slots * kItemRows * sizeof(float);
  if (fp8) { // room for the quantised Q behind the split-KV partials
    out.q8_off = (out.ws.total + 127) & ~(size_t)127;
    out.q8_scale_off = out.q8_off + (size_t)out.total_q * shape.n_heads * shape.head_dim;
    out.ws.total = out.q8_scale_off + (size_t)out.total_q * shape.n_heads * sizeof(float);
  }
  // block-sparse bookkeeping: which mask row an item reads and where its compacted step list goes
  for (DevItem &it : out.items) {
    out.has_dual |= it.dual != 0;
    const DevStream &d = out.streams[it.stream];
    it.mask_row = d.qblock0 + (it.q_row0 - d.q_row0) / kItemRows;
    it.step_off = (int32_t)out.total_steps;
    const int32_t steps = it.sink_tiles + (it.kv_tile_end - it.kv_tile_begin);
    out.total_steps += steps;
    out.max_item_steps = std::max(out.max_item_steps, steps);
  }
  if (out.total_steps > (int64_t)INT32_MAX / 2) return fail(SLACK_EINVAL, "batch too large (key-tile steps)");
  out.sparse_steps_off = (out.ws.total + 15) & ~(size_t)15;
  out.sparse_count_off = (out.sparse_steps_off + (size_t)out.total_steps * sizeof(uint16_t) + 15) & ~(size_t)15;
  out.sparse_total = out.sparse_count_off + out.items.size() * sizeof(int32_t);
  return SLACK_OK;
}

} // namespace slack
