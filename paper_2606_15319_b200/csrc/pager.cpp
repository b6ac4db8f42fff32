// pager.cpp — A0 + A5: page bookkeeping of one worker's paged KV pool (host only, integers only; no CUDA).
//
// PAPER.md P:251 (§4.4): K/V of all streams on a worker live in one pool "mapped to physical pages through a logical page
// table, avoiding fragmentation"; P:84 (§2.1): every finished chunk is "appended to a rolling KV cache for subsequent
// chunks"; the cache "preserves the first few chunks as a global sink and keeps KV entries only for the most recent
// W chunks".  This file is that bookkeeping: a free list of physical page ids, one page table per stream, the commit
// Lc += Lq (A5) and the release of pages that the window of the next chunk no longer covers (A0).  The attention and append
// kernels see its result only as slack_stream descriptors.
//
// Numbering (include/slack.h token -> slot rule): a stream's HELD tokens are numbered 0 .. Lc-1, the sink first; token t
// sits at position base + t, plus gap_slots when t >= sink_len; position p is slot p % P of table page p / P.  Dropping
// tokens that left the window removes them from the numbering: without a sink the numbering restarts at the first kept
// token (base = its slot), with a sink the hole between the sink and the first kept token is gap_slots, and every table
// page that lay wholly inside the hole has been taken out of the table.  Positions therefore stay bounded by
// sink + window + chunk + 2 pages however long the stream runs.
#include <algorithm>
#include <cstdio>
#include <memory>
#include <new>
#include <string>
#include <vector>

#include "../../include/slack.h"

namespace {

struct CacheStream {
  bool open = false;
  int32_t window = 0, sink = 0;
  int32_t base = 0, gap = 0;
  int32_t cache_len = 0;   // held tokens of committed chunks
  int32_t pending_q = -1;  // chunk begun and not yet committed (-1: none)
  std::vector<int32_t> table;
};

int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

} // namespace

struct slack_cache_s {
  int32_t n_pages = 0, page_size = 0, policy = 0;
  std::vector<int32_t> free_list; // stack: back() is handed out next (most recently freed first)
  std::vector<std::unique_ptr<CacheStream>> streams;
  std::string err;
};

namespace {

slack_status fail(slack_cache_s *c, slack_status st, const char *msg) {
  if (c) c->err = msg;
  return st;
}

CacheStream *get(slack_cache_s *c, int32_t id) {
  if (!c || id < 0 || id >= (int32_t)c->streams.size() || !c->streams[id] || !c->streams[id]->open) return nullptr;
  return c->streams[id].get();
}

// A0, first half: drop what the window of a chunk of q_len tokens no longer covers.
void trim(slack_cache_s *c, CacheStream &s, int32_t q_len) {
  if (s.window <= 0) return;
  const int64_t P = c->page_size;
  const int64_t n = (int64_t)s.cache_len + q_len;
  // first visible token behind the sink; tokens of the chunk itself are not in the pool yet and cannot be dropped
  const int64_t lo = std::min<int64_t>(std::max<int64_t>(0, n - s.window), s.cache_len);
  if (lo <= s.sink) return;                                   // the window still touches the sink (or the stream start)
  const int64_t first_local = (int64_t)s.base + s.gap + s.sink; // position of held token `sink`
  const int64_t pos_lo = (int64_t)s.base + s.gap + lo;
  const int64_t first_free = s.sink > 0 ? ceil_div((int64_t)s.base + s.sink, P) : 0; // first table page that holds no sink token
  const int64_t keep_page = pos_lo / P;                            // table page of the first visible token
  const int64_t k = std::max<int64_t>(0, keep_page - first_free);    // pages wholly inside the hole
  const int64_t keep_pos = c->policy == SLACK_TRIM_TOKENS ? pos_lo : std::max(first_local, k > 0 ? keep_page * P : first_local);
  const int64_t dropped = keep_pos - first_local;
  if (dropped <= 0 && k == 0) return;
  for (int64_t i = first_free + k - 1; i >= first_free; --i) c->free_list.push_back(s.table[(size_t)i]);
  s.table.erase(s.table.begin() + first_free, s.table.begin() + first_free + k);
  s.cache_len -= (int32_t)dropped;
  const int64_t new_first = keep_pos - k * P;
  if (s.sink > 0) s.gap = (int32_t)(new_first - ((int64_t)s.base + s.sink));
  else s.base = (int32_t)new_first;
}

void fill(const slack_cache_s *, const CacheStream &s, int32_t q_len, slack_stream *d) {
  d->q_len = q_len;
  d->cache_len = s.cache_len;
  d->base = s.base;
  d->window = s.window;
  d->sink_len = s.sink;
  d->gap_slots = s.gap;
  d->n_table_pages = (int32_t)s.table.size();
  d->reserved = 0;
  d->page_table = s.table.data();
}

} // namespace

extern "C" {

slack_status slack_cache_create(int32_t n_pages, int32_t page_size, int32_t trim_policy, slack_cache_t **out) {
  if (!out) return SLACK_EINVAL;
  *out = nullptr;
  if (n_pages <= 0 || page_size <= 0 || (page_size & (page_size - 1)) != 0) return SLACK_EINVAL;
  if (trim_policy != SLACK_TRIM_PAGES && trim_policy != SLACK_TRIM_TOKENS) return SLACK_EINVAL;
  slack_cache_s *c = new (std::nothrow) slack_cache_s();
  if (!c) return SLACK_ENOMEM;
  c->n_pages = n_pages;
  c->page_size = page_size;
  c->policy = trim_policy;
  c->free_list.resize((size_t)n_pages);
  for (int32_t i = 0; i < n_pages; ++i) c->free_list[(size_t)i] = n_pages - 1 - i; // page 0 is handed out first
  *out = c;
  return SLACK_OK;
}

void slack_cache_destroy(slack_cache_t *c) { delete c; }

const char *slack_cache_last_error(const slack_cache_t *c) { return c ? c->err.c_str() : "NULL cache"; }
int32_t slack_cache_free_pages(const slack_cache_t *c) { return c ? (int32_t)c->free_list.size() : 0; }
int32_t slack_cache_stream_pages(const slack_cache_t *c, int32_t id) {
  CacheStream *s = get(const_cast<slack_cache_s *>(c), id);
  return s ? (int32_t)s->table.size() : -1;
}

slack_status slack_cache_open(slack_cache_t *c, int32_t window, int32_t sink_len, int32_t *stream_id) {
  if (!c || !stream_id) return SLACK_EINVAL;
  if (window < 0 || sink_len < 0) return fail(c, SLACK_EINVAL, "negative window / sink_len");
  int32_t id = -1;
  for (size_t i = 0; i < c->streams.size(); ++i)
    if (!c->streams[i]->open) {
      id = (int32_t)i;
      break;
    }
  if (id < 0) {
    c->streams.emplace_back(new CacheStream());
    id = (int32_t)c->streams.size() - 1;
  }
  CacheStream &s = *c->streams[(size_t)id];
  s = CacheStream();
  s.open = true;
  s.window = window;
  s.sink = sink_len;
  *stream_id = id;
  return SLACK_OK;
}

slack_status slack_cache_close(slack_cache_t *c, int32_t id) {
  CacheStream *s = get(c, id);
  if (!s) return fail(c, SLACK_EINVAL, "no such open stream");
  for (size_t i = s->table.size(); i-- > 0;) c->free_list.push_back(s->table[i]);
  *s = CacheStream();
  return SLACK_OK;
}

slack_status slack_cache_begin_chunk(slack_cache_t *c, int32_t id, int32_t q_len, slack_stream *desc) {
  CacheStream *s = get(c, id);
  if (!s) return fail(c, SLACK_EINVAL, "no such open stream");
  if (!desc || q_len < 0) return fail(c, SLACK_EINVAL, "desc NULL or q_len < 0");
  if (s->pending_q >= 0) {
    if (s->pending_q != q_len) return fail(c, SLACK_EINVAL, "a chunk of another length is begun and not committed");
    fill(c, *s, q_len, desc);
    return SLACK_OK;
  }
  if ((int64_t)s->base + s->gap + s->cache_len + q_len > (int64_t)INT32_MAX / 2)
    return fail(c, SLACK_EINVAL, "stream too long for 32-bit positions");
  trim(c, *s, q_len);
  const int64_t n = (int64_t)s->cache_len + q_len;
  const int64_t end_pos = (int64_t)s->base + s->gap + n;
  const int64_t need = n > 0 ? ceil_div(end_pos, c->page_size) : 0;
  const int64_t more = need - (int64_t)s->table.size();
  if (more > (int64_t)c->free_list.size()) {
    char buf[128];
    snprintf(buf, sizeof buf, "pool exhausted: stream needs %lld more pages, %zu free", (long long)more, c->free_list.size());
    return fail(c, SLACK_ENOMEM, buf);
  }
  for (int64_t i = 0; i < more; ++i) {
    s->table.push_back(c->free_list.back());
    c->free_list.pop_back();
  }
  s->pending_q = q_len;
  fill(c, *s, q_len, desc);
  return SLACK_OK;
}

slack_status slack_cache_commit(slack_cache_t *c, int32_t id) {
  CacheStream *s = get(c, id);
  if (!s) return fail(c, SLACK_EINVAL, "no such open stream");
  if (s->pending_q < 0) return fail(c, SLACK_EINVAL, "no chunk begun on this stream");
  s->cache_len += s->pending_q;
  s->pending_q = -1;
  return SLACK_OK;
}

} // extern "C"
