// api.cu — the C ABI of include/slack.h: context, plan objects, argument checks, TMA descriptors, kernel launches.
// No arithmetic of the method lives here; see append.cu / attn_tc.cu / attn_simt.cu / combine.cu.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <algorithm>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "kernels.h"
#include "slack_internal.h"

using namespace slack;

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

namespace {

// ---- ctx-owned arena: device memory + a pinned host mirror of the same size ---------------------------------------
// Plan tables and the staging tables of slack_kv_append / slack_kv_transfer are cut out of it (first fit, coalescing
// free list).  A block is filled through its host mirror and copied with one cudaMemcpyAsync; it is handed back by
// release_after(events): the block returns to the free list once every event has completed, so nothing ever waits for
// the device on the host (the staging buffer used to be re-used while kernels of an earlier call on another
// stream were still reading it).  Segments are added when the arena runs dry (rare: a few MB hold hundreds of plans).
struct ArenaBlock {
  int seg = -1;
  size_t off = 0, size = 0;
  explicit operator bool() const { return seg >= 0; }
};

struct Arena {
  struct Segment {
    uint8_t *dev = nullptr, *host = nullptr;
    size_t cap = 0;
    std::vector<std::pair<size_t, size_t>> free_list; // (offset, size), sorted by offset, coalesced
  };
  struct Pending {
    ArenaBlock blk;
    std::vector<cudaEvent_t> events;
  };
  std::vector<Segment> segs;
  std::vector<Pending> pending;
  std::vector<cudaEvent_t> event_pool;

  cudaError_t get_event(cudaEvent_t *ev) {
    if (!event_pool.empty()) {
      *ev = event_pool.back();
      event_pool.pop_back();
      return cudaSuccess;
    }
    return cudaEventCreateWithFlags(ev, cudaEventDisableTiming);
  }
  void put_event(cudaEvent_t ev) { event_pool.push_back(ev); }

  void free_now(const ArenaBlock &b) {
    auto &fl = segs[(size_t)b.seg].free_list;
    auto it = std::lower_bound(fl.begin(), fl.end(), std::make_pair(b.off, (size_t)0));
    it = fl.insert(it, {b.off, b.size});
    if (it + 1 != fl.end() && it->first + it->second == (it + 1)->first) {
      it->second += (it + 1)->second;
      fl.erase(it + 1);
    }
    if (it != fl.begin() && (it - 1)->first + (it - 1)->second == it->first) {
      (it - 1)->second += it->second;
      fl.erase(it);
    }
  }
  // blocks whose guarding events have all completed go back to the free lists (never blocks)
  void reclaim() {
    for (size_t i = 0; i < pending.size();) {
      Pending &p = pending[i];
      while (!p.events.empty() && cudaEventQuery(p.events.back()) == cudaSuccess) {
        put_event(p.events.back());
        p.events.pop_back();
      }
      if (p.events.empty()) {
        free_now(p.blk);
        pending[i] = std::move(pending.back());
        pending.pop_back();
      } else {
        ++i;
      }
    }
    (void)cudaGetLastError(); // cudaErrorNotReady from the queries is not an error
  }
  void release_after(const ArenaBlock &b, std::vector<cudaEvent_t> &&events) {
    if (!b) return;
    if (events.empty()) {
      free_now(b);
      return;
    }
    pending.push_back({b, std::move(events)});
  }
  ArenaBlock try_alloc(size_t size) {
    for (size_t si = 0; si < segs.size(); ++si) {
      auto &fl = segs[si].free_list;
      for (size_t i = 0; i < fl.size(); ++i)
        if (fl[i].second >= size) {
          ArenaBlock b;
          b.seg = (int)si;
          b.off = fl[i].first;
          b.size = size;
          fl[i].first += size;
          fl[i].second -= size;
          if (fl[i].second == 0) fl.erase(fl.begin() + (long)i);
          return b;
        }
    }
    return ArenaBlock();
  }
  cudaError_t alloc(size_t size, ArenaBlock *out) {
    size = (size + 255) & ~(size_t)255;
    if (size == 0) size = 256;
    reclaim();
    *out = try_alloc(size);
    if (*out) return cudaSuccess;
    Segment sg;
    sg.cap = std::max<size_t>(size * 2, segs.empty() ? ((size_t)4 << 20) : segs.back().cap * 2);
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(&sg.dev), sg.cap);
    if (e != cudaSuccess) return e;
    e = cudaMallocHost(reinterpret_cast<void **>(&sg.host), sg.cap);
    if (e != cudaSuccess) {
      cudaFree(sg.dev);
      return e;
    }
    sg.free_list.push_back({0, sg.cap});
    segs.push_back(std::move(sg));
    *out = try_alloc(size);
    return *out ? cudaSuccess : cudaErrorMemoryAllocation;
  }
  uint8_t *dev(const ArenaBlock &b) const { return segs[(size_t)b.seg].dev + b.off; }
  uint8_t *host(const ArenaBlock &b) const { return segs[(size_t)b.seg].host + b.off; }
  void destroy() { // after a device synchronisation
    for (Pending &p : pending)
      for (cudaEvent_t e : p.events) cudaEventDestroy(e);
    for (cudaEvent_t e : event_pool) cudaEventDestroy(e);
    for (Segment &sg : segs) {
      cudaFree(sg.dev);
      cudaFreeHost(sg.host);
    }
    pending.clear();
    event_pool.clear();
    segs.clear();
  }
};

constexpr int kProfKinds = 3; // bit index of SLACK_PROF_ATTENTION / _APPEND / _COMBINE

} // namespace

struct slack_ctx {
  int device = -1;
  int sm_count = 148;
  std::string err;
  int last_launches = 0;
  EncodeTiledFn encode = nullptr;
  bool tc_configured = false;
  Arena arena;
  // plan tables are uploaded on a private non-blocking stream: slack_plan never waits for the caller's queued work
  cudaStream_t up_stream = nullptr;
  std::vector<slack_plan_s *> live_plans; // orphaned (ctx = NULL) by slack_destroy
  // time-out record of the in-kernel barrier waits: mapped pinned, 4 words, survives a trapped launch
  unsigned long long *h_dbg = nullptr;
  unsigned long long *d_dbg = nullptr;
#ifdef SLACK_DIAGNOSTICS
  float *dbg_s = nullptr;
  uint32_t *dbg_t = nullptr;
#endif
  // per-launch timing (slack_profile_enable): event pairs per kind, [2i] before, [2i+1] after
  int prof_mask = 0;
  std::vector<cudaEvent_t> prof_events[kProfKinds];
  size_t prof_used[kProfKinds] = {0, 0, 0};
};

struct slack_plan_s {
  slack_ctx *ctx = nullptr; // NULL once the context is gone
  HostPlan hp;
  int max_q_len = 0;
  ArenaBlock blk;           // one arena block holding all tables
  DevStream *d_streams = nullptr;
  int32_t *d_page_tables = nullptr;
  DevItem *d_items = nullptr;
  int32_t *d_cta_begin = nullptr;
  DevCombine *d_combines = nullptr;
  // bookkeeping of a plan in use (a plan's TABLES are immutable; this is not part of them)
  mutable cudaEvent_t ready_ev = nullptr;      // upload finished; NULL once that has been observed
  mutable std::vector<cudaStream_t> used_on;   // streams that ran kernels reading the tables
};

namespace {

slack_status set_err(slack_ctx *ctx, slack_status st, const std::string &msg) {
  if (ctx) ctx->err = msg;
  return st;
}
slack_status cuda_err(slack_ctx *ctx, cudaError_t e, const char *what) {
  char buf[384];
  int n = snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
  if (ctx && ctx->h_dbg && ctx->h_dbg[0] == 0xDEADull && n > 0 && (size_t)n < sizeof buf)
    snprintf(buf + n, sizeof buf - (size_t)n, " [a bounded barrier wait timed out: block %llu thread %llu barrier tag %llu parity %llu]",
             ctx->h_dbg[1] >> 32, ctx->h_dbg[1] & 0xffffffffull, ctx->h_dbg[2] >> 32, ctx->h_dbg[2] & 0xffffffffull);
  return set_err(ctx, SLACK_ECUDA, buf);
}
#define SLACK_CUDA(ctx, call)                                  \
  do {                                                         \
    cudaError_t e__ = (call);                                  \
    if (e__ != cudaSuccess) return cuda_err(ctx, e__, #call);  \
  } while (0)

bool aligned(const void *p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }
size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

slack_status ensure_device(slack_ctx *ctx) {
  if (!ctx) return SLACK_EINVAL;
  if (ctx->device < 0) return set_err(ctx, SLACK_ECUDA, "host-only context: no CUDA device (there is no CPU fallback)");
  int cur = -1;
  SLACK_CUDA(ctx, cudaGetDevice(&cur));
  if (cur != ctx->device) SLACK_CUDA(ctx, cudaSetDevice(ctx->device));
  return SLACK_OK;
}

slack_status check_pool(slack_ctx *ctx, const slack_pool *pool, const HostPlan *hp) {
  if (!pool || !pool->k_pool || !pool->v_pool) return set_err(ctx, SLACK_EINVAL, "pool or pool pointers NULL");
  if (!aligned(pool->k_pool, 16) || !aligned(pool->v_pool, 16)) return set_err(ctx, SLACK_EINVAL, "pool pointers must be 16-byte aligned");
  if (pool->dtype == SLACK_FP8_E4M3 && (!pool->k_scale || !pool->v_scale || !aligned(pool->k_scale, 4) || !aligned(pool->v_scale, 4)))
    return set_err(ctx, SLACK_EINVAL, "FP8 pool: k_scale / v_scale NULL or misaligned");
  if (hp && (pool->n_pages != hp->n_pages || pool->n_heads != hp->n_heads || pool->head_dim != hp->head_dim ||
             pool->page_size != hp->page_size || pool->dtype != hp->dtype))
    return set_err(ctx, SLACK_ESTALE_PLAN, "plan was made for a different pool shape / dtype");
  return SLACK_OK;
}

// 2-D map over [rows][cols] elements with boxes of 128 bytes x box_rows rows (bf16: 64 elements, e4m3 codes: 128)
slack_status make_map(slack_ctx *ctx, CUtensorMap *m, const void *base, uint64_t cols, uint64_t rows, uint32_t box_rows = 128,
                      bool bytes = false) {
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {cols * (bytes ? 1 : 2)};
  const cuuint32_t box[2] = {bytes ? 128u : 64u, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = ctx->encode(m, bytes ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[128];
    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
    return set_err(ctx, SLACK_ECUDA, buf);
  }
  return SLACK_OK;
}

// bf16 rows [rows][cols] read in plain (unswizzled) boxes of 128 rows x 128 elements: the FP8 append stages the 256-byte
// (token, head) rows of one key block with a single TMA instruction
slack_status make_rows_map(slack_ctx *ctx, CUtensorMap *m, const void *base, uint64_t cols, uint64_t rows) {
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {cols * 2};
  const cuuint32_t box[2] = {128u, 128u};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = ctx->encode(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[128];
    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
    return set_err(ctx, SLACK_ECUDA, buf);
  }
  return SLACK_OK;
}

int elem_bytes(int dtype) { return dtype == SLACK_BF16 ? 2 : dtype == SLACK_FP8_E4M3 ? 1 : 4; }

// The first launches that use a plan wait, on the device, for its upload; every stream that reads the tables is noted
// so that slack_plan_destroy can guard the block with an event per stream.
slack_status plan_in_use(slack_ctx *ctx, const slack_plan_s *plan, cudaStream_t cs) {
  if (plan->ready_ev) {
    if (cudaEventQuery(plan->ready_ev) == cudaSuccess) {
      ctx->arena.put_event(plan->ready_ev);
      plan->ready_ev = nullptr;
    } else {
      (void)cudaGetLastError();
      SLACK_CUDA(ctx, cudaStreamWaitEvent(cs, plan->ready_ev, 0));
    }
  }
  if (std::find(plan->used_on.begin(), plan->used_on.end(), cs) == plan->used_on.end()) plan->used_on.push_back(cs);
  return SLACK_OK;
}

// event pair around one kernel launch (slack_profile_enable); returns the "after" event to record, or NULL
slack_status prof_begin(slack_ctx *ctx, int kind_bit, cudaStream_t cs, cudaEvent_t *after) {
  *after = nullptr;
  if (!(ctx->prof_mask & (1 << kind_bit))) return SLACK_OK;
  auto &ev = ctx->prof_events[kind_bit];
  size_t &used = ctx->prof_used[kind_bit];
  while (ev.size() < 2 * (used + 1)) {
    cudaEvent_t e;
    SLACK_CUDA(ctx, cudaEventCreate(&e));
    ev.push_back(e);
  }
  SLACK_CUDA(ctx, cudaEventRecord(ev[2 * used], cs));
  *after = ev[2 * used + 1];
  return SLACK_OK;
}
slack_status prof_end(slack_ctx *ctx, int kind_bit, cudaStream_t cs, cudaEvent_t after) {
  if (!after) return SLACK_OK;
  SLACK_CUDA(ctx, cudaEventRecord(after, cs));
  ctx->prof_used[kind_bit]++;
  return SLACK_OK;
}

} // namespace

extern "C" {

int32_t slack_abi_version(void) { return SLACK_ABI_VERSION; }

slack_status slack_create(slack_ctx **out, int device) {
  if (!out) return SLACK_EINVAL;
  *out = nullptr;
  slack_ctx *ctx = new (std::nothrow) slack_ctx();
  if (!ctx) return SLACK_ENOMEM;
  ctx->device = device;
  if (device >= 0) {
    cudaError_t e = cudaSetDevice(device);
    int sm = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) {
      ctx->sm_count = sm;
      void *fn = nullptr;
      cudaDriverEntryPointQueryResult qres;
      e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
      if (e == cudaSuccess && qres == cudaDriverEntryPointSuccess) ctx->encode = reinterpret_cast<EncodeTiledFn>(fn);
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->up_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) {
      e = cudaHostAlloc(reinterpret_cast<void **>(&ctx->h_dbg), 4 * sizeof(unsigned long long), cudaHostAllocMapped);
      if (e == cudaSuccess) {
        memset(ctx->h_dbg, 0, 4 * sizeof(unsigned long long));
        e = cudaHostGetDevicePointer(reinterpret_cast<void **>(&ctx->d_dbg), ctx->h_dbg, 0);
      }
    }
    if (e != cudaSuccess) {
      delete ctx;
      return SLACK_ECUDA;
    }
  }
  *out = ctx;
  return SLACK_OK;
}

void slack_destroy(slack_ctx *ctx) {
  if (!ctx) return;
  for (slack_plan_s *pl : ctx->live_plans) { // plans may outlive the context: they keep their host tables only
    pl->ctx = nullptr;
    pl->blk = ArenaBlock();
    pl->ready_ev = nullptr;
  }
  if (ctx->device >= 0) {
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize(); // kernels that read arena blocks have finished
    ctx->arena.destroy();
    if (ctx->up_stream) cudaStreamDestroy(ctx->up_stream);
    if (ctx->h_dbg) cudaFreeHost(ctx->h_dbg);
    for (auto &v : ctx->prof_events)
      for (cudaEvent_t e : v) cudaEventDestroy(e);
  }
  delete ctx;
}

const char *slack_last_error(const slack_ctx *ctx) { return ctx ? ctx->err.c_str() : "NULL context"; }
int32_t slack_last_launch_count(const slack_ctx *ctx) { return ctx ? ctx->last_launches : 0; }

#ifdef SLACK_DIAGNOSTICS
/* diagnostics build only (include/slack_diag.h) */
slack_status slack_debug_set(slack_ctx *ctx, int32_t key, void *value) {
  if (!ctx) return SLACK_EINVAL;
  if (key == 0) {
    ctx->dbg_s = reinterpret_cast<float *>(value);
    return SLACK_OK;
  }
  if (key == 1) {
    ctx->dbg_t = reinterpret_cast<uint32_t *>(value);
    return SLACK_OK;
  }
  return set_err(ctx, SLACK_EINVAL, "unknown debug key");
}
#endif

slack_status slack_profile_enable(slack_ctx *ctx, int32_t kinds) {
  if (!ctx) return SLACK_EINVAL;
  if (kinds < 0 || kinds >= (1 << kProfKinds)) return set_err(ctx, SLACK_EINVAL, "unknown profile kind");
  ctx->prof_mask = kinds;
  return SLACK_OK;
}
slack_status slack_profile_read(slack_ctx *ctx, int32_t kind, double *ms_out, int32_t capacity, int32_t *n_launches) {
  if (!ctx || !n_launches || capacity < 0 || (capacity > 0 && !ms_out)) return SLACK_EINVAL;
  *n_launches = 0;
  int bit = -1;
  for (int b = 0; b < kProfKinds; ++b)
    if (kind == (1 << b)) bit = b;
  if (bit < 0) return set_err(ctx, SLACK_EINVAL, "slack_profile_read: kind must be exactly one SLACK_PROF_* bit");
  const size_t used = ctx->prof_used[bit];
  if (used == 0) return SLACK_OK;
  slack_status st = ensure_device(ctx);
  if (st != SLACK_OK) return st;
  const auto &ev = ctx->prof_events[bit];
  for (size_t i = 0; i < used; ++i) {
    float ms = 0.f;
    SLACK_CUDA(ctx, cudaEventSynchronize(ev[2 * i + 1]));
    SLACK_CUDA(ctx, cudaEventElapsedTime(&ms, ev[2 * i], ev[2 * i + 1]));
    if ((int32_t)i < capacity) ms_out[i] = ms;
  }
  *n_launches = (int32_t)used;
  ctx->prof_used[bit] = 0;
  return SLACK_OK;
}

/* ------------------------------------------------------------------------------------------------ plan */
slack_status slack_plan(slack_ctx *ctx, const slack_pool *pool_shape, int32_t n_streams, const slack_stream *streams,
                        const slack_plan_opts *opts, slack_plan_t **plan_out) {
  if (!ctx) return SLACK_EINVAL;
  if (!pool_shape || !plan_out) return set_err(ctx, SLACK_EINVAL, "pool_shape or plan NULL");
  *plan_out = nullptr;
  slack_plan_opts o{};
  if (opts) o = *opts;
  slack_plan_s *pl = new (std::nothrow) slack_plan_s();
  if (!pl) return set_err(ctx, SLACK_ENOMEM, "out of host memory");
  pl->ctx = ctx;
  std::string err;
  slack_status st;
  try {
    st = build_plan(*pool_shape, n_streams, streams, o, ctx->sm_count, pl->hp, err);
  } catch (const std::bad_alloc &) {
    delete pl;
    return set_err(ctx, SLACK_ENOMEM, "out of host memory while planning");
  }
  if (st != SLACK_OK) {
    delete pl;
    return set_err(ctx, st, err);
  }
  for (const DevStream &s : pl->hp.streams) pl->max_q_len = s.q_len > pl->max_q_len ? s.q_len : pl->max_q_len;

  if (ctx->device >= 0) {
    slack_status ds = ensure_device(ctx);
    if (ds != SLACK_OK) {
      delete pl;
      return ds;
    }
    const HostPlan &hp = pl->hp;
    const size_t b_streams = align_up(hp.streams.size() * sizeof(DevStream) + 16, 256);
    const size_t b_pt = align_up(hp.page_tables.size() * sizeof(int32_t), 256);
    const size_t b_items = align_up(hp.items.size() * sizeof(DevItem) + 16, 256);
    const size_t b_cta = align_up(hp.cta_begin.size() * sizeof(int32_t), 256);
    const size_t b_comb = align_up(hp.combines.size() * sizeof(DevCombine) + 16, 256);
    const size_t total = b_streams + b_pt + b_items + b_cta + b_comb;
    cudaError_t e = ctx->arena.alloc(total, &pl->blk);
    if (e != cudaSuccess) {
      delete pl;
      return cuda_err(ctx, e, "plan tables: arena allocation");
    }
    uint8_t *h = ctx->arena.host(pl->blk);
    memset(h, 0, total);
    size_t off = 0;
    auto put = [&](const void *src, size_t n, size_t padded) {
      if (n) memcpy(h + off, src, n);
      const size_t at = off;
      off += padded;
      return at;
    };
    const size_t o_streams = put(hp.streams.data(), hp.streams.size() * sizeof(DevStream), b_streams);
    const size_t o_pt = put(hp.page_tables.data(), hp.page_tables.size() * sizeof(int32_t), b_pt);
    const size_t o_items = put(hp.items.data(), hp.items.size() * sizeof(DevItem), b_items);
    const size_t o_cta = put(hp.cta_begin.data(), hp.cta_begin.size() * sizeof(int32_t), b_cta);
    const size_t o_comb = put(hp.combines.data(), hp.combines.size() * sizeof(DevCombine), b_comb);
    uint8_t *b = ctx->arena.dev(pl->blk);
    // asynchronous upload from the pinned mirror; the first launches that use the plan wait for ready_ev on the device
    e = cudaMemcpyAsync(b, h, total, cudaMemcpyHostToDevice, ctx->up_stream);
    if (e == cudaSuccess) e = ctx->arena.get_event(&pl->ready_ev);
    if (e == cudaSuccess) e = cudaEventRecord(pl->ready_ev, ctx->up_stream);
    if (e != cudaSuccess) {
      cudaStreamSynchronize(ctx->up_stream);
      ctx->arena.free_now(pl->blk);
      delete pl;
      return cuda_err(ctx, e, "plan upload");
    }
    pl->d_streams = reinterpret_cast<DevStream *>(b + o_streams);
    pl->d_page_tables = reinterpret_cast<int32_t *>(b + o_pt);
    pl->d_items = reinterpret_cast<DevItem *>(b + o_items);
    pl->d_cta_begin = reinterpret_cast<int32_t *>(b + o_cta);
    pl->d_combines = reinterpret_cast<DevCombine *>(b + o_comb);
  }
  ctx->live_plans.push_back(pl);
  *plan_out = pl;
  return SLACK_OK;
}

void slack_plan_destroy(slack_plan_t *plan) {
  if (!plan) return;
  slack_ctx *ctx = plan->ctx;
  if (ctx) {
    auto it = std::find(ctx->live_plans.begin(), ctx->live_plans.end(), plan);
    if (it != ctx->live_plans.end()) ctx->live_plans.erase(it);
    if (plan->blk && ctx->device >= 0) {
      int cur = -1;
      if (cudaGetDevice(&cur) == cudaSuccess && cur != ctx->device) cudaSetDevice(ctx->device);
      // the block returns to the arena once the upload and every stream that read the tables have passed this point
      std::vector<cudaEvent_t> guard;
      if (plan->ready_ev) guard.push_back(plan->ready_ev);
      bool ok = true;
      for (cudaStream_t cs : plan->used_on) {
        cudaEvent_t ev;
        if (ctx->arena.get_event(&ev) != cudaSuccess || cudaEventRecord(ev, cs) != cudaSuccess) {
          ok = false;
          break;
        }
        guard.push_back(ev);
      }
      if (!ok) { // cannot guard it: fall back to waiting for the device once
        cudaDeviceSynchronize();
        (void)cudaGetLastError();
        for (cudaEvent_t ev : guard) ctx->arena.put_event(ev);
        guard.clear();
      }
      ctx->arena.release_after(plan->blk, std::move(guard));
    }
  }
  delete plan;
}

size_t slack_plan_workspace_bytes(const slack_plan_t *plan) { return plan ? plan->hp.ws.total : 0; }
size_t slack_plan_sparse_workspace_bytes(const slack_plan_t *plan) { return plan ? plan->hp.sparse_total : 0; }
int32_t slack_plan_mask_rows(const slack_plan_t *plan) { return plan ? plan->hp.mask_rows : 0; }
int32_t slack_plan_mask_min_words(const slack_plan_t *plan) { return plan ? plan->hp.mask_words_min : 0; }
int32_t slack_plan_num_items(const slack_plan_t *plan) { return plan ? (int32_t)plan->hp.items.size() : 0; }
int32_t slack_plan_num_partial_slots(const slack_plan_t *plan) { return plan ? plan->hp.n_partial_slots : 0; }
int32_t slack_plan_kernel_kind(const slack_plan_t *plan) { return plan ? plan->hp.kernel_kind : -1; }

int32_t slack_plan_get_items(const slack_plan_t *plan, slack_work_item *items, int32_t capacity) {
  if (!plan || !items || capacity <= 0) return 0;
  const HostPlan &hp = plan->hp;
  const int32_t n = (int32_t)hp.items.size() < capacity ? (int32_t)hp.items.size() : capacity;
  for (int32_t i = 0; i < n; ++i) {
    const DevItem &d = hp.items[i];
    slack_work_item &w = items[i];
    w.stream = d.stream;
    w.head = d.head;
    w.q_row0 = d.q_row0;
    w.q_rows = d.q_rows;
    w.kv_tile_begin = d.kv_tile_begin;
    w.kv_tile_end = d.kv_tile_end;
    w.pos_lo = d.pos_lo;
    w.pos_hi = d.pos_hi;
    w.sink_tiles = d.sink_tiles;
    w.sink_pos_hi = d.sink_hi;
    w.partial_slot = d.partial_slot;
    w.cta = hp.item_cta[i];
    w.dual = d.dual;
  }
  return n;
}

/* ------------------------------------------------------------------------------------------------ append */
slack_status slack_kv_append_planned(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *k_new,
                                     const void *v_new, void *cuda_stream) {
  if (!ctx) return SLACK_EINVAL;
  ctx->last_launches = 0;
  if (!plan) return set_err(ctx, SLACK_EINVAL, "plan NULL");
  slack_status st = ensure_device(ctx);
  if (st != SLACK_OK) return st;
  if (plan->ctx != ctx) return set_err(ctx, SLACK_EINVAL, "plan belongs to another context");
  st = check_pool(ctx, pool, &plan->hp);
  if (st != SLACK_OK) return st;
  if (plan->hp.total_q == 0) return SLACK_OK;
  if (!k_new || !v_new || !aligned(k_new, 16) || !aligned(v_new, 16))
    return set_err(ctx, SLACK_EINVAL, "k_new / v_new NULL or not 16-byte aligned");
  const HostPlan &hp = plan->hp;
  cudaStream_t cs = reinterpret_cast<cudaStream_t>(cuda_stream);
  if ((st = plan_in_use(ctx, plan, cs)) != SLACK_OK) return st;
  cudaEvent_t ev_after;
  if ((st = prof_begin(ctx, 1, cs, &ev_after)) != SLACK_OK) return st;
  CUtensorMap tm_kn, tm_vn;
  if (hp.dtype == SLACK_FP8_E4M3) {
    if ((st = make_rows_map(ctx, &tm_kn, k_new, (uint64_t)hp.n_heads * hp.head_dim, (uint64_t)hp.total_q)) != SLACK_OK) return st;
    if ((st = make_rows_map(ctx, &tm_vn, v_new, (uint64_t)hp.n_heads * hp.head_dim, (uint64_t)hp.total_q)) != SLACK_OK) return st;
  }
  if (hp.dtype == SLACK_FP8_E4M3) // k_new / v_new are bf16: the append quantises (quant.cu)
    SLACK_CUDA(ctx, launch_kv_append_fp8(tm_kn, tm_vn, pool->k_pool, pool->v_pool, pool->k_scale, pool->v_scale, plan->d_streams,
                                         hp.n_streams, plan->max_q_len, plan->d_page_tables, hp.n_heads, hp.page_size, ctx->d_dbg, cs,
                                         &ctx->last_launches));
  else
    SLACK_CUDA(ctx, launch_kv_append(k_new, v_new, pool->k_pool, pool->v_pool, plan->d_streams, hp.n_streams, plan->max_q_len,
                                     plan->d_page_tables, hp.n_heads, hp.head_dim, hp.page_size, elem_bytes(hp.dtype),
                                     ctx->sm_count, cs, &ctx->last_launches));
  return prof_end(ctx, 1, cs, ev_after);
}

slack_status slack_kv_append(slack_ctx *ctx, const slack_pool *pool, int32_t n_streams, const slack_stream *streams,
                             const void *k_new, const void *v_new, void *cuda_stream) {
  if (!ctx) return SLACK_EINVAL;
  ctx->last_launches = 0;
  slack_status st = ensure_device(ctx);
  if (st != SLACK_OK) return st;
  st = check_pool(ctx, pool, nullptr);
  if (st != SLACK_OK) return st;
  // validation and table building are the planner's (force_simt: no work items are needed for an append)
  HostPlan hp;
  std::string err;
  slack_plan_opts o{};
  o.force_simt = pool->dtype != SLACK_FP8_E4M3;
  try {
    st = build_plan(*pool, n_streams, streams, o, ctx->sm_count, hp, err);
  } catch (const std::bad_alloc &) {
    return set_err(ctx, SLACK_ENOMEM, "out of host memory");
  }
  if (st != SLACK_OK) return set_err(ctx, st, err);
  if (hp.total_q == 0) return SLACK_OK;
  if (!k_new || !v_new || !aligned(k_new, 16) || !aligned(v_new, 16))
    return set_err(ctx, SLACK_EINVAL, "k_new / v_new NULL or not 16-byte aligned");
  const size_t b_streams = align_up(hp.streams.size() * sizeof(DevStream), 256);
  const size_t b_pt = align_up(hp.page_tables.size() * sizeof(int32_t), 256);
  const size_t total = b_streams + b_pt;
  cudaStream_t cs = reinterpret_cast<cudaStream_t>(cuda_stream);
  // descriptor tables: one arena block per call, filled through its pinned mirror, released by an event recorded
  // BEHIND the kernel that reads it (two appends on different streams never share a staging buffer)
  ArenaBlock blk;
  SLACK_CUDA(ctx, ctx->arena.alloc(total, &blk));
  uint8_t *h = ctx->arena.host(blk);
  uint8_t *d = ctx->arena.dev(blk);
  memcpy(h, hp.streams.data(), hp.streams.size() * sizeof(DevStream));
  memcpy(h + b_streams, hp.page_tables.data(), hp.page_tables.size() * sizeof(int32_t));
  int max_q = 0;
  for (const DevStream &s : hp.streams) max_q = s.q_len > max_q ? s.q_len : max_q;
  CUtensorMap tm_kn, tm_vn;
  if (hp.dtype == SLACK_FP8_E4M3) {
    slack_status ms = make_rows_map(ctx, &tm_kn, k_new, (uint64_t)hp.n_heads * hp.head_dim, (uint64_t)hp.total_q);
    if (ms == SLACK_OK) ms = make_rows_map(ctx, &tm_vn, v_new, (uint64_t)hp.n_heads * hp.head_dim, (uint64_t)hp.total_q);
    if (ms != SLACK_OK) {
      ctx->arena.free_now(blk);
      return ms;
    }
  }
  cudaError_t e = cudaMemcpyAsync(d, h, total, cudaMemcpyHostToDevice, cs);
  if (e == cudaSuccess && hp.dtype == SLACK_FP8_E4M3)
    e = launch_kv_append_fp8(tm_kn, tm_vn, pool->k_pool, pool->v_pool, pool->k_scale, pool->v_scale, reinterpret_cast<DevStream *>(d),
                             hp.n_streams, max_q, reinterpret_cast<int32_t *>(d + b_streams), hp.n_heads, hp.page_size, ctx->d_dbg, cs,
                             &ctx->last_launches);
  else if (e == cudaSuccess)
    e = launch_kv_append(k_new, v_new, pool->k_pool, pool->v_pool, reinterpret_cast<DevStream *>(d), hp.n_streams, max_q,
                         reinterpret_cast<int32_t *>(d + b_streams), hp.n_heads, hp.head_dim, hp.page_size,
                         elem_bytes(hp.dtype), ctx->sm_count, cs, &ctx->last_launches);
  cudaEvent_t done = nullptr;
  cudaError_t e2 = ctx->arena.get_event(&done);
  if (e2 == cudaSuccess) e2 = cudaEventRecord(done, cs);
  if (e2 != cudaSuccess) { // cannot guard the block: wait for the stream once, then free it
    cudaStreamSynchronize(cs);
    if (done) ctx->arena.put_event(done);
    ctx->arena.free_now(blk);
  } else {
    ctx->arena.release_after(blk, std::vector<cudaEvent_t>{done});
  }
  if (e != cudaSuccess) return cuda_err(ctx, e, "slack_kv_append");
  return SLACK_OK;
}

/* ------------------------------------------------------------------------------------------------ state-plane transfer */
slack_status slack_kv_transfer(slack_ctx *ctx, int32_t n_layers, const slack_pool *src_pools, const slack_pool *dst_pools,
                               int32_t n_pages, const int32_t *src_page_ids, const int32_t *dst_page_ids,
                               int32_t head_begin, int32_t head_end, void *cuda_stream, void *const *layer_done_events) {
  if (!ctx) return SLACK_EINVAL;
  ctx->last_launches = 0;
  slack_status st = ensure_device(ctx);
  if (st != SLACK_OK) return st;
  if (n_layers < 0 || n_pages < 0) return set_err(ctx, SLACK_EINVAL, "negative n_layers / n_pages");
  if (n_layers == 0 || n_pages == 0) return SLACK_OK;
  if (!src_pools || !dst_pools || !src_page_ids || !dst_page_ids) return set_err(ctx, SLACK_EINVAL, "NULL argument");
  const slack_pool &s0 = src_pools[0];
  const slack_pool &d0 = dst_pools[0];
  const bool fp8 = s0.dtype == SLACK_FP8_E4M3; // codes move like any other element type; the block scales move with them
  if (s0.n_heads <= 0 || s0.head_dim <= 0 || s0.page_size <= 0 || (s0.dtype != SLACK_BF16 && s0.dtype != SLACK_F32 && !fp8))
    return set_err(ctx, SLACK_EINVAL, "bad source pool shape / dtype");
  if (fp8 && s0.page_size % 128 != 0) return set_err(ctx, SLACK_EUNSUPPORTED, "FP8 pools need page_size >= 128");
  if (((size_t)s0.page_size * s0.head_dim * elem_bytes(s0.dtype)) % 16 != 0)
    return set_err(ctx, SLACK_EUNSUPPORTED, "a (page, head) slice must be a multiple of 16 bytes");
  if (head_begin < 0 || head_end > s0.n_heads || head_begin >= head_end)
    return set_err(ctx, SLACK_EINVAL, "head range must satisfy 0 <= head_begin < head_end <= n_heads");
  bool same_pool = false; // some layer copies inside one pool: a page may then not be both source and destination
  for (int32_t l = 0; l < n_layers; ++l) {
    const slack_pool &a = src_pools[l];
    const slack_pool &b = dst_pools[l];
    if ((st = check_pool(ctx, &a, nullptr)) != SLACK_OK || (st = check_pool(ctx, &b, nullptr)) != SLACK_OK) return st;
    if (a.n_heads != s0.n_heads || a.head_dim != s0.head_dim || a.page_size != s0.page_size || a.dtype != s0.dtype ||
        a.n_pages != s0.n_pages || b.n_heads != s0.n_heads || b.head_dim != s0.head_dim || b.page_size != s0.page_size ||
        b.dtype != s0.dtype || b.n_pages != d0.n_pages)
      return set_err(ctx, SLACK_EINVAL, "all layers' pools must share one shape per side, and both sides H, D, P and dtype");
    same_pool |= a.k_pool == b.k_pool || a.v_pool == b.v_pool || a.k_pool == b.v_pool || a.v_pool == b.k_pool;
  }
  {
    std::vector<uint8_t> seen((size_t)std::max(d0.n_pages, 0), 0);
    for (int32_t i = 0; i < n_pages; ++i) {
      if (src_page_ids[i] < 0 || src_page_ids[i] >= s0.n_pages) return set_err(ctx, SLACK_EINVAL, "source page id out of range");
      if (dst_page_ids[i] < 0 || dst_page_ids[i] >= d0.n_pages) return set_err(ctx, SLACK_EINVAL, "destination page id out of range");
      if (seen[dst_page_ids[i]]) return set_err(ctx, SLACK_EINVAL, "destination page listed twice");
      seen[dst_page_ids[i]] = 1;
    }
    if (same_pool)
      for (int32_t i = 0; i < n_pages; ++i)
        if (src_page_ids[i] < d0.n_pages && seen[src_page_ids[i]])
          return set_err(ctx, SLACK_EINVAL, "source and destination are the same pool and a page is both read and written");
  }
  cudaStream_t cs = reinterpret_cast<cudaStream_t>(cuda_stream);
  const size_t half = align_up((size_t)n_pages * sizeof(int32_t), 256);
  const size_t total = 2 * half;
  ArenaBlock blk; // id lists: released by an event behind the LAST layer's kernel
  SLACK_CUDA(ctx, ctx->arena.alloc(total, &blk));
  uint8_t *h = ctx->arena.host(blk);
  memcpy(h, src_page_ids, (size_t)n_pages * sizeof(int32_t));
  memcpy(h + half, dst_page_ids, (size_t)n_pages * sizeof(int32_t));
  const int32_t *d_src = reinterpret_cast<const int32_t *>(ctx->arena.dev(blk));
  const int32_t *d_dst = reinterpret_cast<const int32_t *>(ctx->arena.dev(blk) + half);
  cudaError_t e = cudaMemcpyAsync(ctx->arena.dev(blk), h, total, cudaMemcpyHostToDevice, cs);
  for (int32_t l = 0; l < n_layers && e == cudaSuccess; ++l) { // layer-major: layer l is complete when event l fires
    e = launch_kv_transfer(src_pools[l].k_pool, src_pools[l].v_pool, dst_pools[l].k_pool, dst_pools[l].v_pool, d_src, d_dst,
                           n_pages, s0.n_heads, s0.head_dim, s0.page_size, elem_bytes(s0.dtype), head_begin, head_end,
                           ctx->sm_count, cs, &ctx->last_launches);
    if (e == cudaSuccess && fp8)
      e = launch_kv_scale_transfer(src_pools[l].k_scale, src_pools[l].v_scale, dst_pools[l].k_scale, dst_pools[l].v_scale, d_src, d_dst,
                                   n_pages, s0.n_heads, s0.page_size, head_begin, head_end, cs, &ctx->last_launches);
    if (e == cudaSuccess && layer_done_events && layer_done_events[l])
      e = cudaEventRecord(reinterpret_cast<cudaEvent_t>(layer_done_events[l]), cs);
  }
  cudaEvent_t done = nullptr;
  cudaError_t e2 = ctx->arena.get_event(&done);
  if (e2 == cudaSuccess) e2 = cudaEventRecord(done, cs);
  if (e2 != cudaSuccess) {
    cudaStreamSynchronize(cs);
    if (done) ctx->arena.put_event(done);
    ctx->arena.free_now(blk);
  } else {
    ctx->arena.release_after(blk, std::vector<cudaEvent_t>{done});
  }
  if (e != cudaSuccess) return cuda_err(ctx, e, "slack_kv_transfer");
  return SLACK_OK;
}

/* ------------------------------------------------------------------------------------------------ attention */
} // extern "C"

namespace {
// A3 + A4, dense (block_mask == NULL) or block-sparse.
slack_status attention_impl(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *q, void *out,
                            float *lse, float scale, const uint32_t *block_mask, int32_t mask_words, void *workspace,
                            size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SLACK_EINVAL;
  ctx->last_launches = 0;
  if (!plan) return set_err(ctx, SLACK_EINVAL, "plan NULL");
  slack_status st = ensure_device(ctx);
  if (st != SLACK_OK) return st;
  if (plan->ctx != ctx) return set_err(ctx, SLACK_EINVAL, "plan belongs to another context");
  st = check_pool(ctx, pool, &plan->hp);
  if (st != SLACK_OK) return st;
  const HostPlan &hp = plan->hp;
  if (hp.total_q == 0) return SLACK_OK;
  if (!q || !out || !aligned(q, 16) || !aligned(out, 16)) return set_err(ctx, SLACK_EINVAL, "q / out NULL or not 16-byte aligned");
  if (!(scale > 0.f) || !(scale < 1e30f)) return set_err(ctx, SLACK_EINVAL, "scale must be a positive finite number");
  cudaStream_t cs = reinterpret_cast<cudaStream_t>(cuda_stream);
  const bool fp8 = hp.dtype == SLACK_FP8_E4M3;
  if (block_mask) {
    if (fp8) return set_err(ctx, SLACK_EUNSUPPORTED, "block-sparse attention over an FP8 pool is not built");
    if (!aligned(block_mask, 4)) return set_err(ctx, SLACK_EINVAL, "block_mask must be 4-byte aligned");
    if (mask_words < hp.mask_words_min) return set_err(ctx, SLACK_EINVAL, "mask_words smaller than slack_plan_mask_min_words()");
    if (hp.max_item_steps > 65535)
      return set_err(ctx, SLACK_EUNSUPPORTED, "block-sparse path: an item spans more than 65535 key tiles (8.3 M keys)");
  }

  if (hp.kernel_kind == 1) {
    if ((st = plan_in_use(ctx, plan, cs)) != SLACK_OK) return st;
    SLACK_CUDA(ctx, launch_attn_simt(hp.dtype, q, pool->k_pool, pool->v_pool, out, lse, plan->d_streams, hp.n_streams, hp.total_q,
                                     plan->d_page_tables, hp.n_heads, hp.head_dim, hp.page_size, scale, block_mask, mask_words,
                                     cs, &ctx->last_launches));
    return SLACK_OK;
  }

  const size_t ws_need = block_mask ? hp.sparse_total : hp.ws.total;
  if (ws_need > 0) {
    if (!workspace || workspace_bytes < ws_need)
      return set_err(ctx, SLACK_ENOMEM, block_mask ? "workspace NULL or smaller than slack_plan_sparse_workspace_bytes()"
                                                   : "workspace NULL or smaller than slack_plan_workspace_bytes()");
    if (!aligned(workspace, 16)) return set_err(ctx, SLACK_EINVAL, "workspace must be 16-byte aligned");
  }
  if (!aligned(q, 128) || !aligned(pool->k_pool, 128) || !aligned(pool->v_pool, 128))
    return set_err(ctx, SLACK_EINVAL, "tensor-core path: q and pool pointers must be 128-byte aligned (TMA)");
  if (!ctx->encode) return set_err(ctx, SLACK_ECUDA, "cuTensorMapEncodeTiled entry point not available");
  if (!ctx->tc_configured) {
    SLACK_CUDA(ctx, attn_tc_configure());
    SLACK_CUDA(ctx, attn_tc2_configure());
    ctx->tc_configured = true;
  }
  // pair plans run on CTA pairs (attn_tc2.cu); the block-sparse call walks the same items one CTA at a time
  const bool pairs = hp.kernel_kind == 2 && !block_mask;
  CUtensorMap tm_q, tm_k, tm_v;
  const uint64_t pool_rows = (uint64_t)hp.n_pages * hp.n_heads * hp.page_size;
  uint8_t *q8 = fp8 ? reinterpret_cast<uint8_t *>(workspace) + hp.q8_off : nullptr; // FP8: Q is quantised into the workspace first
  float *q8_scale = fp8 ? reinterpret_cast<float *>(reinterpret_cast<uint8_t *>(workspace) + hp.q8_scale_off) : nullptr;
  if ((st = make_map(ctx, &tm_q, fp8 ? (const void *)q8 : q, (uint64_t)hp.n_heads * hp.head_dim, (uint64_t)hp.total_q, 128, fp8)) != SLACK_OK) return st;
  if ((st = make_map(ctx, &tm_k, pool->k_pool, (uint64_t)hp.head_dim, pool_rows, pairs ? 64 : 128, fp8)) != SLACK_OK) return st;
  if ((st = make_map(ctx, &tm_v, pool->v_pool, (uint64_t)hp.head_dim, pool_rows, 128, fp8)) != SLACK_OK) return st;
  if ((st = plan_in_use(ctx, plan, cs)) != SLACK_OK) return st;
  if (fp8) SLACK_CUDA(ctx, launch_q_quant(q, q8, q8_scale, hp.total_q, hp.n_heads, cs, &ctx->last_launches));
  TcParams p{};
  p.items = plan->d_items;
  p.cta_begin = plan->d_cta_begin;
  p.page_tables = plan->d_page_tables;
  p.out = out;
  p.lse = lse;
  p.ws_o = reinterpret_cast<float *>(workspace);
  p.ws_lse = workspace ? reinterpret_cast<float *>(reinterpret_cast<uint8_t *>(workspace) + hp.ws.lse_off) : nullptr;
#ifdef SLACK_DIAGNOSTICS
  p.dbg_s = ctx->dbg_s;
  p.dbg_t = ctx->dbg_t;
#endif
  p.dbg_flag = ctx->d_dbg;
  p.n_heads = hp.n_heads;
  p.head_dim = hp.head_dim;
  int pl2 = 0;
  while ((1 << pl2) < hp.page_size) ++pl2;
  p.page_log2 = pl2;
  p.total_q = hp.total_q;
  p.has_dual = hp.has_dual ? 1 : 0;
  p.scale = scale;
  if (fp8) {
    p.k_scale = pool->k_scale;
    p.v_scale = pool->v_scale;
    p.q_scale = q8_scale;
  }
  if (block_mask) { // the mask may change with every call: list each item's selected key-tile steps first
    uint8_t *w8 = reinterpret_cast<uint8_t *>(workspace);
    uint16_t *steps = reinterpret_cast<uint16_t *>(w8 + hp.sparse_steps_off);
    int32_t *item_steps = reinterpret_cast<int32_t *>(w8 + hp.sparse_count_off);
    SLACK_CUDA(ctx, launch_sparse_steps(plan->d_items, (int)hp.items.size(), block_mask, hp.n_heads, mask_words, steps,
                                        item_steps, cs, &ctx->last_launches));
    p.steps = steps;
    p.item_steps = item_steps;
    p.dbg_t = nullptr; // the clock-trace instantiation is dense-only
  }
  cudaEvent_t ev_after;
  if ((st = prof_begin(ctx, 0, cs, &ev_after)) != SLACK_OK) return st;
  if (pairs)
    SLACK_CUDA(ctx, launch_attn_tc2(p, tm_q, tm_k, tm_v, 2 * hp.n_queues, cs, &ctx->last_launches));
  else
    SLACK_CUDA(ctx, launch_attn_tc(p, tm_q, tm_k, tm_v, hp.n_queues, cs, &ctx->last_launches));
  if ((st = prof_end(ctx, 0, cs, ev_after)) != SLACK_OK) return st;
  if (!hp.combines.empty()) {
    if ((st = prof_begin(ctx, 2, cs, &ev_after)) != SLACK_OK) return st;
    SLACK_CUDA(ctx, launch_combine(plan->d_combines, (int)hp.combines.size(), p.ws_o, p.ws_lse, out, lse, hp.n_heads, hp.head_dim,
                                   hp.total_q, cs, &ctx->last_launches));
    if ((st = prof_end(ctx, 2, cs, ev_after)) != SLACK_OK) return st;
  }
  return SLACK_OK;
}
} // namespace

extern "C" {

slack_status slack_chunk_attention(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *q, void *out,
                                   float *lse, float scale, void *workspace, size_t workspace_bytes, void *cuda_stream) {
  return attention_impl(ctx, plan, pool, q, out, lse, scale, nullptr, 0, workspace, workspace_bytes, cuda_stream);
}

slack_status slack_chunk_attention_sparse(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *q,
                                          void *out, float *lse, float scale, const uint32_t *block_mask, int32_t mask_words,
                                          void *workspace, size_t workspace_bytes, void *cuda_stream) {
  if (!ctx) return SLACK_EINVAL;
  if (!block_mask) return set_err(ctx, SLACK_EINVAL, "block_mask NULL (use slack_chunk_attention for dense attention)");
  return attention_impl(ctx, plan, pool, q, out, lse, scale, block_mask, mask_words, workspace, workspace_bytes, cuda_stream);
}

} // extern "C"

/* ------------------------------------------------------------------------------- attention without a caller workspace */
// slack_chunk_attention_static: the split-KV partials (and the FP8 path's quantised Q) live in ONE file-scope device array
// instead of a caller-provided workspace, for callers that may not allocate (CUDA graph capture, tight serving loops).
// Every GPU that loads libslack.so holds the array's SLACK_STATIC_WORKSPACE_BYTES until the process exits.
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[SLACK_STATIC_WORKSPACE_BYTES];

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress reports, looked up once per device with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_scratch_mu;
void *g_scratch_ptr[kMaxDevices] = {};

slack_status static_scratch(slack_ctx *ctx, void **ptr) {
  slack_status st = ensure_device(ctx); // makes ctx->device the current device
  if (st != SLACK_OK) return st;
  if (ctx->device >= kMaxDevices) return set_err(ctx, SLACK_EUNSUPPORTED, "static workspace: device ordinal >= 64");
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_ptr[ctx->device]) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess) return cuda_err(ctx, e, "cudaGetSymbolAddress(static workspace)");
    if (!p || !aligned(p, 256)) return set_err(ctx, SLACK_ECUDA, "static workspace: unexpected device address");
    g_scratch_ptr[ctx->device] = p;
  }
  *ptr = g_scratch_ptr[ctx->device];
  return SLACK_OK;
}

} // namespace

extern "C" {

slack_status slack_static_workspace_init(slack_ctx *ctx, size_t *max_bytes) {
  if (!ctx) return SLACK_EINVAL;
  if (max_bytes) *max_bytes = (size_t)SLACK_STATIC_WORKSPACE_BYTES;
  void *p = nullptr;
  return static_scratch(ctx, &p);
}

slack_status slack_chunk_attention_static(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *q,
                                          void *out, float *lse, float scale, void *cuda_stream) {
  if (!ctx) return SLACK_EINVAL;
  ctx->last_launches = 0;
  if (!plan) return set_err(ctx, SLACK_EINVAL, "plan NULL");
  const size_t need = plan->hp.ws.total;
  if (need > (size_t)SLACK_STATIC_WORKSPACE_BYTES) {
    char buf[256];
    snprintf(buf, sizeof buf,
             "slack_chunk_attention_static: the plan needs %zu bytes of workspace, the static workspace holds %zu "
             "(SLACK_STATIC_WORKSPACE_BYTES); use slack_chunk_attention with a caller-provided workspace",
             need, (size_t)SLACK_STATIC_WORKSPACE_BYTES);
    return set_err(ctx, SLACK_ENOMEM, buf);
  }
  void *ws = nullptr;
  slack_status st = static_scratch(ctx, &ws);
  if (st != SLACK_OK) return st;
  // the per-launch profiling of slack_profile_enable creates events on demand: not on this path
  const int prof_mask = ctx->prof_mask;
  ctx->prof_mask = 0;
  // nothing in the workspace has to start at zero: every byte the combine kernel (or the FP8 attention kernel) reads
  // was written earlier in this same call (partial outputs + lse of every planned piece; the quantised Q)
  st = attention_impl(ctx, plan, pool, q, out, lse, scale, nullptr, 0, ws, (size_t)SLACK_STATIC_WORKSPACE_BYTES, cuda_stream);
  ctx->prof_mask = prof_mask;
  return st;
}

} // extern "C"
