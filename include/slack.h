/* slack.h — C ABI of libslack: ragged, batched chunk attention over per-stream paged KV caches (B200, sm_100a).
 *
 * What the calls compute, and where that is defined
 * -------------------------------------------------
 * An AR-DiT generates a stream chunk by chunk; each chunk's tokens attend to the cached K/V of the stream's
 * earlier chunks and the finished chunk's K/V is appended to a rolling KV cache (§1, §2.1).
 * The cache is bounded by a rolling window over the most recent chunks (§2.1, knob (3) P:88, W in {1,3,7}
 * chunks P:568 App. A) and lives in a per-worker PAGED pool addressed through a logical page table
 * (§3.2, §4.4).  Several streams' caches are co-resident in one GPU's pool (§4.1).
 * Everything the paper leaves open (mask inside the chunk, what the window counts, pool layout, scale,
 * append-then-attend, co-batching) follows BASELINE.json north_star/configs as read in DESIGN.md "Readings".
 *
 * For stream s, head h, with Lq = q_len, Lc = cache_len, n = Lc + Lq, Wt = window:
 *     lo      = (Wt > 0) ? max(0, n - Wt) : 0
 *     visible = { t : lo <= t < n }                        (own chunk included; bidirectional inside the chunk)
 *     out_i   = sum_{t in visible} softmax_t(scale * <q_i, k_t>) * v_t        for every query row i of the chunk
 *     lse_i   = ln sum_{t in visible} exp(scale * <q_i, k_t>)
 *
 * Token -> slot rule (the single source of truth for "page-table indexing"):
 *     held token t of a stream sits at POSITION pos(t) = base + t (+ gap_slots if t >= sink_len; see slack_stream),
 *     i.e. at physical page  page_table[pos / page_size], slot pos % page_size, element offset
 *     ((page * n_heads + h) * page_size + slot) * head_dim + d of a pool tensor laid out
 *     [n_pages][n_heads][page_size][head_dim] (head_dim contiguous).
 *
 * Ownership: every device buffer (pools, q, k_new, v_new, out, lse, workspace) is CALLER-owned.  The library owns
 * only the context, plans and their small device-side tables, which live in a ctx-owned arena (device memory plus a
 * pinned host mirror, allocated once and grown rarely).  Host descriptor arrays (slack_stream, page tables) are read
 * during the call only.  All device work is enqueued on the caller's CUDA stream.  No call synchronises the device
 * except slack_destroy: slack_plan uploads its tables on a private stream and the first launch that uses the plan waits
 * for that copy ON THE DEVICE; slack_plan_destroy and the staging of slack_kv_append / slack_kv_transfer hand their
 * arena blocks back through CUDA events recorded behind the last kernel that reads them.  A CUDA stream a plan was
 * used on must outlive the plan.
 * Errors: every call returns a slack_status and never aborts, throws or prints; slack_last_error() gives a text.
 * Every in-kernel barrier wait is bounded: a wait that times out traps the launch, the next call reports SLACK_ECUDA
 * and its text names the block, thread and barrier that gave up.
 * A context is not thread-safe; plans are immutable after creation.
 * There is NO CPU fallback: without a CUDA device only host-only contexts (device = -1) exist, and they can plan
 * (for inspection) but every data-path call on them returns SLACK_ECUDA.
 */
#ifndef SLACK_H_
#define SLACK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SLACK_ABI_VERSION 3

typedef enum {
  SLACK_OK = 0,
  SLACK_EINVAL = 1,       /* malformed descriptors: negative lengths, base >= page_size, short page table, page id out of
                             range, a physical page owned twice in the batch, misaligned (<16 B) pointer, NULL argument */
  SLACK_EUNSUPPORTED = 2, /* valid but not built: head_dim not in {64,128}, page_size not a power of two >= 16; FP8 pools
                             with head_dim != 128, page_size < 128, force_simt or the block-sparse call */
  SLACK_ENOMEM = 3,       /* host or device allocation failed, or workspace_bytes too small */
  SLACK_ECUDA = 4,        /* a CUDA runtime/driver call failed, or the context has no device */
  SLACK_ESTALE_PLAN = 5   /* plan does not match the pool shape / dtype passed with it */
} slack_status;

/* SLACK_FP8_E4M3 is a POOL dtype only (PAPER.md P:88 knob (4) "quantization mode Q", Q in {FP16, FP8}
 * P:568; "online FP8 attention quantization ... without quantizing model weights").  Such a pool holds OCP e4m3 codes
 * (1 byte per element, same [n_pages][n_heads][page_size][head_dim] layout) plus one fp32 scale per (page, head, 128-slot
 * key block) for K and for V; q, k_new, v_new and out stay bf16.  Quantisation rule (reading A19; the oracle
 * states it in full): code = e4m3(x / scale), round to nearest even, saturating at +-448, both divisions in IEEE fp32;
 * scale = amax / 448 over the tokens the append writes into the block (all of head_dim; amax = 0 -> 1); an append SETS
 * a block's scale iff none of the stream's earlier tokens [0, cache_len) lies in that block, otherwise it keeps the
 * stored scale.  Inside the attention call Q is quantised per (row, head) and P per element (e4m3); accumulation fp32. */
typedef enum { SLACK_BF16 = 0, SLACK_F32 = 1, SLACK_FP8_E4M3 = 2 } slack_dtype;
#define SLACK_SCALE_BLOCK 128 /* slots per K/V scale of an FP8 pool = the key tile of slack_work_item */

typedef struct slack_ctx slack_ctx;   /* opaque */
typedef struct slack_plan_s slack_plan_t; /* opaque */

/* One layer's pool ("paged pool", "logical page table").  k_pool / v_pool: DEVICE pointers, each
 * [n_pages][n_heads][page_size][head_dim] of `dtype`, head_dim contiguous, 16-byte aligned (128-byte for bf16 with
 * head_dim 128: required by TMA).  slack_plan reads only the shape fields (pointers may be NULL there). */
typedef struct {
  void *k_pool;
  void *v_pool;
  int32_t n_pages, n_heads, head_dim, page_size;
  int32_t dtype;    /* slack_dtype */
  int32_t reserved; /* 0 */
  float *k_scale;   /* SLACK_FP8_E4M3 pools: DEVICE fp32 [n_pages][n_heads][page_size / 128], written by slack_kv_append, */
  float *v_scale;   /* read by slack_chunk_attention; NULL (ignored) for the other dtypes                                */
} slack_pool;

/* One stream of the batch; HOST memory. */
typedef struct {
  int32_t q_len;             /* Lq: tokens of the new chunk (0 = legal no-op)                                   */
  int32_t cache_len;         /* Lc: tokens of earlier chunks held for this stream                               */
  int32_t base;              /* slot of logical token 0 inside page_table[0]; 0 <= base < page_size             */
  int32_t window;            /* Wt: max visible keys INCLUDING the own chunk; 0 = unlimited              */
  int32_t sink_len;          /* "sink + local": the first sink_len tokens stay visible when the window has
                                moved past them: visible = [0, sink) U [max(sink, lo), n); 0 = no sink            */
  int32_t gap_slots;         /* unused slots between the end of the sink and the first held token behind it: token
                                t >= sink_len lives at position base + gap_slots + t (t < sink_len: base + t).  This is
                                how tokens that left the window are DROPPED from a sink stream ("keeps KV entries
                                only for the most recent W chunks"): they vanish from the numbering, cache_len counts
                                held tokens only, their whole pages leave the table, and the cache stays bounded
                                however long the stream runs.  0 = contiguous.  Needs sink_len > 0 and
                                cache_len >= sink_len when non-zero                                                */
  int32_t n_table_pages;     /* >= ceil((base + gap_slots + Lc + Lq) / page_size)                               */
  int32_t reserved;          /* 0                                                                                */
  const int32_t *page_table; /* HOST: logical page -> physical page id in [0, n_pages)                          */
} slack_stream;

/* Planner options; NULL = all defaults. */
typedef struct {
  int32_t sm_count;     /* CTAs the attention kernel is planned for; 0 = the device's SM count (148 on B200;
                           host-only contexts default to 148)                                                   */
  int32_t force_splits; /* 0 = automatic split-KV; k >= 1 = cut every (stream, head, q-tile) item's key range into
                           exactly min(k, #kv tiles) parts (1 = never split)                                     */
  int32_t force_simt;   /* 1 = plan for the fp32-accumulating SIMT validation kernel even where the tensor-core path
                           applies (debug / cross-check); f32 pools always use it                                */
  int32_t cta_pairs;    /* tensor-core path: 0 = automatic, 1 = one CTA per work item, 2 = CTA pairs (two SMs walk a
                           work item together, 128 query rows each, and share every K/V tile: tcgen05 cta_group::2;
                           the plan then has sm_count / 2 queues; needs an even sm_count; bf16 head_dim 128 only,
                           one CTA per item otherwise)                                                          */
} slack_plan_opts;

/* One unit of attention work as planned (inspection only; see slack_plan_get_items). Key tiles are 128 pool slots,
 * anchored to page slots: tile index T covers positions [128*T, 128*T+128) of the stream's position space
 * pos = base + t.  */
typedef struct {
  int32_t stream;        /* index into the batch                                                                 */
  int32_t head;
  int32_t q_row0;        /* first query row (global row of the ragged concat)                                    */
  int32_t q_rows;        /* valid rows, 1..256 (two 128-row MMA tiles)                                           */
  int32_t kv_tile_begin; /* [begin, end) in position-tile units                                                  */
  int32_t kv_tile_end;
  int32_t pos_lo;        /* visible positions [pos_lo, pos_hi) = [pos(lo), pos(n-1) + 1)                         */
  int32_t pos_hi;
  int32_t sink_tiles;    /* tiles of the sink [base, sink_pos_hi) visited BEFORE the window tiles (0: none; only the
                            first piece of a split row carries them), starting at tile base / 128                  */
  int32_t sink_pos_hi;   /* base + sink_len when the item visits sink tiles, else base                            */
  int32_t partial_slot;  /* -1: writes `out` directly; >= 0: writes workspace slot (split-KV), combined afterwards */
  int32_t cta;           /* queue that holds this item: CTA 0..sm_count-1, or CTA pair 0..sm_count/2-1 (pair plans) */
  int32_t dual;          /* 1: this item and the NEXT one of the same queue (both <= 128 rows, same number of key tiles)
                            are walked together by one CTA, one per query-tile slot (decode-like chunks, 72-row tails) */
} slack_work_item;

/* ---- context ------------------------------------------------------------------------------------------------ */
/* device >= 0: CUDA device ordinal.  device = -1: host-only context (planning/inspection, no CUDA call is made).  */
slack_status slack_create(slack_ctx **ctx, int device);
void slack_destroy(slack_ctx *ctx);
const char *slack_last_error(const slack_ctx *ctx); /* ctx-owned string, valid until the next call on ctx */
int32_t slack_abi_version(void);

/* ---- A1: KV append ("appended to a rolling KV cache") -------------------------------------------------- */
/* Copies k_new / v_new (DEVICE, ragged concat [sum Lq][n_heads][head_dim] in stream order, 16-byte aligned) into
 * the slots of logical tokens [Lc, Lc+Lq) of every stream.  Pure copy: bit-exact, touches no other byte.
 * Re-appending at the same position overwrites (a later denoising step of the same chunk).  Asynchronous on
 * `cuda_stream` (a cudaStream_t; NULL = default stream).  The descriptor tables are staged through a ctx-owned
 * pinned buffer; for the per-layer hot loop use slack_kv_append_planned, which re-uses the plan's device tables. */
slack_status slack_kv_append(slack_ctx *ctx, const slack_pool *pool, int32_t n_streams, const slack_stream *streams,
                             const void *k_new, const void *v_new, void *cuda_stream);
slack_status slack_kv_append_planned(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool,
                                     const void *k_new, const void *v_new, void *cuda_stream);

/* ---- A2: plan (host) ---------------------------------------------------------------------------------------- */
/* Validates the batch, cuts it into (stream, head, q-tile, kv-tile-range) work items, balances them over the SMs
 * (split-KV where a key range is cut), builds the combine list and uploads the tables (asynchronous, see "Ownership").
 * The plan depends only on the stream descriptors and (n_heads, head_dim, page_size, dtype): it is valid for every
 * layer and denoising step of the chunk batch (same page ids in every layer's pool).  slack_plan_destroy never blocks;
 * it may be called before or after slack_destroy of the plan's context. */
slack_status slack_plan(slack_ctx *ctx, const slack_pool *pool_shape, int32_t n_streams,
                        const slack_stream *streams, const slack_plan_opts *opts, slack_plan_t **plan);
void slack_plan_destroy(slack_plan_t *plan);
size_t slack_plan_workspace_bytes(const slack_plan_t *plan); /* device bytes slack_chunk_attention needs (may be 0) */
int32_t slack_plan_num_items(const slack_plan_t *plan);
int32_t slack_plan_num_partial_slots(const slack_plan_t *plan);
int32_t slack_plan_kernel_kind(const slack_plan_t *plan);    /* 0 = tcgen05 kernel, one CTA per item; 1 = SIMT kernel;
                                                                2 = tcgen05 kernel, CTA pairs.  The tcgen05 kernel
                                                                serves bf16 pools (head_dim 64 or 128) and FP8 pools
                                                                with page_size >= 128; the SIMT kernel the rest    */
/* Copies up to `capacity` planned items (in queue order) to `items`; returns how many were written. */
int32_t slack_plan_get_items(const slack_plan_t *plan, slack_work_item *items, int32_t capacity);

/* ---- A3 + A4: chunk attention and split-KV combine ------------------------------------------------------------ */
/* Precondition: the own chunk's K/V is already appended (pool holds logical tokens [0, Lc+Lq) of every stream).
 * q, out: DEVICE [sum Lq][n_heads][head_dim] of the pool dtype, bf16 for FP8 pools (16-byte aligned; 128-byte for the
 * tensor-core paths);
 * lse: optional DEVICE fp32 [n_heads][sum Lq] (natural log), may be NULL; workspace: DEVICE, >=
 * slack_plan_workspace_bytes(plan) bytes, 16-byte aligned, may be NULL when that is 0.  Asynchronous on cuda_stream. */
slack_status slack_chunk_attention(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *q,
                                   void *out, float *lse, float scale, void *workspace, size_t workspace_bytes,
                                   void *cuda_stream);

/* ---- A3 + A4 without a caller workspace ------------------------------------------------------------------------ */
/* For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): slack_chunk_attention with the workspace in a static device array inside the library instead of an
 * argument.  Same arguments, preconditions, kernels and results otherwise (dense attention; bit-identical output).
 * LIMIT: slack_plan_workspace_bytes(plan) <= SLACK_STATIC_WORKSPACE_BYTES (32 MiB: the automatic plans of BASELINE.json
 * configs[1]-[4] need 0-26 MB), else SLACK_ENOMEM with a message and nothing is launched.  Every GPU that loads the
 * library holds those 32 MiB until the process exits.  The call itself allocates and frees nothing (no cudaMalloc /
 * cudaFree, no event or stream creation; launches are not recorded by slack_profile_enable).
 * SHARING: every call on a device uses the same array, which keeps the previous call's contents; nothing in it has to be
 * cleared (each call writes every byte it later reads), but two calls that overlap on the GPU - different streams,
 * different contexts or threads, the same device - RACE on it: order them (one stream, or events).
 * slack_static_workspace_init resolves the array's device address for ctx's device (once per device; the attention call
 * does the same on first use) and reports the limit; call it at set-up, e.g. before a stream capture begins. */
#define SLACK_STATIC_WORKSPACE_BYTES (32u << 20)
slack_status slack_static_workspace_init(slack_ctx *ctx, size_t *max_bytes /* may be NULL */);
slack_status slack_chunk_attention_static(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *q,
                                          void *out, float *lse, float scale, void *cuda_stream);

/* ---- A3, block-sparse variant -------------------------------------------------------------- */
/* PAPER.md P:88 knob (2): "skips nonselected attention blocks with sparse masks", controlled by the attention sparsity
 * rho in {0, .6, .7, .8, .9}.  The block-SELECTION rule is Light Forcing's and not part of this path:
 * the mask is an input.  Semantics: query row i of a stream (chunk-local) belongs to query block i / 256; key token t
 * belongs to key block pos(t) / 128 (its position, see the token -> slot rule; the 128-position key tiles of slack_work_item); row i uses key t iff t is
 * visible (window / sink, as in slack_chunk_attention) AND its key block is selected for (query block, head).  A row
 * that is left without any key gets out = 0 and lse = -inf.
 * block_mask: DEVICE uint32 [slack_plan_mask_rows(plan)][n_heads][mask_words]; mask row r = the r-th 256-row query block
 * of the batch, counting ceil(Lq/256) blocks per stream in stream order; bit (kb % 32) of word kb / 32 = key block kb;
 * bits of blocks without a visible key are ignored; mask_words >= slack_plan_mask_min_words(plan).  The mask is read
 * when the call executes on `cuda_stream`, so it may be produced on the device and may differ in every layer and
 * denoising step while the plan stays valid.  workspace: >= slack_plan_sparse_workspace_bytes(plan) bytes (it holds the
 * split-KV partials and, per planned item, the list of its selected key tiles).  Other arguments as in
 * slack_chunk_attention.  f32 pools / force_simt plans evaluate the same definition on the SIMT kernel. */
#define SLACK_MASK_BLOCK_Q 256
#define SLACK_MASK_BLOCK_K 128
slack_status slack_chunk_attention_sparse(slack_ctx *ctx, const slack_plan_t *plan, const slack_pool *pool, const void *q,
                                          void *out, float *lse, float scale, const uint32_t *block_mask,
                                          int32_t mask_words, void *workspace, size_t workspace_bytes, void *cuda_stream);
size_t slack_plan_sparse_workspace_bytes(const slack_plan_t *plan);
int32_t slack_plan_mask_rows(const slack_plan_t *plan);      /* sum over streams of ceil(q_len / 256)                 */
int32_t slack_plan_mask_min_words(const slack_plan_t *plan); /* ceil(max over streams of ceil(end position / 128) / 32) */

/* ---- state-plane page transfer -------------------------------------------------------------- */
/* PAPER.md P:255 "transfer(stream, src, dst, page_range)": the single primitive behind credit-aware eviction,
 * re-homing and elastic SP; requests return immediately, run on a dedicated CUDA stream,
 * and are issued in LAYER-MAJOR order so the destination can start layer k once layer k's pages have arrived;
 * only the head partition assigned to the donor worker moves.
 * For each layer l = 0 .. n_layers-1, in order: page src_page_ids[i] of src_pools[l] is copied, bit for bit, into page
 * dst_page_ids[i] of dst_pools[l], heads [head_begin, head_end) only (in the [n_pages][H][P][D] layout a page's head
 * slice is one contiguous run); no other byte of the destination changes.  FP8 pools: the block scales of the moved
 * (page, head) slices are copied with the codes (a second small kernel per layer).  One kernel per layer on `cuda_stream`
 * (asynchronous: give it a side stream to overlap with compute); if layer_done_events is not NULL, entry l (a
 * cudaEvent_t, may be NULL) is recorded right after layer l's copy, which is what a consumer of layer l waits for.
 * src_pools / dst_pools: HOST arrays of n_layers descriptors; all layers of one side share n_pages, both sides share
 * n_heads, head_dim, page_size and dtype; the pool pointers are unified virtual addresses valid on this device: HBM of
 * this GPU, pinned (mapped) host memory for eviction / offload, or a peer GPU's HBM with peer access enabled.
 * src_page_ids / dst_page_ids: HOST int32[n_pages], read during the call; destination ids must be distinct.  The
 * caller's page tables are its own business: after the transfer the stream's table on the destination side is
 * dst_page_ids in the same logical order.  Errors: SLACK_EINVAL for ids out of range, duplicate destinations, mismatched
 * shapes, an empty head range, or - when a layer's source and destination are the same pool - a page that is both
 * read and written by the call (the copies of one launch are unordered). */
slack_status slack_kv_transfer(slack_ctx *ctx, int32_t n_layers, const slack_pool *src_pools, const slack_pool *dst_pools,
                               int32_t n_pages, const int32_t *src_page_ids, const int32_t *dst_page_ids,
                               int32_t head_begin, int32_t head_end, void *cuda_stream, void *const *layer_done_events);

/* Number of kernels the last slack_chunk_attention / slack_kv_append call on this ctx launched (bench bookkeeping). */
int32_t slack_last_launch_count(const slack_ctx *ctx);

/* ---- A0 + A5: page bookkeeping of one worker's pool (host only, integers only) -------------------------------- */
/* the K/V of all streams on a worker live in one paged pool "mapped to physical pages through a logical
 * page table, avoiding fragmentation"; every finished chunk is "appended to a rolling KV cache for subsequent
 * chunks"; the cache "preserves the first few chunks as a global sink and keeps KV entries only for the most
 * recent W chunks".  A slack_cache_t does exactly that bookkeeping for the page ids of ONE pool shape (the same ids
 * index every layer's pool): a free list, one page table per stream, the commit Lc += Lq, and the release of pages that
 * left the window.  It owns no device memory and makes no CUDA call.
 *
 *   slack_cache_open        new stream with its window Wt (tokens, 0 = unlimited) and sink length; no page yet
 *   slack_cache_begin_chunk A0: first drops what the window of the chunk about to be generated no longer covers
 *                           (lo = max(sink, Lc + q_len - Wt)): pages that hold no visible position go back to the free
 *                           list UNCLEARED, and the dropped tokens leave the numbering (cache_len, base or gap_slots
 *                           shrink accordingly; policy below); then takes pages from the free list until the table
 *                           covers [0, Lc + q_len); fills *desc, ready for slack_plan / slack_kv_append.
 *                           desc->page_table points into the cache and stays valid until the next call that names this
 *                           stream.  Calling it again before the commit with the same q_len returns the same descriptor
 *                           (the S denoising steps of a chunk re-append and re-attend with one descriptor).
 *                           SLACK_ENOMEM when the free list runs dry (nothing is taken in that case).
 *   slack_cache_commit      A5: the chunk is final: Lc += q_len.
 *   slack_cache_close       all pages of the stream go back to the free list.
 * trim_policy: SLACK_TRIM_PAGES drops whole pages only (the first held token is then the first slot of a page or the
 * stream's old start; `window` clips the rest inside the kernel); SLACK_TRIM_TOKENS also drops the invisible tokens at the
 * head of the first kept page (base, or gap_slots for a sink stream, walks through the page).  Both give identical
 * attention results.  Freed pages are handed out again most-recently-freed first. */
typedef struct slack_cache_s slack_cache_t; /* opaque */
typedef enum { SLACK_TRIM_PAGES = 0, SLACK_TRIM_TOKENS = 1 } slack_trim_policy;
slack_status slack_cache_create(int32_t n_pages, int32_t page_size, int32_t trim_policy, slack_cache_t **cache);
void slack_cache_destroy(slack_cache_t *cache);
slack_status slack_cache_open(slack_cache_t *cache, int32_t window, int32_t sink_len, int32_t *stream_id);
slack_status slack_cache_begin_chunk(slack_cache_t *cache, int32_t stream_id, int32_t q_len, slack_stream *desc);
slack_status slack_cache_commit(slack_cache_t *cache, int32_t stream_id);
slack_status slack_cache_close(slack_cache_t *cache, int32_t stream_id);
int32_t slack_cache_free_pages(const slack_cache_t *cache);
int32_t slack_cache_stream_pages(const slack_cache_t *cache, int32_t stream_id); /* pages the stream holds; -1: no such stream */
const char *slack_cache_last_error(const slack_cache_t *cache);

/* ---- measurement (bench.py's per-kernel figures) --------------------------------------------------- */
/* slack_profile_enable: `kinds` = OR of SLACK_PROF_*; while a kind is enabled every launch of that kernel is bracketed
 * by a CUDA event pair on the caller's stream.  slack_profile_read waits for the recorded pairs of one kind, copies up
 * to `capacity` per-launch durations (milliseconds, launch order) to `ms`, stores the number recorded in *n_launches and
 * resets that kind's record.  Measurement only: the events cost two stream operations per launch and switch off the
 * programmatic-dependent-launch overlap around the bracketed kernel. */
#define SLACK_PROF_ATTENTION 1 /* the attention kernel (not its combine)  */
#define SLACK_PROF_APPEND 2    /* the KV append kernel                    */
#define SLACK_PROF_COMBINE 4   /* the split-KV combine kernel             */
slack_status slack_profile_enable(slack_ctx *ctx, int32_t kinds);
slack_status slack_profile_read(slack_ctx *ctx, int32_t kind, double *ms, int32_t capacity, int32_t *n_launches);

#ifdef __cplusplus
}
#endif
#endif /* SLACK_H_ */
