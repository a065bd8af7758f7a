/*
 * segpa.h -- C ABI of the B200-native SegPagedAttention library (libsegpa.so).
 *
 * SegPagedAttention is the storage and execution substrate of RedKnot (arxiv 2606.06256,
 * PAPER.md:233-284, Sec. 4.3, Algorithm 2): the KV cache is decomposed per (layer, KV head) into
 * head segments stored in pages; a per-layer metadata pass selects, per KV head, the pages its
 * policy makes visible (GLOBAL: the full range; LOCAL: sink pages + recent-window pages),
 * translates them to physical pages and packs (h, B_h, |U_h|, p); then ONE fused variable-length
 * attention runs over all heads' page lists, with no dense [B,H,L,D] tensor and no mask.
 *
 * Conventions
 *   - Plain C, no exceptions cross this boundary; every call returns a segpa_status_t and applies
 *     nothing on error.  segpa_last_error() gives a human-readable reason.
 *   - "device" pointers are CUDA device pointers on the cache's device; "host" pointers are
 *     ordinary host memory, copied during the call (the caller may free them on return).
 *   - cuda_stream arguments are a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - bf16 = IEEE bfloat16 bit patterns (uint16_t).
 *   - A cache is not thread-safe; use one host thread per cache at a time.
 *   - There is no CPU fallback: on a box without a CUDA device, segpa_create_cache with
 *     device >= 0 fails with SEGPA_ERR_CUDA.  device == -1 creates a PLANNING-ONLY cache (host
 *     bookkeeping, builder and scheduler work; no device memory; append_pages accepts attach
 *     calls only; attention_fwd returns SEGPA_ERR_STATE).
 *
 * Terms
 *   stream   = (layer, kv_head, seq_id): the ordered tokens of ONE KV head of one request, of
 *              length kv_len.  It is the concatenation of the paper's head segments (l, h, s), each
 *              mapped to its own consecutive virtual pages by T_seg and to physical pages by T_page
 *              (PAPER.md:235); virtual page v of a stream is index v of its page table.  A stream
 *              written by COPY appends alone is ONE head segment: token j lives in page
 *              pt[j / page_size], slot j % page_size.  Every ATTACH adds a head segment that starts on
 *              a fresh page (so does the first COPY after one): a segment whose length is not a multiple
 *              of page_size leaves the rest of its last page unused in mid-stream ("ragged chunk
 *              tail"), and the page table holds sum ceil(n_s / page_size) pages.  Token indices,
 *              positions and windows never see those unused slots.
 *   segment  = execution segment: one (request, KV head) unit of a layer's attention call, i.e.
 *              one tuple (h, B_h, |U_h|, p) of the per-layer varlen metadata M_l,
 *              plus its query rows.
 */
#ifndef SEGPA_H_
#define SEGPA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SEGPA_VERSION 1

typedef enum {
    SEGPA_OK = 0,
    SEGPA_ERR_INVALID = 1,     /* bad argument; message says which */
    SEGPA_ERR_OOM = 2,         /* page pool or device/host memory exhausted */
    SEGPA_ERR_CUDA = 3,        /* a CUDA call failed (also: no device) */
    SEGPA_ERR_UNSUPPORTED = 4, /* shape outside what the kernels are built for */
    SEGPA_ERR_STATE = 5        /* call not valid in this state (e.g. fwd on a planning-only cache) */
} segpa_status_t;

typedef enum { SEGPA_GLOBAL = 0, SEGPA_LOCAL = 1 } segpa_head_class_t;

typedef struct segpa_cache segpa_cache_t;       /* opaque */
typedef struct segpa_segments segpa_segments_t; /* opaque; owned by the cache that built it */

/* ------------------------------------------------------------------------------------------- */
/* Per-head paged KV pool ("head-segmented KV layout"; "allocates     */
/* pages per head, so local heads occupy only their short windows").                            */
/* ------------------------------------------------------------------------------------------- */

typedef struct {
    int32_t num_layers;   /* >= 1 */
    int32_t num_q_heads;  /* Hq; multiple of num_kv_heads; G = Hq / Hkv <= 16 */
    int32_t num_kv_heads; /* Hkv */
    int32_t head_dim;     /* D: 64 or 128 */
    int32_t page_size;    /* P tokens per page: 16 or 32 */
    int32_t device;       /* CUDA device ordinal, or -1 = planning-only cache */
    int64_t num_pages;    /* pool capacity in pages; one page holds P tokens of ONE KV head */
    void *k_pool;         /* optional caller-owned device memory of segpa_pool_bytes() bytes, */
    void *v_pool;         /*   else NULL (library allocates). Contents are library-private.     */
    int32_t tiles_per_item; /* 128-row query tiles a work item of the attention kernel holds: 0 = default (2:
                               two tiles share every K/V stage), or 1 / 2.  A tuning knob of the one kernel,
                               fixed for the cache's lifetime; results do not depend on it beyond rounding order. */
    int32_t reserved;     /* 0 */
} segpa_cache_desc_t;

/* Bytes needed for each of k_pool / v_pool when the caller owns them ((num_pages + 1) pages: the
 * extra page is the library's always-zero page). */
int64_t segpa_pool_bytes(const segpa_cache_desc_t *desc);

/*
 * Create a cache.  The pool is zero-filled.  Physical page layout is private to the library
 * (a page is stored as the shared-memory image the attention kernel consumes, so that one bulk
 * copy moves a page).
 * Errors: INVALID (null, counts < 1, Hq % Hkv != 0, tiles_per_item not in 0..2), UNSUPPORTED (head_dim, page_size, G > 16,
 * device is not compute capability 10.x), CUDA, OOM.
 */
segpa_status_t segpa_create_cache(const segpa_cache_desc_t *desc, segpa_cache_t **out);

/*
 * Extend the stream (layer, kv_head, seq_id) by n_tokens tokens (creating it if absent).
 *
 *  - COPY mode (k_src and v_src non-NULL): device bf16 rows; row t of the new tokens is at
 *    k_src + t * src_row_stride_elems (D contiguous elements).  Rows are scattered into the
 *    stream's pages by a kernel on cuda_stream.  If the stream's last page is partial, was started
 *    by a COPY append of this stream and is referenced by no other stream, the new tokens first fill
 *    it; otherwise (the last head segment was attached, or another stream has attached that page)
 *    they start a new head segment on a fresh page and the partial page keeps its unused slots.
 *    Further pages are taken from page_ids (host int32, in order, n_page_ids of them = the number
 *    of pages the new tokens start, each must be free) or, if page_ids == NULL, from the allocator.
 *    Slots of a newly started page beyond the stream's end are zero-filled (masked probabilities
 *    multiply them, so they must stay finite).
 *  - ATTACH mode (k_src == v_src == NULL, page_ids non-NULL): the pages already hold the data
 *    (filled earlier through another stream); they are appended to this stream's page table
 *    without copying and their reference count is incremented.  This is both PIC chunk splicing
 *    ("directly reusing the prefix-robust local segments") and shared-prefix
 *    aliasing.  The attached tokens are a head segment of their own: they start on a fresh page
 *    whatever the stream's current length, n_tokens may be any length >= 1 (a reused chunk need not
 *    be a multiple of page_size; only the first n_tokens slots of the pages belong to the stream) and
 *    n_page_ids == ceil(n_tokens / page_size).  On a planning-only cache pages may be attached
 *    without ever having been filled.
 *
 * Errors: INVALID (indices out of range, n_tokens < 1, page id out of range / not free in COPY
 * mode / not in use in ATTACH mode on a device cache, wrong n_page_ids, one of k_src / v_src NULL),
 * OOM (no free page), STATE (COPY on a planning-only cache), CUDA.
 */
segpa_status_t segpa_append_pages(segpa_cache_t *cache, int32_t layer, int32_t kv_head,
                                  int64_t seq_id, const void *k_src, const void *v_src,
                                  int64_t src_row_stride_elems, int64_t n_tokens,
                                  const int32_t *page_ids, int32_t n_page_ids, void *cuda_stream);

/*
 * Batched form of segpa_append_pages: the n requests are applied in order (a later request may
 * attach pages an earlier one of the same batch fills, or extend the same stream) with ONE
 * descriptor upload and ONE scatter-kernel launch on cuda_stream for all COPY-mode requests.
 * This is how a layer's batch of new K/V rows is stored (a1 of the hot path).  All-or-nothing: on
 * error no stream, page table or reference count has changed.  Field meaning and errors are those
 * of segpa_append_pages; the message names the failing request index.
 */
typedef struct {
    int32_t layer;
    int32_t kv_head;
    int64_t seq_id;
    const void *k_src;            /* bf16 rows (device, or host if src_is_host), or NULL (with v_src NULL) = ATTACH */
    const void *v_src;
    int64_t src_row_stride_elems;
    int64_t n_tokens;
    const int32_t *page_ids;      /* host; NULL = allocator chooses (COPY mode only) */
    int32_t n_page_ids;
    int32_t src_is_host;          /* 0: k_src / v_src are device pointers.  1: HOST pointers (pinned memory for the
                                     copies to be asynchronous; any 2-byte alignment and row stride >= D): the rows
                                     are copied to a staging buffer owned by the cache on cuda_stream, ahead of the
                                     scatter launch; the host buffers must stay valid until that work completes. */
} segpa_append_req_t;

segpa_status_t segpa_append_pages_batch(segpa_cache_t *cache, const segpa_append_req_t *reqs, int32_t n,
                                        void *cuda_stream);

/*
 * True eviction ("true eviction ... rather than zero-filling"): remove pages
 * [first_page_index, first_page_index + n_pages) from a stream's page table.  Their reference counts
 * are decremented (pages reaching zero return to the free list) and the entries become holes
 * (reported as -1 by segpa_stream_info); the stream keeps its length.  This is how the middle of a
 * LOCAL head's stream (between the sink tokens and the recent window) is dropped.  A later
 * segpa_build_segments whose visible set (sink pages + window pages) touches a hole fails with
 * INVALID; holes outside it are never read.
 * Errors: INVALID (no such stream, range outside the page table, a page already evicted; the stream's
 * partial last page cannot be evicted).
 */
segpa_status_t segpa_evict_pages(segpa_cache_t *cache, int32_t layer, int32_t kv_head, int64_t seq_id,
                                 int32_t first_page_index, int32_t n_pages);

/*
 * RoPE-based positional alignment of reused keys (Alg. 1 line 1 "RoPEAlign"):
 *     K(p_on) = R(p_on) R(p_off)^-1 K(p_off) = R(delta_pos) K(p_off),   delta_pos = p_on - p_off,
 * applied IN PLACE to the K rows of tokens [first_token, first_token + n_tokens) of a stream (a reused
 * chunk moves as a unit, so one delta per call).  R(p) is the RoPE rotation: for pair index d in
 * [0, D/2) the elements (d, d + D/2) of a key (the "rotate-half" pairing of the Llama / Qwen / Mistral
 * families the paper evaluates; reading A20) are rotated by the angle p * rope_base^(-2d/D).
 * The per-pair cos / sin are formed in double precision (on the device), the rotation runs in fp32 and
 * the result is rounded to bf16 (RNE).  V is untouched.  Asynchronous on cuda_stream.
 * Errors: INVALID (no such stream, range outside it, rope_base <= 1, a page of the range is shared
 * with another stream (refcount > 1: rotating it would move the other stream's keys too) or evicted),
 * STATE (planning-only cache), CUDA.
 */
segpa_status_t segpa_rope_align(segpa_cache_t *cache, int32_t layer, int32_t kv_head, int64_t seq_id,
                                int64_t first_token, int64_t n_tokens, int64_t delta_pos, double rope_base,
                                void *cuda_stream);

/* Batched form: every reused chunk of a batch (each with its own stream, token range and delta) in ONE
 * descriptor upload and ONE kernel launch.  Ranges must not overlap.  All-or-nothing validation. */
typedef struct {
    int32_t layer;
    int32_t kv_head;
    int64_t seq_id;
    int64_t first_token;
    int64_t n_tokens;
    int64_t delta_pos;
} segpa_rope_req_t;

segpa_status_t segpa_rope_align_batch(segpa_cache_t *cache, const segpa_rope_req_t *reqs, int32_t n,
                                      double rope_base, void *cuda_stream);

/*
 * Copy the K and V rows of tokens [first_token, first_token + n_tokens) of a stream out of the paged pool
 * into device bf16 buffers [n_tokens][D] (row stride given; either destination may be NULL).  The inverse of
 * COPY-mode append: export of a head's KV (e.g. for transfer to another worker) and test read-back.
 * Errors: INVALID (no such stream, range outside it or touching an evicted page, bad stride), STATE, CUDA.
 */
segpa_status_t segpa_gather_rows(segpa_cache_t *cache, int32_t layer, int32_t kv_head, int64_t seq_id,
                                 int64_t first_token, int64_t n_tokens, void *k_dst, void *v_dst,
                                 int64_t dst_row_stride_elems, void *cuda_stream);

/*
 * segpa_gather_rows for callers that may not allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same arguments, same result bit for bit, and the call makes NO cudaMalloc /
 * cudaFree / allocating library call.  Its scratch -- the device copy of the page ids the token range covers, which
 * segpa_gather_rows keeps in a staging buffer that grows on demand -- is a fixed array of SEGPA_NOALLOC_MAX_PAGES
 * int32 entries (64 KB) inside the library image, held by every GPU that loads the library until the process exits.
 * Limit: the range [first_token, first_token + n_tokens) may cover at most SEGPA_NOALLOC_MAX_PAGES pages of the stream
 * (262144 tokens at page_size 16); a longer range is refused with SEGPA_ERR_INVALID and a message that says so (split it,
 * or use segpa_gather_rows).  All calls share the one array, which keeps the last call's ids: each call overwrites the
 * entries it uses in stream order (nothing needs clearing), so calls on ONE stream may follow each other freely, but
 * two calls that can overlap on the GPU (different streams with no dependency between them) race on it.
 * Other errors: as segpa_gather_rows.
 */
#define SEGPA_NOALLOC_MAX_PAGES 16384
segpa_status_t segpa_gather_rows_noalloc(segpa_cache_t *cache, int32_t layer, int32_t kv_head, int64_t seq_id,
                                         int64_t first_token, int64_t n_tokens, void *k_dst, void *v_dst,
                                         int64_t dst_row_stride_elems, void *cuda_stream);

/* Drop every stream of the cache (all pages return to the free list).  Segment objects built
 * earlier keep their translated page lists and must not be used afterwards. */
segpa_status_t segpa_clear_streams(segpa_cache_t *cache);

/* Drop a stream: its pages' reference counts are decremented; pages reaching zero return to the
 * free list.  Errors: INVALID (no such stream). */
segpa_status_t segpa_free_stream(segpa_cache_t *cache, int32_t layer, int32_t kv_head,
                                 int64_t seq_id);

/* Query a stream.  kv_len / n_pages may be NULL.  If page_ids_out != NULL, up to cap ids are
 * written.  Errors: INVALID (no such stream). */
segpa_status_t segpa_stream_info(const segpa_cache_t *cache, int32_t layer, int32_t kv_head,
                                 int64_t seq_id, int64_t *kv_len, int32_t *n_pages,
                                 int32_t *page_ids_out, int32_t cap);

/* Pool occupancy: pages in use (refcount > 0) and free. Either pointer may be NULL. */
segpa_status_t segpa_pool_stats(const segpa_cache_t *cache, int64_t *pages_in_use,
                                int64_t *pages_free);

/* ------------------------------------------------------------------------------------------- */
/* Segment descriptor builder + tile scheduler (Alg. 2 lines 1-14).           */
/* ------------------------------------------------------------------------------------------- */

typedef struct {
    int64_t seq_id;      /* request; the stream is (layer, kv_head, seq_id) */
    int32_t kv_head;     /* h */
    int32_t head_class;  /* p = P(l, h): SEGPA_GLOBAL or SEGPA_LOCAL */
    int32_t window;      /* LOCAL: W = number of visible keys INCLUDING the query's own position
                            (paper's w = W - 1; reading A1). >= 1.
                            Ignored for GLOBAL. */
    int32_t n_sink;      /* LOCAL: the first n_sink tokens stay visible besides the window (S_sink,
                            PAPER.md:219); >= 0.  Ignored for GLOBAL. */
    int64_t q_row_start; /* first row of this segment's queries in q / out */
    int32_t q_len;       /* 1 <= q_len <= kv_len; query t has position kv_len - q_len + t
                            (bottom-right aligned, the flash_attn_varlen convention) */
    int32_t reserved;    /* 0 */
} segpa_segment_req_t;

/*
 * Build one layer's metadata M_l and the tile schedule for n segments.
 *
 * Per segment: visible positions are [0, kv_len) for GLOBAL and
 * [0, n_sink) U [max(0, kv_len - q_len - W + 1), kv_len) for LOCAL (Alg. 2 lines 6-10: sink pages +
 * recent pages; a work item of a segment with sinks visits two KV block ranges); the pages covering
 * them are translated to physical ids (line 12); pages outside the visible range are replaced by
 * the always-zero page, so evicted pages are never read ("true eviction").  Query
 * rows are cut into tiles of floor(128 / G) tokens x G query heads (GQA packing: the G heads of a
 * KV head share every K/V page load); each tile gets exactly the KV block range it attends to,
 * so no work is issued for fully masked blocks.  Long tiles are split along KV when the grid
 * would otherwise be unbalanced; work items are then assigned longest-first to the least-loaded CTA of
 * the persistent grid (LPT), each CTA running its items in descending cost order.
 * The descriptors are uploaded with one async copy per array on cuda_stream.
 *
 * Queries of segment (seq_id, kv_head) are rows q_row_start .. q_row_start + q_len - 1, heads
 * kv_head*G .. kv_head*G + G - 1 (contiguous GQA groups).  (row, head) pairs not covered by any
 * segment are never written by attention_fwd.
 *
 * Errors: INVALID (n < 1, unknown stream, q_len < 1 or > kv_len, LOCAL with window < 1, bad
 * class, negative q_row_start or n_sink, two segments overlapping on (row, head), a visible page that was
 * evicted), OOM, CUDA.
 */
segpa_status_t segpa_build_segments(segpa_cache_t *cache, int32_t layer,
                                    const segpa_segment_req_t *reqs, int32_t n,
                                    segpa_segments_t **out, void *cuda_stream);

/* Release a segments object.  Does not synchronise the device: its buffers are recycled by later
 * build_segments calls only after the work that last used them (upload, attention_fwd) has
 * completed (tracked with an event on the stream it was last used on). */
segpa_status_t segpa_free_segments(segpa_cache_t *cache, segpa_segments_t *segs);

typedef struct {
    int32_t n_segments;
    int32_t n_tiles;          /* (segment, token-range) tiles of <= 128 rows */
    int32_t n_items;          /* work items after KV splitting */
    int32_t n_split_tiles;    /* tiles cut into more than one item */
    int32_t tile_tokens;      /* floor(128 / G) */
    int32_t block_keys;       /* 128 */
    int64_t kv_blocks;        /* sum over items of visited 128-key blocks */
    int64_t attended_pairs;   /* (query, key, q head) triples actually attended */
    int64_t q_rows;           /* max(q_row_start + q_len) */
    int64_t visible_kv_tokens;/* sum over segments of tokens in visible pages (algorithmic K/V reads) */
    int64_t workspace_bytes;  /* split-KV partials */
} segpa_plan_stats_t;

segpa_status_t segpa_segments_stats(const segpa_segments_t *segs, segpa_plan_stats_t *out);

typedef struct {
    int32_t segment;   /* index into reqs */
    int32_t t0;        /* first token of the tile within the segment's q range */
    int32_t n_tok;     /* tokens in the tile (rows = n_tok * G) */
    int32_t kb_lo;     /* first visited 128-key block */
    int32_t kb_hi;     /* one past the last visited block */
    int32_t split;     /* -1: writes the output directly; >= 0: index of this item's partial */
    int32_t n_splits;  /* number of items this tile was cut into */
    int32_t tile;      /* tile id (items of one tile share it) */
    int32_t cta;       /* CTA of the persistent grid the item is assigned to */
    int32_t reserved;
} segpa_item_t;

/* Copy up to cap work items (in schedule order: CTA by CTA, each CTA's items by descending cost) to
 * host memory; *n_out = total count. */
segpa_status_t segpa_segments_items(const segpa_segments_t *segs, segpa_item_t *items_out,
                                    int32_t cap, int32_t *n_out);

/* Per-segment translated page list as uploaded (length *n_out; zero page = num_pages). */
segpa_status_t segpa_segments_pages(const segpa_segments_t *segs, int32_t segment,
                                    int32_t *first_page_index, int32_t *page_ids_out, int32_t cap,
                                    int32_t *n_out);

/* ------------------------------------------------------------------------------------------- */
/* Fused attention (Alg. 2 lines 15-16).                                      */
/* ------------------------------------------------------------------------------------------- */

/*
 * out[row][head][:] = softmax_j( softmax_scale * q[row][head] . K[j] ) V[j]  over the visible keys
 * of the covering segment; lse[head][row] = ln sum_j exp(softmax_scale * q . K[j]) (natural log of
 * the scaled scores).  bf16 x bf16 products accumulate in fp32 on the tensor cores; softmax runs
 * in fp32; probabilities are rounded to bf16 before the PV product; out is rounded to bf16 (RNE).
 * MergeHeads (Alg. 2 line 16) is the output layout itself.
 *
 *   q, out : device bf16, row r / head h / element d at  base + r*row_stride + h*D + d
 *   lse    : device fp32 [Hq][lse_stride], lse_stride >= T; may be NULL
 *   T      : number of rows in q / out (>= the plan's q_rows)
 *
 * Asynchronous on cuda_stream; deterministic (no floating-point atomics; split-KV partials are
 * merged in a fixed order).  Errors: INVALID, STATE (planning-only cache, or segments built by
 * another cache), CUDA (also reports an earlier asynchronous failure).
 */
segpa_status_t segpa_attention_fwd(segpa_cache_t *cache, const segpa_segments_t *segs,
                                   const void *q, int64_t q_row_stride_elems, float softmax_scale,
                                   void *out, int64_t out_row_stride_elems, float *lse,
                                   int64_t lse_stride, int64_t T, void *cuda_stream);

/*
 * Same computation with HOST buffers (pinned memory for the copies to be asynchronous): q/out are dense
 * [T][Hq][D] bf16, lse [Hq][T] fp32 (may be NULL).  The plan is cut into chunks of consecutive query rows (about
 * 16 MB of q each; 32 MB when the first call on the segments object is the _async one); the host->device copy of chunk k+1, the kernels of chunk k (on cuda_stream) and the device->host
 * copy of chunk k-1 run concurrently on three streams, so the call is bounded by the larger PCIe direction, not by
 * the sum.  Results are bit-identical to segpa_attention_fwd on the same plan.  Differences from the device entry
 * point: the call returns after the last copy back has completed (synchronous), and (row, head) pairs that no segment
 * covers are written as zeros (out and lse) rather than left untouched.  Staging buffers are owned by the cache and
 * reused.  This is the end-to-end path bench.py times.  Errors: as segpa_attention_fwd, plus OOM (staging).
 */
segpa_status_t segpa_attention_fwd_host(segpa_cache_t *cache, const segpa_segments_t *segs,
                                        const void *q_host, float softmax_scale, void *out_host,
                                        float *lse_host, int64_t T, void *cuda_stream);

/*
 * segpa_attention_fwd_host without the wait at the end: the call returns once everything is enqueued, and out_host /
 * lse_host are complete only after segpa_host_wait(cache) (or after a later synchronous segpa_attention_fwd_host on
 * the cache has returned).  Consecutive calls (the layers of a step) then overlap: the cache holds two sets of staging
 * buffers, so the q rows of call k+1 go up while the kernels and the copies back of call k still run, and the link is
 * busy in both directions across layer boundaries.  At most two calls are in flight; a third waits (on the device) for
 * the first to finish.  q_host must stay valid and out_host / lse_host untouched until the wait.  Same results, bit for
 * bit, same errors.  segpa_host_wait: blocks the host until every asynchronous call on the cache has completed;
 * Errors: INVALID (null), CUDA.
 */
segpa_status_t segpa_attention_fwd_host_async(segpa_cache_t *cache, const segpa_segments_t *segs,
                                              const void *q_host, float softmax_scale, void *out_host,
                                              float *lse_host, int64_t T, void *cuda_stream);
segpa_status_t segpa_host_wait(segpa_cache_t *cache);

/*
 * LSE merge ("splitting the key set ... and merging them with LSE gives the same result as
 * softmax over their union"): (out_a, lse_a) and (out_b, lse_b) are attention results of the SAME queries over
 * two DISJOINT key sets (e.g. an offline-cached part and an online part); writes the result over the union:
 *     lse = ln(e^lse_a + e^lse_b),   out = (e^lse_a out_a + e^lse_b out_b) / (e^lse_a + e^lse_b).
 * Layouts as in segpa_attention_fwd (out_*: device bf16 [T][Hq][D] with one common row stride, a multiple of 8
 * elements, 16-byte aligned; lse_*: device fp32 [Hq][lse_stride]).  A (row, head) whose lse is -inf on one side takes the other side's result; out / lse
 * may alias out_a / lse_a.  Asynchronous on cuda_stream.  Errors: INVALID, STATE (planning-only cache), CUDA.
 */
segpa_status_t segpa_merge(segpa_cache_t *cache, const void *out_a, const float *lse_a, const void *out_b,
                           const float *lse_b, void *out, float *lse, int64_t row_stride_elems,
                           int64_t lse_stride, int64_t T, void *cuda_stream);

/* ------------------------------------------------------------------------------------------- */
/* Attention mass and salient-token selection (Alg. 1 line 19 SelectImportantTokens; */
/* "computes attention mass over tokens and selects ... the smallest set of tokens whose cumulative */
/* attention mass exceeds a threshold tau").  The step right after the fused attention. */
/* ------------------------------------------------------------------------------------------- */

/* Layout of the mass / selection arrays: segment s occupies entries [offsets[s], offsets[s] + kv_len_s)
 * (offsets[s+1] - offsets[s] = kv_len_s rounded up to 128).  Writes min(cap, n + 1) offsets; *n_out = n. */
segpa_status_t segpa_segments_mass_layout(const segpa_segments_t *segs, int64_t *offsets_out, int32_t cap,
                                          int32_t *n_out);

/*
 * mass[offsets[s] + j] = sum over the query rows t and the G query heads g of segment s of p(t, g, j), where
 * p(t, g, j) = exp(softmax_scale * q . K[j] - lse[g][t]) is the probability the fused attention gave key j
 * (0 for keys the row does not see).  q, softmax_scale and lse are those of a completed segpa_attention_fwd
 * with the same segments; the probabilities are recomputed on the tensor cores (S^T = K Q^T per 128-key block),
 * they are never stored.  Entries of keys no query sees, and the padding up to the next multiple of 128, are 0.
 * mass: device fp32 with at least offsets[n] entries.  Asynchronous on cuda_stream; deterministic.
 * Errors: INVALID, STATE (planning-only cache, foreign or stale segments), UNSUPPORTED (a segment's stream has
 * ragged chunk tails: the mass kernel works on single-segment streams), OOM, CUDA.
 */
segpa_status_t segpa_attention_mass(segpa_cache_t *cache, const segpa_segments_t *segs, const void *q,
                                    int64_t q_row_stride_elems, float softmax_scale, const float *lse,
                                    int64_t lse_stride, int64_t T, float *mass, int64_t mass_len,
                                    void *cuda_stream);

/*
 * Per segment, the smallest set of keys whose cumulative mass reaches tau * (the segment's total mass):
 * selected[offsets[s] + j] = 1 / 0 (device uint8, same layout as mass), n_selected[s] = its size (device int32
 * [n_segments]).  Keys are taken in order of decreasing mass; among keys of equal mass at the boundary the
 * lowest positions are taken.  0 < tau <= 1.  Errors: INVALID, STATE, CUDA.
 */
segpa_status_t segpa_mass_select(segpa_cache_t *cache, const segpa_segments_t *segs, const float *mass, float tau,
                                 uint8_t *selected, int32_t *n_selected, void *cuda_stream);

/* Number of kernel launches the last attention_fwd on this cache issued (1, or 2 with split-KV). */
int32_t segpa_last_launch_count(const segpa_cache_t *cache);

/* ------------------------------------------------------------------------------------------- */

/* Frees the pool (unless caller-owned), all streams and all segment objects. NULL is OK. */
segpa_status_t segpa_destroy(segpa_cache_t *cache);

/* Message for the most recent error on this thread (never NULL). */
const char *segpa_last_error(void);

int32_t segpa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SEGPA_H_ */
