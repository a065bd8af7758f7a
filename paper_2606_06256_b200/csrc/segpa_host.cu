// Host runtime of libsegpa.so: per-head paged KV pool, page tables, segment descriptor builder,
// tile scheduler and the extern "C" entry points declared in include/segpa.h.
// Operation semantics follow PAPER.md Sec. 4.3 / Algorithm 2; see DESIGN.md.
#include "../../include/segpa.h"
#include "segpa_internal.h"

#include <cuda.h>   // CUtensorMap types only; the encoder is fetched with cudaGetDriverEntryPoint (no -lcuda)

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <queue>
#include <string>
#include <unordered_map>
#include <vector>

using namespace segpa;

namespace {

thread_local std::string g_err = "";

segpa_status_t fail(segpa_status_t st, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return st;
}

struct StreamKey {
    int32_t layer, kv_head;
    int64_t seq;
    bool operator==(const StreamKey& o) const { return layer == o.layer && kv_head == o.kv_head && seq == o.seq; }
};
struct StreamKeyHash {
    size_t operator()(const StreamKey& k) const {
        uint64_t h = (uint64_t)k.seq * 0x9E3779B97F4A7C15ull;
        h ^= ((uint64_t)(uint32_t)k.layer << 32 | (uint32_t)k.kv_head) + 0x7F4A7C15u + (h << 6) + (h >> 2);
        return (size_t)h;
    }
};
// Head segments: a stream is the concatenation of head segments, each on its own consecutive
// pages, so a segment whose length is not a multiple of P leaves unused slots behind its tail in mid-stream.  The
// stream is kept in SLOT space (slot = page index * P + slot in page): token j sits at slot j + pad(j), where pad(j)
// is the cumulative number of unused slots before j's segment.  Only the points where the padding grows are stored.
struct PadPoint {
    int64_t tok;   // first token of a head segment that starts on a fresh page after a partial one
    int64_t pad;   // unused slots before it, cumulative: tokens >= tok (up to the next point) sit at slot tok' + pad
};
struct StreamRec {
    std::vector<int32_t> pages;
    int64_t kv_len = 0;
    std::vector<PadPoint> pads;   // ascending; empty = the stream is dense (token j in page j / P, slot j % P)
    bool tail_open = false;       // the partial last page was started by a COPY append of this stream (it may be filled further)
    int64_t n_holes = 0;          // evicted pages (entries -1 of `pages`)
    int64_t slot_len() const { return kv_len + (pads.empty() ? 0 : pads.back().pad); }
    int64_t slot_of(int64_t tok) const {
        int64_t pad = 0;
        for (const PadPoint& pp : pads) { if (pp.tok <= tok) pad = pp.pad; else break; }
        return tok + pad;
    }
    // append_pages_batch: index of this stream's last COPY job in the batch with stamp `batch_stamp`
    uint64_t batch_stamp = 0;
    int32_t batch_job = -1;
};

struct DeviceGuard {
    int prev = -1;
    bool active = false;
    explicit DeviceGuard(int dev) {
        if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) {
            cudaSetDevice(dev);
            active = true;
        }
    }
    ~DeviceGuard() { if (active) cudaSetDevice(prev); }
};

}  // namespace

namespace {

// Pinned host + device buffer pair reused by successive uploads.  `ev` marks the completion of the
// last work that used the pair; it is waited for (on the host) before the pair is overwritten.
struct Staging {
    void* h = nullptr;
    void* d = nullptr;
    size_t cap = 0;
    cudaEvent_t ev = nullptr;
    bool pending = false;
    cudaEvent_t up = nullptr;   // upload of h -> d has completed (staging_upload)
};

cudaError_t staging_acquire(Staging& s, size_t bytes) {
    cudaError_t e = cudaSuccess;
    if (!s.ev) {
        e = cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming);
        if (e != cudaSuccess) return e;
    }
    if (s.pending) {
        e = cudaEventSynchronize(s.ev);
        s.pending = false;
        if (e != cudaSuccess) return e;
    }
    if (bytes > s.cap) {
        if (s.h) cudaFreeHost(s.h);
        if (s.d) cudaFree(s.d);
        s.h = s.d = nullptr;
        s.cap = 0;
        const size_t cap = std::max<size_t>(bytes + bytes / 2, 64 << 10);
        e = cudaMallocHost(&s.h, cap);
        if (e == cudaSuccess) e = cudaMalloc(&s.d, cap);
        if (e != cudaSuccess) {
            if (s.h) cudaFreeHost(s.h);
            s.h = nullptr;
            return e;
        }
        s.cap = cap;
    }
    return cudaSuccess;
}

// h -> d on the cache's own copy stream, then `st` waits for it: descriptors go up while the work already queued
// in `st` (the previous step's kernels) is still running, instead of queueing behind it.  Safe because the pair
// is only handed out (staging_acquire) once its last consumer has finished.
cudaError_t staging_upload(Staging& s, size_t bytes, cudaStream_t up_stream, cudaStream_t st) {
    if (!up_stream) return cudaMemcpyAsync(s.d, s.h, bytes, cudaMemcpyHostToDevice, st);
    cudaError_t e = cudaSuccess;
    if (!s.up) e = cudaEventCreateWithFlags(&s.up, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMemcpyAsync(s.d, s.h, bytes, cudaMemcpyHostToDevice, up_stream);
    if (e == cudaSuccess) e = cudaEventRecord(s.up, up_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, s.up, 0);
    return e;
}

void staging_release(Staging& s, cudaStream_t st) {
    if (s.ev && cudaEventRecord(s.ev, st) == cudaSuccess) s.pending = true;
}

void staging_free(Staging& s) {
    if (s.h) cudaFreeHost(s.h);
    if (s.d) cudaFree(s.d);
    if (s.ev) cudaEventDestroy(s.ev);
    if (s.up) cudaEventDestroy(s.up);
    s = Staging();
}

// Device-side storage of one segments object (descriptor blob, scheduler cursor, split-KV
// workspace); recycled through the cache's free list instead of cudaMalloc / cudaFree per build.
struct SegBuf {
    Staging blob;
    Staging mass_blob;    // attention-mass plan (items, per-CTA slices, layout), uploaded at the first mass call
    Staging host_blob;    // row-chunked plan of segpa_attention_fwd_host (items, per-CTA slices, combine entries per chunk)
    int* counter = nullptr;
    float* ws_o = nullptr;
    float* ws_ml = nullptr;
    size_t ws_rows = 0;   // capacity in partial rows
};

void segbuf_free(SegBuf* b) {
    if (!b) return;
    staging_free(b->blob);
    staging_free(b->mass_blob);
    staging_free(b->host_blob);
    if (b->counter) cudaFree(b->counter);
    if (b->ws_o) cudaFree(b->ws_o);
    if (b->ws_ml) cudaFree(b->ws_ml);
    delete b;
}

}  // namespace

struct segpa_segments {
    segpa_cache* cache = nullptr;
    int32_t layer = 0;
    std::vector<segpa_segment_req_t> reqs;
    std::vector<SegDev> segs;
    std::vector<ItemDev> items;
    struct ItemMeta { int32_t tile; int32_t split; int32_t n_splits; };
    std::vector<ItemMeta> item_meta;   // per item (same order as items): what segpa_segments_items reports besides ItemDev
    std::vector<int32_t> pages;
    std::vector<PadDev> pads;       // token -> slot maps of the ragged streams among the segments
    std::vector<CombDev> combs;
    std::vector<int32_t> cta_off;   // items of CTA q: [cta_off[q], cta_off[q+1])
    std::vector<int64_t> mass_off;  // [n + 1]: layout of the attention-mass array (kv_len rounded up to 128 per segment)
    bool has_ragged = false;             // some segment's stream has head segments with partial last pages
    bool narrow = false;                 // every tile holds <= 16 rows (decode-shaped plan; FwdParams::narrow)
    mutable bool mass_planned = false;   // mass plan built and uploaded (lazily, by the first segpa_attention_mass)
    mutable int mass_n_cta = 0;
    mutable size_t m_off_items = 0, m_off_cta = 0, m_off_layout = 0, m_off_kvlen = 0;
    // segpa_attention_fwd_host: the plan cut into row chunks, each with its own launch, so that the H2D copy of
    // chunk k+1, the kernels of chunk k and the D2H copy of chunk k-1 overlap (built at the first call)
    struct HostChunk {
        int64_t row_lo, row_hi;      // rows copied in / out with this chunk
        int64_t need_hi;             // its items read Q rows below this (<= row_hi of the next chunk)
        size_t off_items, off_cta, off_combs;
        int n_items, n_cta, n_combs, comb_max_rows;
    };
    mutable std::vector<HostChunk> hchunks;
    mutable bool host_planned = false;
    segpa_plan_stats_t stats{};
    int tiles_per_item = 1;
    // device
    SegBuf* buf = nullptr;
    mutable cudaStream_t last_stream = nullptr;   // stream of the last upload / attention_fwd
    size_t off_segs = 0, off_items = 0, off_pages = 0, off_combs = 0, off_cta = 0, off_pads = 0;

    // back to the state of a fresh object, keeping the vectors' storage (objects are recycled through the
    // cache: a plan is built on the critical path of every layer and must not go through malloc / page faults)
    void reset() {
        cache = nullptr; layer = 0;
        reqs.clear(); segs.clear(); items.clear(); item_meta.clear(); pages.clear(); pads.clear(); combs.clear(); cta_off.clear(); mass_off.clear();
        mass_planned = false; mass_n_cta = 0; has_ragged = false; narrow = false;
        hchunks.clear(); host_planned = false;
        m_off_items = m_off_cta = m_off_layout = m_off_kvlen = 0;
        stats = segpa_plan_stats_t{};
        tiles_per_item = 1;
        buf = nullptr; last_stream = nullptr;
        off_segs = off_items = off_pages = off_combs = off_cta = off_pads = 0;
    }
};

// build_segments scratch, kept in the cache between calls (same reason)
struct PlanTile { int seg, t0, n_tok, kb_lo, kb_hi, cost; bool sink; };
struct PlanIv { int32_t kv_head; int64_t lo, hi; };
struct PlanScratch {
    std::vector<PlanTile> tiles;
    std::vector<PlanIv> ivs;
    std::vector<int> order, start, item_cta, count, cursor;
    std::vector<int64_t> heap;
    std::vector<ItemDev> it2;
    std::vector<segpa_segments::ItemMeta> im2;
};

struct segpa_cache {
    segpa_cache_desc_t desc{};
    int G = 1;
    int page_bytes = 0;
    bool planning_only = false;
    bool own_pool = true;
    uint8_t* k_pool = nullptr;
    uint8_t* v_pool = nullptr;
    std::vector<int32_t> refcnt;
    std::vector<int32_t> free_list;  // may hold stale entries (refcnt != 0: pages taken by caller-given id): skipped on pop
    std::vector<uint8_t> in_free;    // page id is somewhere in free_list (so a release never adds a second entry)
    int64_t n_free = 0;
    int64_t n_shared_pages = 0;      // pages with reference count > 1 (kept as the counts change): while it is 0 no stream shares a page
    std::unordered_map<StreamKey, StreamRec, StreamKeyHash> streams;
    std::vector<segpa_segments*> seg_objs;
    std::vector<SegBuf*> free_bufs;   // released device storage, oldest first
    size_t n_seg_bufs = 0;            // SegBufs alive (in free_bufs or owned by a segments object)
    std::vector<segpa_segments*> free_seg_objs;   // recycled host-side plan objects
    PlanScratch plan;
    std::vector<int32_t> append_touched;   // append_pages_batch scratch, kept between calls
    Staging append_stage[2];         // alternating, so staging a batch does not wait for the previous one
    int append_turn = 0;
    uint64_t batch_stamp = 0;        // one per append_pages_batch call (StreamRec::batch_stamp)
    int num_sms = 148;
    cudaStream_t up_stream = nullptr;   // descriptor uploads (staging_upload)
    int kernel_kind = 1;  // 1 = tcgen05 (the product); 0 = SIMT cross-check kernel, only in the test build (-DSEGPA_BRINGUP)
    int tiles_per_item = 2;   // 128-row tiles per work item (desc.tiles_per_item; fixed at create)
    int last_launches = 0;
    // host-buffer entry points: device staging, copy streams and events
    // Q / out / LSE staging of segpa_attention_fwd_host: two sets, so that a call may be enqueued (the _async entry
    // point) while the copies back of the previous one are still running.  The synchronous entry point uses set 0.
    struct HostStage {
        uint16_t* q = nullptr;
        uint16_t* out = nullptr;
        float* lse = nullptr;
        size_t q_bytes = 0, lse_bytes = 0;
        cudaEvent_t done = nullptr;      // recorded on d2h_stream after the set's last copy back
        bool pending = false;            // done has been recorded and not yet waited for by the host
    } hs[2];
    int hs_turn = 0;
    uint16_t* st_kv = nullptr;          // K / V rows of host-source append requests (src_is_host)
    size_t st_kv_bytes = 0;
    cudaEvent_t st_kv_ev = nullptr;     // the scatter that last read st_kv has completed
    bool st_kv_pending = false;
    cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
    std::vector<cudaEvent_t> host_events;
};

namespace {

int32_t pop_free_page(segpa_cache* c) {
    while (!c->free_list.empty()) {
        int32_t id = c->free_list.back();
        c->free_list.pop_back();
        c->in_free[(size_t)id] = 0;
        if (c->refcnt[id] == 0) return id;
    }
    return -1;
}

void release_page(segpa_cache* c, int32_t id) {
    if (c->refcnt[id] == 2) --c->n_shared_pages;
    if (--c->refcnt[id] == 0) {
        if (!c->in_free[(size_t)id]) {
            c->free_list.push_back(id);
            c->in_free[(size_t)id] = 1;
        }
        ++c->n_free;
    }
}

// returns the object's device storage to the cache's free list (no device synchronisation)
void free_segments_obj(segpa_cache* c, segpa_segments* s) {
    if (!s) return;
    if (s->buf) {
        staging_release(s->buf->blob, s->last_stream);
        if (s->mass_planned) staging_release(s->buf->mass_blob, s->last_stream);
        if (s->host_planned) staging_release(s->buf->host_blob, s->last_stream);
        c->free_bufs.push_back(s->buf);
    }
    if (c->free_seg_objs.size() < 64) {
        s->reset();
        c->free_seg_objs.push_back(s);
    } else {
        delete s;
    }
}

inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

// TMA descriptor of Q [T][Hq][D] bf16 (row stride given): box {64 elements, G heads, tile_tokens tokens},
// SWIZZLE_128B, out-of-range tokens zero-filled.  One box = one 64-element half of a 128-row Q tile.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

const char* encode_q_map(TensorMap* out, const void* q, int64_t T, int Hq, int D, int G, int tile_tokens,
                         int64_t row_stride_elems) {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qr) != cudaSuccess || !f ||
            qr != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            return "cuTensorMapEncodeTiled is not available from the driver";
        }
        fn = (EncodeTiledFn)f;
    }
    static_assert(sizeof(CUtensorMap) == sizeof(TensorMap), "tensor map size");
    static_assert(SEGPA_NOALLOC_MAX_PAGES == kNoAllocMaxPages, "header and kernel file must agree on the scratch size");
    const cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)Hq, (cuuint64_t)T};
    const cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)row_stride_elems * 2};
    const cuuint32_t box[3] = {64u, (cuuint32_t)G, (cuuint32_t)tile_tokens};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    CUresult r = fn((CUtensorMap*)out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(q), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? nullptr : "cuTensorMapEncodeTiled failed";
}

// attended (query, key) pairs of the queries at positions [i0, i1]: sum of min(i + 1, W) (Alg. 2 policy;
// PAPER.md:219 with W = w + 1; GLOBAL passes a W larger than any position)
inline int64_t visible_pairs(int64_t i0, int64_t i1, int64_t W) {
    auto tri = [](int64_t a, int64_t b) { return a > b ? (int64_t)0 : (a + b) * (b - a + 1) / 2; };   // a + ... + b
    const int64_t knee = W - 1;                       // positions <= knee see i + 1 keys, later ones see W
    const int64_t ramp = tri(i0 + 1, std::min(i1, knee) + 1);
    const int64_t flat = i1 > knee ? (i1 - std::max(i0, knee + 1) + 1) * W : 0;
    return ramp + flat;
}

}  // namespace

namespace {

// Cuts the token range [t0, t0 + n) of a stream at its head-segment boundaries: f(tok_lo, n_piece, slot_lo) for
// every maximal piece whose tokens are consecutive in slot space.
template <class F>
void for_each_piece(const StreamRec& rec, int64_t t0, int64_t n, F f) {
    int64_t t = t0;
    const int64_t end = t0 + n;
    size_t k = 0;
    int64_t pad = 0;
    while (k < rec.pads.size() && rec.pads[k].tok <= t) pad = rec.pads[k++].pad;
    while (t < end) {
        const int64_t stop = (k < rec.pads.size()) ? std::min(end, rec.pads[k].tok) : end;
        f(t, stop - t, t + pad);
        t = stop;
        if (k < rec.pads.size() && rec.pads[k].tok <= t) pad = rec.pads[k++].pad;
    }
}

// LPT: items by descending cost, each given to the least-loaded CTA of the persistent grid;
// a CTA's items stay in descending order.  Cost = visited blocks + a fixed per-item term (pipeline refill, Q load,
// epilogue: about 0.6 block-times measured), in thirds of a block.  Reorders `items` (and `meta`, if given) CTA by
// CTA and fills cta_off ([n_cta + 1]).  Flat arrays only: a plan is built on the critical path of every layer.
// Returns the sum of the items' costs.
int64_t lpt_assign(PlanScratch& ps, std::vector<ItemDev>& items_v, std::vector<segpa_segments::ItemMeta>* meta, int num_sms,
                   std::vector<int32_t>& cta_off) {
    const int n_items_all = (int)items_v.size();
    const int n_cta = std::min(n_items_all, num_sms);
    // descending cost, ties by ascending index: a counting sort (costs are block counts, small integers)
    std::vector<int>& order = ps.order;
    order.resize((size_t)n_items_all);
    {
        int max_cost = 0;
        for (const ItemDev& it : items_v) max_cost = std::max(max_cost, it.cost);
        std::vector<int>& start = ps.start;
        start.assign((size_t)max_cost + 2, 0);
        for (const ItemDev& it : items_v) ++start[(size_t)(max_cost - it.cost) + 1];
        for (int k2 = 0; k2 <= max_cost; ++k2) start[(size_t)k2 + 1] += start[(size_t)k2];
        for (int i = 0; i < n_items_all; ++i) order[(size_t)start[(size_t)(max_cost - items_v[(size_t)i].cost)]++] = i;
    }
    // Each item, in that order, goes to the least-loaded CTA.  The loads are kept as one ascending run of
    // keys load * 1024 + cta (distinct, so the minimum is unique) inside a longer array: the minimum leaves at
    // the head, the CTA's new key is inserted from the tail.  With costs descending the new key belongs at or
    // near the tail, so an assignment costs a few moves (a binary heap's dependent loads per level cost more)
    std::vector<int64_t>& run = ps.heap;
    run.resize((size_t)n_cta + (size_t)n_items_all);
    for (int q = 0; q < n_cta; ++q) run[(size_t)q] = q;
    std::vector<int>&item_cta = ps.item_cta, &count = ps.count, &cursor = ps.cursor;
    item_cta.resize((size_t)n_items_all);
    count.assign((size_t)n_cta, 0);
    {
        int64_t* a = run.data();
        const ItemDev* items = items_v.data();
        const int64_t fixed3 = 2;   // the fixed per-item term, in thirds of a block (a sweep over 0..6 moved cfg2 / cfg4 by < 0.5 %)
        size_t head = 0, tail = (size_t)n_cta;
        for (int idx : order) {
            const int64_t top = a[head++];
            const int q = (int)(top & 1023);
            item_cta[(size_t)idx] = q;
            ++count[(size_t)q];
            const int64_t blocks3 = 3 * (int64_t)items[idx].cost;
            const int64_t key = top + (((items[idx].flags & 1) ? (blocks3 + 1) / 2 : blocks3) + fixed3) * 1024;   // strided: two chains
            size_t pos = tail++;
            while (pos > head && a[pos - 1] > key) {
                a[pos] = a[pos - 1];
                --pos;
            }
            a[pos] = key;
        }
    }
    // per-CTA slices: CTA by CTA, each CTA's items in the order they were assigned (descending cost)
    cta_off.assign((size_t)n_cta + 1, 0);
    for (int q = 0; q < n_cta; ++q) cta_off[(size_t)q + 1] = cta_off[(size_t)q] + count[(size_t)q];
    std::vector<ItemDev>& it2 = ps.it2;
    std::vector<segpa_segments::ItemMeta>& im2 = ps.im2;
    it2.resize((size_t)n_items_all);
    if (meta) im2.resize((size_t)n_items_all);
    cursor.assign(cta_off.begin(), cta_off.end() - 1);
    int64_t kv_blocks = 0;
    for (int idx : order) {
        const int at = cursor[(size_t)item_cta[(size_t)idx]]++;
        it2[(size_t)at] = items_v[(size_t)idx];
        if (meta) im2[(size_t)at] = (*meta)[(size_t)idx];
        kv_blocks += items_v[(size_t)idx].cost;
    }
    items_v.swap(it2);
    if (meta) meta->swap(im2);
    return kv_blocks;
}

// fills FwdParams from a cache + segments object (everything but q / out / lse, their strides, the Q tensor map and
// the per-launch item arrays)
void fill_fwd_params(FwdParams& p, const segpa_cache* c, const segpa_segments* s) {
    const uint8_t* d_blob = (const uint8_t*)s->buf->blob.d;
    p.segs = (const SegDev*)(d_blob + s->off_segs);
    p.items = (const ItemDev*)(d_blob + s->off_items);
    p.pages = (const int*)(d_blob + s->off_pages);
    p.pads = (const PadDev*)(d_blob + s->off_pads);
    p.combs = (const CombDev*)(d_blob + s->off_combs);
    p.cta_off = (const int*)(d_blob + s->off_cta);
    p.n_cta = (int)s->cta_off.size() - 1;
    p.n_items = (int)s->items.size();
    p.n_combs = (int)s->combs.size();
    p.comb_max_rows = 0;
    p.comb_max_parts = 0;
    for (const CombDev& cd : s->combs) {
        p.comb_max_rows = std::max(p.comb_max_rows, cd.n_tok * c->G);
        p.comb_max_parts = std::max(p.comb_max_parts, cd.n_splits * ((cd.flags & 1) ? 2 : 1));
    }
    p.counter = s->buf->counter;
    p.k_pool = c->k_pool;
    p.v_pool = c->v_pool;
    p.ws_o = s->buf->ws_o;
    p.ws_ml = s->buf->ws_ml;
    p.Hq = c->desc.num_q_heads;
    p.Hkv = c->desc.num_kv_heads;
    p.G = c->G;
    p.D = c->desc.head_dim;
    p.P = c->desc.page_size;
    p.tile_tokens = kTileRows / c->G;
    p.tiles_per_item = s->tiles_per_item;
    p.page_bytes = c->page_bytes;
    p.num_sms = c->num_sms;
    p.has_ragged = s->has_ragged ? 1 : 0;
    p.narrow = s->narrow ? 1 : 0;
}

}  // namespace

extern "C" {

const char* segpa_last_error(void) { return g_err.c_str(); }
int32_t segpa_version(void) { return SEGPA_VERSION; }

int64_t segpa_pool_bytes(const segpa_cache_desc_t* d) {
    if (!d || d->num_pages < 1 || d->page_size < 1 || d->head_dim < 1) return 0;
    return (d->num_pages + 1) * (int64_t)d->page_size * d->head_dim * 2;
}

segpa_status_t segpa_create_cache(const segpa_cache_desc_t* d, segpa_cache_t** out) {
    if (!d || !out) return fail(SEGPA_ERR_INVALID, "create_cache: null argument");
    *out = nullptr;
    if (d->num_layers < 1 || d->num_q_heads < 1 || d->num_kv_heads < 1 || d->num_pages < 1)
        return fail(SEGPA_ERR_INVALID, "create_cache: counts must be >= 1");
    if (d->num_q_heads % d->num_kv_heads != 0)
        return fail(SEGPA_ERR_INVALID, "create_cache: num_q_heads %d not a multiple of num_kv_heads %d",
                    d->num_q_heads, d->num_kv_heads);
    if (d->head_dim != 64 && d->head_dim != 128)
        return fail(SEGPA_ERR_UNSUPPORTED, "create_cache: head_dim %d (supported: 64, 128)", d->head_dim);
    if (d->page_size != 16 && d->page_size != 32)
        return fail(SEGPA_ERR_UNSUPPORTED, "create_cache: page_size %d (supported: 16, 32)", d->page_size);
    if (d->num_q_heads / d->num_kv_heads > 16)
        return fail(SEGPA_ERR_UNSUPPORTED, "create_cache: GQA group %d > 16", d->num_q_heads / d->num_kv_heads);
    if (d->num_pages >= INT32_MAX - 1) return fail(SEGPA_ERR_INVALID, "create_cache: num_pages too large");
    if ((d->k_pool == nullptr) != (d->v_pool == nullptr))
        return fail(SEGPA_ERR_INVALID, "create_cache: give both k_pool and v_pool or neither");
    if (d->device < -1) return fail(SEGPA_ERR_INVALID, "create_cache: bad device %d", d->device);
    if (d->tiles_per_item < 0 || d->tiles_per_item > 2) return fail(SEGPA_ERR_INVALID, "create_cache: tiles_per_item %d (0 = default, 1 or 2)", d->tiles_per_item);

    segpa_cache* c = new (std::nothrow) segpa_cache();
    if (!c) return fail(SEGPA_ERR_OOM, "create_cache: host allocation failed");
    c->desc = *d;
    c->G = d->num_q_heads / d->num_kv_heads;
    c->page_bytes = d->page_size * d->head_dim * 2;
    c->planning_only = (d->device == -1);
    c->tiles_per_item = d->tiles_per_item == 0 ? 2 : d->tiles_per_item;
    try {
        c->refcnt.assign((size_t)d->num_pages, 0);
        c->free_list.resize((size_t)d->num_pages);
        for (int64_t i = 0; i < d->num_pages; ++i) c->free_list[(size_t)i] = (int32_t)(d->num_pages - 1 - i);
        c->in_free.assign((size_t)d->num_pages, 1);
    } catch (const std::bad_alloc&) {
        delete c;
        return fail(SEGPA_ERR_OOM, "create_cache: host allocation failed");
    }
    c->n_free = d->num_pages;

    if (!c->planning_only) {
        int ndev = 0;
        cudaError_t e = cudaGetDeviceCount(&ndev);
        if (e != cudaSuccess || d->device >= ndev) {
            delete c;
            return fail(SEGPA_ERR_CUDA, "create_cache: no CUDA device %d (%s); there is no CPU fallback",
                        d->device, e == cudaSuccess ? "ordinal out of range" : cudaGetErrorString(e));
        }
        cudaDeviceProp prop{};
        cudaGetDeviceProperties(&prop, d->device);
        if (prop.major != 10) {
            delete c;
            return fail(SEGPA_ERR_UNSUPPORTED, "create_cache: device %d is sm_%d%d; this library is built for sm_100a",
                        d->device, prop.major, prop.minor);
        }
        c->num_sms = prop.multiProcessorCount;
        DeviceGuard g(d->device);
        if (cudaStreamCreateWithFlags(&c->up_stream, cudaStreamNonBlocking) != cudaSuccess) {
            cudaGetLastError();
            c->up_stream = nullptr;   // uploads then go through the caller's stream
        }
        const size_t bytes = (size_t)segpa_pool_bytes(d);
        if (d->k_pool) {
            c->own_pool = false;
            c->k_pool = (uint8_t*)d->k_pool;
            c->v_pool = (uint8_t*)d->v_pool;
        } else {
            if (cudaMalloc(&c->k_pool, bytes) != cudaSuccess || cudaMalloc(&c->v_pool, bytes) != cudaSuccess) {
                cudaGetLastError();
                if (c->k_pool) cudaFree(c->k_pool);
                delete c;
                return fail(SEGPA_ERR_OOM, "create_cache: cudaMalloc of 2 x %zu bytes failed", bytes);
            }
        }
        if (cudaMemset(c->k_pool, 0, bytes) != cudaSuccess || cudaMemset(c->v_pool, 0, bytes) != cudaSuccess) {
            cudaError_t e2 = cudaGetLastError();
            if (c->own_pool) { cudaFree(c->k_pool); cudaFree(c->v_pool); }
            delete c;
            return fail(SEGPA_ERR_CUDA, "create_cache: memset failed: %s", cudaGetErrorString(e2));
        }
    }
    *out = c;
    return SEGPA_OK;
}

segpa_status_t segpa_destroy(segpa_cache_t* c) {
    if (!c) return SEGPA_OK;
    DeviceGuard g(c->desc.device);
    if (!c->planning_only) cudaDeviceSynchronize();
    for (auto* s : c->seg_objs) free_segments_obj(c, s);
    for (auto* b : c->free_bufs) segbuf_free(b);
    for (auto* s : c->free_seg_objs) delete s;
    staging_free(c->append_stage[0]);
    staging_free(c->append_stage[1]);
    if (c->up_stream) cudaStreamDestroy(c->up_stream);
    for (auto& h : c->hs) {
        if (h.q) cudaFree(h.q);
        if (h.out) cudaFree(h.out);
        if (h.lse) cudaFree(h.lse);
        if (h.done) cudaEventDestroy(h.done);
    }
    if (c->st_kv) cudaFree(c->st_kv);
    if (c->st_kv_ev) cudaEventDestroy(c->st_kv_ev);
    if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
    if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
    for (cudaEvent_t ev : c->host_events) cudaEventDestroy(ev);
    if (c->own_pool && c->k_pool) { cudaFree(c->k_pool); cudaFree(c->v_pool); }
    delete c;
    return SEGPA_OK;
}

segpa_status_t segpa_append_pages_batch(segpa_cache_t* c, const segpa_append_req_t* reqs, int32_t n,
                                        void* cuda_stream) {
    if (!c || !reqs) return fail(SEGPA_ERR_INVALID, "append_pages: null argument");
    if (n < 1) return fail(SEGPA_ERR_INVALID, "append_pages: batch size %d < 1", n);
    const int P = c->desc.page_size, D = c->desc.head_dim;

    // Requests are applied to the host state in order; `undo` lets a later failure restore it exactly.
    struct Undo { StreamKey key; bool created; int64_t old_len; size_t n_new; size_t old_pads; bool old_tail_open; };
    std::vector<Undo> undo;
    std::vector<ScatterJob> jobs;
    std::vector<int32_t>& touched = c->append_touched;     // page ids the scatter kernel indexes, job after job
    touched.clear();
    const uint64_t stamp = ++c->batch_stamp;
    // host-source requests (src_is_host): their rows are staged in st_kv ([K rows of all such requests][V rows]) by
    // async copies on cuda_stream ahead of the scatter launch
    struct HostCopy { const void* k; const void* v; int64_t stride, n, off_rows; };
    std::vector<HostCopy> host_copies;
    int64_t host_rows = 0, host_rows_total = 0;
    for (int32_t i = 0; i < n; ++i)
        if (reqs[i].src_is_host == 1 && reqs[i].k_src && reqs[i].n_tokens > 0) host_rows_total += reqs[i].n_tokens;
    if (host_rows_total > 0 && !c->planning_only) {
        DeviceGuard g(c->desc.device);
        const size_t need_bytes = (size_t)host_rows_total * D * 2 * 2;
        if (need_bytes > c->st_kv_bytes) {
            if (c->st_kv_pending) { cudaEventSynchronize(c->st_kv_ev); c->st_kv_pending = false; }
            if (c->st_kv) cudaFree(c->st_kv);
            c->st_kv = nullptr;
            c->st_kv_bytes = 0;
            if (cudaMalloc((void**)&c->st_kv, need_bytes + need_bytes / 4) != cudaSuccess) {
                cudaGetLastError();
                return fail(SEGPA_ERR_OOM, "append_pages: staging allocation of %zu bytes for host-source rows failed", need_bytes);
            }
            c->st_kv_bytes = need_bytes + need_bytes / 4;
        }
    }
    long long total_chunks = 0;
    try {
        size_t ub = 0;   // one allocation at most (an upper bound of the ids listed: new pages + a refilled last page per job)
        for (int32_t i = 0; i < n; ++i) ub += (size_t)(std::max<int64_t>(reqs[i].n_tokens, 0) / P) + 2;
        touched.reserve(ub);
        undo.reserve((size_t)n);
        jobs.reserve((size_t)n);
    } catch (const std::bad_alloc&) {
        return fail(SEGPA_ERR_OOM, "append_pages: host allocation failed");
    }
    auto rollback = [&]() {
        for (size_t u = undo.size(); u-- > 0;) {
            auto it = c->streams.find(undo[u].key);
            StreamRec& rec = it->second;
            for (size_t k = 0; k < undo[u].n_new; ++k) {
                release_page(c, rec.pages.back());
                rec.pages.pop_back();
            }
            rec.kv_len = undo[u].old_len;
            rec.pads.resize(undo[u].old_pads);
            rec.tail_open = undo[u].old_tail_open;
            if (undo[u].created) c->streams.erase(it);
        }
    };
#define APPEND_FAIL(code, ...) do { rollback(); return fail(code, __VA_ARGS__); } while (0)

    try {
        for (int32_t i = 0; i < n; ++i) {
            const segpa_append_req_t& r = reqs[i];
            if (r.layer < 0 || r.layer >= c->desc.num_layers) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: layer %d out of range", i, r.layer);
            if (r.kv_head < 0 || r.kv_head >= c->desc.num_kv_heads) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: kv_head %d out of range", i, r.kv_head);
            if (r.n_tokens < 1) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: n_tokens %lld < 1", i, (long long)r.n_tokens);
            if ((r.k_src == nullptr) != (r.v_src == nullptr)) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: give both k_src and v_src, or neither (attach)", i);
            if (r.n_page_ids < 0 || (r.n_page_ids > 0 && !r.page_ids)) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: bad page_ids", i);
            const bool attach = (r.k_src == nullptr);
            if (r.src_is_host != 0 && r.src_is_host != 1) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: src_is_host must be 0 or 1", i);
            const bool from_host = !attach && r.src_is_host == 1;
            if (!attach && c->planning_only) APPEND_FAIL(SEGPA_ERR_STATE, "append_pages[%d]: copy mode on a planning-only cache", i);
            if (!attach && r.src_row_stride_elems < D) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: src_row_stride_elems %lld < head_dim", i, (long long)r.src_row_stride_elems);
            if (!attach && !from_host && ((r.src_row_stride_elems % 8) || ((uintptr_t)r.k_src % 16) || ((uintptr_t)r.v_src % 16)))
                APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: k_src / v_src must be 16-byte aligned with a row stride multiple of 8 elements", i);

            const StreamKey key{r.layer, r.kv_head, r.seq_id};
            auto it = c->streams.find(key);
            const bool created = (it == c->streams.end());
            const int64_t cur_len = created ? 0 : it->second.kv_len;
            const int64_t cur_slots_raw = created ? 0 : it->second.slot_len();
            const int64_t cur_pages = created ? 0 : (int64_t)it->second.pages.size();   // = ceil(slot_len / P)
            // The new tokens continue inside the stream's partial last page only if that page was started by a COPY
            // append of this very stream and nobody else refers to it.  Otherwise (ATTACH of a reused chunk; new tokens
            // after an attached chunk whose length is not a multiple of P; a last page shared with another stream) they
            // form a new head segment on a fresh page, and the rest of the partial page stays unused in mid-stream
            // (every head segment has its own consecutive pages).
            const bool partial = cur_slots_raw % P != 0;
            const bool in_place = partial && !attach && it->second.tail_open && c->refcnt[it->second.pages.back()] == 1;
            const int64_t new_pad = (partial && !in_place) ? P - cur_slots_raw % P : 0;
            const int64_t cur_slots = cur_slots_raw + new_pad;
            const int64_t new_len = cur_len + r.n_tokens;
            if (cur_slots + r.n_tokens > (int64_t)INT32_MAX - 2 * kBlockKeys) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: stream too long", i);
            const int64_t need = cdiv(cur_slots + r.n_tokens, P) - cur_pages;

            if (attach) {
                if (!r.page_ids) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: attach needs page_ids", i);
                if (r.n_page_ids != need) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: attach needs %lld page ids, got %d", i, (long long)need, r.n_page_ids);
            } else if (r.page_ids) {
                if (r.n_page_ids != need) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: need %lld page ids, got %d", i, (long long)need, r.n_page_ids);
            } else {
                if (need > c->n_free) APPEND_FAIL(SEGPA_ERR_OOM, "append_pages[%d]: pool exhausted (%lld pages needed, %lld free)", i, (long long)need, (long long)c->n_free);
            }

            // Apply the request.  The given page ids are checked as they are taken (one pass over the pool state,
            // which is random access into a table far larger than the host caches); a bad id undoes this request's
            // partial application together with the earlier requests (rollback).
            StreamRec& rec = c->streams[key];
            undo.push_back(Undo{key, created, cur_len, 0, rec.pads.size(), rec.tail_open});
            rec.pages.reserve(rec.pages.size() + (size_t)need);
            if (new_pad > 0) rec.pads.push_back(PadPoint{cur_len, (rec.pads.empty() ? 0 : rec.pads.back().pad) + new_pad});
            if (in_place) {
                // An earlier COPY job of this batch that ended in the same page must not zero-fill the slots this
                // job writes (both run in one launch, unordered): its writes stop at its own last token.
                if (rec.batch_stamp == stamp && rec.batch_job >= 0) jobs[(size_t)rec.batch_job].n_write = jobs[(size_t)rec.batch_job].n_tokens;
            }
            if (!attach) {
                ScatterJob jb{};
                jb.k_src = (const uint16_t*)r.k_src;
                jb.v_src = (const uint16_t*)r.v_src;
                jb.src_stride = r.src_row_stride_elems;
                if (from_host) {
                    host_copies.push_back(HostCopy{r.k_src, r.v_src, r.src_row_stride_elems, r.n_tokens, host_rows});
                    jb.k_src = c->st_kv + (size_t)host_rows * D;
                    jb.v_src = c->st_kv + (size_t)(host_rows_total + host_rows) * D;
                    jb.src_stride = D;
                    host_rows += r.n_tokens;
                }
                jb.n_tokens = r.n_tokens;
                jb.chunk_begin = total_chunks;
                jb.page_off = (long long)touched.size();
                jb.first_slot = (int)(cur_slots % P);
                jb.n_pages = (int)need + (in_place ? 1 : 0);
                if (in_place) touched.push_back(rec.pages.back());   // (a partial last page is never a hole: evict_pages refuses it)
                jb.n_write = (long long)jb.n_pages * P - jb.first_slot;     // rows + the zero-filled tail of the last page
                total_chunks += jb.n_write * (D >> 3);
                rec.batch_stamp = stamp;
                rec.batch_job = (int32_t)jobs.size();
                jobs.push_back(jb);
            }
            rec.tail_open = !attach;
            for (int64_t k = 0; k < need; ++k) {
                int32_t id;
                if (r.page_ids) {
                    id = r.page_ids[k];
                    if (k + 16 < need) {   // the table is walked in the (random) order of the ids: fetch ahead
                        const int32_t nx = r.page_ids[k + 16];
                        if (nx >= 0 && nx < c->desc.num_pages) __builtin_prefetch(&c->refcnt[nx], 1);
                    }
                    if (id < 0 || id >= c->desc.num_pages) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: page id %d out of range", i, id);
                    const int32_t rc = c->refcnt[id];
                    if (attach) {
                        if (!c->planning_only && rc == 0) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: attach of page %d which holds no data", i, id);
                    } else if (rc != 0) {
                        // taken: by an earlier entry of this very request (duplicate), or before it
                        if (std::find(r.page_ids, r.page_ids + k, id) != r.page_ids + k) APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: duplicate page id %d", i, id);
                        APPEND_FAIL(SEGPA_ERR_INVALID, "append_pages[%d]: page %d is not free", i, id);
                    }
                } else {
                    id = pop_free_page(c);
                }
                ++undo.back().n_new;
                if (c->refcnt[id] == 0) --c->n_free;
                if (++c->refcnt[id] == 2) ++c->n_shared_pages;
                rec.pages.push_back(id);
                if (!attach) touched.push_back(id);
            }
            rec.kv_len = new_len;
        }
    } catch (const std::bad_alloc&) {
        APPEND_FAIL(SEGPA_ERR_OOM, "append_pages: host allocation failed");
    }

    // device part: one descriptor upload + one scatter launch for the whole batch
    if (!jobs.empty()) {
        DeviceGuard g(c->desc.device);
        cudaStream_t st = (cudaStream_t)cuda_stream;
        Staging& sg = c->append_stage[c->append_turn];
        c->append_turn ^= 1;
        const size_t jobs_bytes = (jobs.size() * sizeof(ScatterJob) + 255) & ~(size_t)255;
        const size_t bytes = jobs_bytes + touched.size() * sizeof(int32_t);
        cudaError_t e = staging_acquire(sg, bytes);
        if (e == cudaSuccess) {
            memcpy(sg.h, jobs.data(), jobs.size() * sizeof(ScatterJob));
            memcpy((uint8_t*)sg.h + jobs_bytes, touched.data(), touched.size() * sizeof(int32_t));
            e = staging_upload(sg, bytes, c->up_stream, st);
        }
        if (e == cudaSuccess && !host_copies.empty()) {
            // the scatter of an earlier host-source batch (possibly on another stream) must have read st_kv
            if (c->st_kv_pending) e = cudaStreamWaitEvent(st, c->st_kv_ev, 0);
            for (size_t h = 0; h < host_copies.size() && e == cudaSuccess; ++h) {
                const HostCopy& hc = host_copies[h];
                uint16_t* kd = c->st_kv + (size_t)hc.off_rows * D;
                uint16_t* vd = c->st_kv + (size_t)(host_rows_total + hc.off_rows) * D;
                if (hc.stride == D) {   // contiguous rows: one plain copy each
                    e = cudaMemcpyAsync(kd, hc.k, (size_t)hc.n * D * 2, cudaMemcpyHostToDevice, st);
                    if (e == cudaSuccess) e = cudaMemcpyAsync(vd, hc.v, (size_t)hc.n * D * 2, cudaMemcpyHostToDevice, st);
                } else {
                    e = cudaMemcpy2DAsync(kd, (size_t)D * 2, hc.k, (size_t)hc.stride * 2, (size_t)D * 2, (size_t)hc.n, cudaMemcpyHostToDevice, st);
                    if (e == cudaSuccess)
                        e = cudaMemcpy2DAsync(vd, (size_t)D * 2, hc.v, (size_t)hc.stride * 2, (size_t)D * 2, (size_t)hc.n, cudaMemcpyHostToDevice, st);
                }
            }
        }
        if (e == cudaSuccess)
            e = launch_scatter_pages(c->k_pool, c->v_pool, (const ScatterJob*)sg.d, (int)jobs.size(),
                                     (const int*)((const uint8_t*)sg.d + jobs_bytes), total_chunks, D, P, st);
        if (e == cudaSuccess) staging_release(sg, st);
        if (e == cudaSuccess && !host_copies.empty()) {
            if (!c->st_kv_ev) e = cudaEventCreateWithFlags(&c->st_kv_ev, cudaEventDisableTiming);
            if (e == cudaSuccess && cudaEventRecord(c->st_kv_ev, st) == cudaSuccess) c->st_kv_pending = true;
        }
        if (e != cudaSuccess) {
            cudaGetLastError();
            APPEND_FAIL(SEGPA_ERR_CUDA, "append_pages: %s", cudaGetErrorString(e));
        }
    }
#undef APPEND_FAIL
    return SEGPA_OK;
}

segpa_status_t segpa_append_pages(segpa_cache_t* c, int32_t layer, int32_t kv_head, int64_t seq_id,
                                  const void* k_src, const void* v_src, int64_t src_row_stride_elems,
                                  int64_t n_tokens, const int32_t* page_ids, int32_t n_page_ids,
                                  void* cuda_stream) {
    segpa_append_req_t r{};
    r.layer = layer;
    r.kv_head = kv_head;
    r.seq_id = seq_id;
    r.k_src = k_src;
    r.v_src = v_src;
    r.src_row_stride_elems = src_row_stride_elems;
    r.n_tokens = n_tokens;
    r.page_ids = page_ids;
    r.n_page_ids = n_page_ids;
    return segpa_append_pages_batch(c, &r, 1, cuda_stream);
}

segpa_status_t segpa_evict_pages(segpa_cache_t* c, int32_t layer, int32_t kv_head, int64_t seq_id,
                                 int32_t first_page_index, int32_t n_pages) {
    if (!c) return fail(SEGPA_ERR_INVALID, "evict_pages: null cache");
    auto it = c->streams.find(StreamKey{layer, kv_head, seq_id});
    if (it == c->streams.end()) return fail(SEGPA_ERR_INVALID, "evict_pages: no stream (%d, %d, %lld)", layer, kv_head, (long long)seq_id);
    StreamRec& rec = it->second;
    const int P = c->desc.page_size;
    if (first_page_index < 0 || n_pages < 1 || (int64_t)first_page_index + n_pages > (int64_t)rec.pages.size())
        return fail(SEGPA_ERR_INVALID, "evict_pages: range [%d, %d) outside the stream's %zu pages", first_page_index, first_page_index + n_pages, rec.pages.size());
    if (rec.slot_len() % P != 0 && (size_t)first_page_index + n_pages == rec.pages.size())
        return fail(SEGPA_ERR_INVALID, "evict_pages: the stream's partial last page cannot be evicted");
    for (int32_t i = 0; i < n_pages; ++i)
        if (rec.pages[(size_t)first_page_index + i] < 0) return fail(SEGPA_ERR_INVALID, "evict_pages: page index %d is already evicted", first_page_index + i);
    for (int32_t i = 0; i < n_pages; ++i) {
        release_page(c, rec.pages[(size_t)first_page_index + i]);
        rec.pages[(size_t)first_page_index + i] = -1;
        ++rec.n_holes;
    }
    return SEGPA_OK;
}

namespace {

// pages covering tokens [first_token, first_token + n) of a stream, uploaded through the append staging
// buffers; *first_slot = slot of first_token inside the first page.  Returns nullptr and sets *why on error.
const int* stage_token_range(segpa_cache* c, const StreamRec& rec, int64_t first_token, int64_t n, bool need_exclusive,
                             cudaStream_t st, int64_t* first_page, Staging** used, const char** why, segpa_status_t* code) {
    const int P = c->desc.page_size;
    *code = SEGPA_ERR_INVALID;
    if (first_token < 0 || n < 1 || first_token + n > rec.kv_len) { *why = "token range outside the stream"; return nullptr; }
    const int64_t pg_lo = rec.slot_of(first_token) / P, pg_hi = rec.slot_of(first_token + n - 1) / P + 1;
    for (int64_t pg = pg_lo; pg < pg_hi; ++pg) {
        const int32_t id = rec.pages[(size_t)pg];
        if (id < 0) { *why = "the range touches an evicted page"; return nullptr; }
        if (need_exclusive && c->refcnt[id] > 1) { *why = "a page of the range is shared with another stream"; return nullptr; }
    }
    Staging& sg = c->append_stage[c->append_turn];
    c->append_turn ^= 1;
    const size_t bytes = (size_t)(pg_hi - pg_lo) * sizeof(int32_t);
    cudaError_t e = staging_acquire(sg, bytes);
    if (e == cudaSuccess) {
        memcpy(sg.h, rec.pages.data() + pg_lo, bytes);
        e = cudaMemcpyAsync(sg.d, sg.h, bytes, cudaMemcpyHostToDevice, st);
    }
    if (e != cudaSuccess) { cudaGetLastError(); *why = cudaGetErrorString(e); *code = SEGPA_ERR_CUDA; return nullptr; }
    *first_page = pg_lo;
    *used = &sg;
    return (const int*)sg.d;
}

}  // namespace

segpa_status_t segpa_rope_align_batch(segpa_cache_t* c, const segpa_rope_req_t* reqs, int32_t n, double rope_base,
                                      void* cuda_stream) {
    if (!c || !reqs) return fail(SEGPA_ERR_INVALID, "rope_align: null argument");
    if (n < 1) return fail(SEGPA_ERR_INVALID, "rope_align: batch size %d < 1", n);
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "rope_align: planning-only cache has no device");
    if (!(rope_base > 1.0)) return fail(SEGPA_ERR_INVALID, "rope_align: rope_base must be > 1");
    const int D = c->desc.head_dim, P = c->desc.page_size;
    // Pass 1: streams, ranges, overlaps; count the jobs (pieces contiguous in slot space) and the page ids they list.
    // a token may be rotated once per batch: overlapping ranges would make the result order-dependent
    struct Rng { const StreamRec* rec; int64_t lo, hi; };
    std::vector<Rng> seen;
    size_t n_jobs = 0, n_ids = 0;
    try {
        seen.reserve((size_t)n);
        for (int32_t i = 0; i < n; ++i) {
            const segpa_rope_req_t& r = reqs[i];
            auto it = c->streams.find(StreamKey{r.layer, r.kv_head, r.seq_id});
            if (it == c->streams.end()) return fail(SEGPA_ERR_INVALID, "rope_align[%d]: no stream (%d, %d, %lld)", i, r.layer, r.kv_head, (long long)r.seq_id);
            const StreamRec& rec = it->second;
            if (r.first_token < 0 || r.n_tokens < 1 || r.first_token + r.n_tokens > rec.kv_len)
                return fail(SEGPA_ERR_INVALID, "rope_align[%d]: token range outside the stream", i);
            for (const Rng& g : seen)
                if (g.rec == &rec && r.first_token < g.hi && g.lo < r.first_token + r.n_tokens)
                    return fail(SEGPA_ERR_INVALID, "rope_align[%d]: token range overlaps an earlier request of the batch", i);
            seen.push_back(Rng{&rec, r.first_token, r.first_token + r.n_tokens});
            for_each_piece(rec, r.first_token, r.n_tokens, [&](int64_t, int64_t n_piece, int64_t slot_lo) {
                ++n_jobs;
                n_ids += (size_t)((slot_lo + n_piece - 1) / P - slot_lo / P + 1);
            });
        }
    } catch (const std::bad_alloc&) {
        return fail(SEGPA_ERR_OOM, "rope_align: host allocation failed");
    }
    DeviceGuard g(c->desc.device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Staging& sg = c->append_stage[c->append_turn];
    c->append_turn ^= 1;
    auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
    const size_t off_ids = al(n_jobs * sizeof(RopeJob));
    const size_t bytes = off_ids + n_ids * sizeof(int32_t);
    cudaError_t e = staging_acquire(sg, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "rope_align: %s", cudaGetErrorString(e)); }
    // Pass 2: the jobs and their page ids are written straight into the pinned staging buffer; every page is checked on
    // the way (evicted: id < 0; shared with another stream: rotating it would move that stream's keys too).  The
    // reference counts are read in the (random) order of the ids: fetched ahead.
    RopeJob* jobs = (RopeJob*)sg.h;
    int32_t* ids = (int32_t*)((uint8_t*)sg.h + off_ids);
    size_t nj = 0, ni = 0;
    long long total_units = 0;                     // CTAs of the rotation kernel: kRopeUnitChunks half-row chunks of one job each
    int32_t min_id = 0, max_ref = 0;
    const int32_t* refcnt = c->refcnt.data();
    const int32_t n_pool = (int32_t)c->desc.num_pages;
    for (int32_t i = 0; i < n; ++i) {
        const segpa_rope_req_t& r = reqs[i];
        const StreamRec& rec = *seen[(size_t)i].rec;
        for_each_piece(rec, r.first_token, r.n_tokens, [&](int64_t, int64_t n_piece, int64_t slot_lo) {
            RopeJob jb{};
            jb.unit_begin = (int)total_units;
            jb.page_off = (long long)ni;
            jb.n_tokens = n_piece;
            jb.delta_pos = r.delta_pos;   // R(p_on) R(p_off)^-1 = R(delta); the per-pair cos / sin are formed on the device in fp64
            jb.first_slot = (int)(slot_lo % P);
            const int32_t* pg = rec.pages.data() + slot_lo / P;
            const int64_t np = (slot_lo + n_piece - 1) / P - slot_lo / P + 1;
            if (c->n_shared_pages == 0 && rec.n_holes == 0) {
                // no page of the cache is shared and the stream has no hole: nothing to check page by page
                memcpy(ids + ni, pg, (size_t)np * sizeof(int32_t));
                ni += (size_t)np;
            } else
            for (int64_t k = 0; k < np; ++k) {
                const int32_t id = pg[k];
                if (k + 16 < np && (uint32_t)pg[k + 16] < (uint32_t)n_pool) __builtin_prefetch(refcnt + pg[k + 16]);
                min_id = std::min(min_id, id);
                max_ref = std::max(max_ref, refcnt[id < 0 ? 0 : id]);
                ids[ni++] = id;
            }
            total_units += (n_piece * (D >> 4) + kRopeUnitChunks - 1) / kRopeUnitChunks;
            jobs[nj++] = jb;
        });
    }
    if (min_id < 0 || max_ref > 1) {   // (the search for the message only on failure; nothing has been launched)
        for (int32_t i = 0; i < n; ++i) {
            const segpa_rope_req_t& r = reqs[i];
            const StreamRec& rec = *seen[(size_t)i].rec;
            const int64_t pg_lo = rec.slot_of(r.first_token) / P, pg_hi = rec.slot_of(r.first_token + r.n_tokens - 1) / P + 1;
            for (int64_t pg = pg_lo; pg < pg_hi; ++pg) {
                const int32_t id = rec.pages[(size_t)pg];
                if (id < 0) return fail(SEGPA_ERR_INVALID, "rope_align[%d]: the range touches an evicted page", i);
                if (c->refcnt[id] > 1) return fail(SEGPA_ERR_INVALID, "rope_align[%d]: page %d is shared with another stream", i, id);
            }
        }
        return fail(SEGPA_ERR_INVALID, "rope_align: a page of a range is evicted or shared with another stream");
    }
    e = staging_upload(sg, bytes, c->up_stream, st);
    if (e == cudaSuccess)
        e = launch_rope_align(c->k_pool, (const RopeJob*)sg.d, (int)n_jobs, (const int*)((const uint8_t*)sg.d + off_ids),
                              (int)total_units, rope_base, D, P, st);
    if (e == cudaSuccess) staging_release(sg, st);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "rope_align: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}

segpa_status_t segpa_rope_align(segpa_cache_t* c, int32_t layer, int32_t kv_head, int64_t seq_id, int64_t first_token,
                                int64_t n_tokens, int64_t delta_pos, double rope_base, void* cuda_stream) {
    segpa_rope_req_t r{};
    r.layer = layer;
    r.kv_head = kv_head;
    r.seq_id = seq_id;
    r.first_token = first_token;
    r.n_tokens = n_tokens;
    r.delta_pos = delta_pos;
    return segpa_rope_align_batch(c, &r, 1, rope_base, cuda_stream);
}

segpa_status_t segpa_gather_rows(segpa_cache_t* c, int32_t layer, int32_t kv_head, int64_t seq_id, int64_t first_token,
                                 int64_t n_tokens, void* k_dst, void* v_dst, int64_t dst_row_stride_elems, void* cuda_stream) {
    if (!c) return fail(SEGPA_ERR_INVALID, "gather_rows: null cache");
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "gather_rows: planning-only cache has no device");
    const int D = c->desc.head_dim;
    if (dst_row_stride_elems < D || (dst_row_stride_elems % 8) || ((uintptr_t)k_dst % 16) || ((uintptr_t)v_dst % 16))
        return fail(SEGPA_ERR_INVALID, "gather_rows: destinations must be 16-byte aligned with a row stride >= head_dim, multiple of 8 elements");
    auto it = c->streams.find(StreamKey{layer, kv_head, seq_id});
    if (it == c->streams.end()) return fail(SEGPA_ERR_INVALID, "gather_rows: no stream (%d, %d, %lld)", layer, kv_head, (long long)seq_id);
    DeviceGuard g(c->desc.device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int64_t first_page = 0;
    Staging* used = nullptr;
    const char* why = "";
    segpa_status_t code = SEGPA_OK;
    const StreamRec& rec = it->second;
    const int* ids = stage_token_range(c, rec, first_token, n_tokens, false, st, &first_page, &used, &why, &code);
    if (!ids) return fail(code, "gather_rows: %s", why);
    const int P = c->desc.page_size;
    cudaError_t e = cudaSuccess;
    for_each_piece(rec, first_token, n_tokens, [&](int64_t tok_lo, int64_t n_piece, int64_t slot_lo) {
        if (e != cudaSuccess) return;
        uint16_t* kd = k_dst ? (uint16_t*)k_dst + (tok_lo - first_token) * dst_row_stride_elems : nullptr;
        uint16_t* vd = v_dst ? (uint16_t*)v_dst + (tok_lo - first_token) * dst_row_stride_elems : nullptr;
        e = launch_gather_rows(c->k_pool, c->v_pool, ids + (slot_lo / P - first_page), (int)(slot_lo % P), n_piece, kd, vd,
                               dst_row_stride_elems, D, P, st);
    });
    staging_release(*used, st);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "gather_rows: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}

segpa_status_t segpa_gather_rows_noalloc(segpa_cache_t* c, int32_t layer, int32_t kv_head, int64_t seq_id, int64_t first_token,
                                         int64_t n_tokens, void* k_dst, void* v_dst, int64_t dst_row_stride_elems,
                                         void* cuda_stream) {
    if (!c) return fail(SEGPA_ERR_INVALID, "gather_rows_noalloc: null cache");
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "gather_rows_noalloc: planning-only cache has no device");
    const int D = c->desc.head_dim, P = c->desc.page_size;
    if (!k_dst && !v_dst) return fail(SEGPA_ERR_INVALID, "gather_rows_noalloc: give k_dst, v_dst or both");
    if (dst_row_stride_elems < D || (dst_row_stride_elems % 8) || ((uintptr_t)k_dst % 16) || ((uintptr_t)v_dst % 16))
        return fail(SEGPA_ERR_INVALID, "gather_rows_noalloc: destinations must be 16-byte aligned with a row stride >= head_dim, multiple of 8 elements");
    auto it = c->streams.find(StreamKey{layer, kv_head, seq_id});
    if (it == c->streams.end()) return fail(SEGPA_ERR_INVALID, "gather_rows_noalloc: no stream (%d, %d, %lld)", layer, kv_head, (long long)seq_id);
    const StreamRec& rec = it->second;
    if (first_token < 0 || n_tokens < 1 || first_token + n_tokens > rec.kv_len)
        return fail(SEGPA_ERR_INVALID, "gather_rows_noalloc: token range outside the stream");
    const int64_t pg_lo = rec.slot_of(first_token) / P, pg_hi = rec.slot_of(first_token + n_tokens - 1) / P + 1;
    if (pg_hi - pg_lo > SEGPA_NOALLOC_MAX_PAGES)
        return fail(SEGPA_ERR_INVALID, "gather_rows_noalloc: the range covers %lld pages; the fixed scratch of this entry point holds %d "
                    "(%lld tokens at this page size): split the range, or use segpa_gather_rows", (long long)(pg_hi - pg_lo),
                    SEGPA_NOALLOC_MAX_PAGES, (long long)SEGPA_NOALLOC_MAX_PAGES * P);
    for (int64_t pg = pg_lo; pg < pg_hi; ++pg)
        if (rec.pages[(size_t)pg] < 0) return fail(SEGPA_ERR_INVALID, "gather_rows_noalloc: the range touches an evicted page");
    DeviceGuard g(c->desc.device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int* ids = nullptr;
    cudaError_t e = noalloc_stage_page_ids(rec.pages.data() + pg_lo, (int)(pg_hi - pg_lo), st, &ids);
    for_each_piece(rec, first_token, n_tokens, [&](int64_t tok_lo, int64_t n_piece, int64_t slot_lo) {
        if (e != cudaSuccess) return;
        uint16_t* kd = k_dst ? (uint16_t*)k_dst + (tok_lo - first_token) * dst_row_stride_elems : nullptr;
        uint16_t* vd = v_dst ? (uint16_t*)v_dst + (tok_lo - first_token) * dst_row_stride_elems : nullptr;
        e = launch_gather_rows(c->k_pool, c->v_pool, ids + (slot_lo / P - pg_lo), (int)(slot_lo % P), n_piece, kd, vd,
                               dst_row_stride_elems, D, P, st);
    });
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "gather_rows_noalloc: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}

segpa_status_t segpa_clear_streams(segpa_cache_t* c) {
    if (!c) return fail(SEGPA_ERR_INVALID, "clear_streams: null cache");
    c->streams.clear();
    std::fill(c->refcnt.begin(), c->refcnt.end(), 0);
    c->n_shared_pages = 0;
    c->free_list.resize((size_t)c->desc.num_pages);
    for (int64_t i = 0; i < c->desc.num_pages; ++i) c->free_list[(size_t)i] = (int32_t)(c->desc.num_pages - 1 - i);
    std::fill(c->in_free.begin(), c->in_free.end(), 1);
    c->n_free = c->desc.num_pages;
    return SEGPA_OK;
}

segpa_status_t segpa_free_stream(segpa_cache_t* c, int32_t layer, int32_t kv_head, int64_t seq_id) {
    if (!c) return fail(SEGPA_ERR_INVALID, "free_stream: null cache");
    auto it = c->streams.find(StreamKey{layer, kv_head, seq_id});
    if (it == c->streams.end()) return fail(SEGPA_ERR_INVALID, "free_stream: no stream (%d, %d, %lld)", layer, kv_head, (long long)seq_id);
    for (auto id : it->second.pages)
        if (id >= 0) release_page(c, id);
    c->streams.erase(it);
    return SEGPA_OK;
}

segpa_status_t segpa_stream_info(const segpa_cache_t* c, int32_t layer, int32_t kv_head, int64_t seq_id,
                                 int64_t* kv_len, int32_t* n_pages, int32_t* page_ids_out, int32_t cap) {
    if (!c) return fail(SEGPA_ERR_INVALID, "stream_info: null cache");
    auto it = c->streams.find(StreamKey{layer, kv_head, seq_id});
    if (it == c->streams.end()) return fail(SEGPA_ERR_INVALID, "stream_info: no stream (%d, %d, %lld)", layer, kv_head, (long long)seq_id);
    if (kv_len) *kv_len = it->second.kv_len;
    if (n_pages) *n_pages = (int32_t)it->second.pages.size();
    if (page_ids_out)
        for (int32_t i = 0; i < cap && i < (int32_t)it->second.pages.size(); ++i) page_ids_out[i] = it->second.pages[i];
    return SEGPA_OK;
}

segpa_status_t segpa_pool_stats(const segpa_cache_t* c, int64_t* in_use, int64_t* n_free) {
    if (!c) return fail(SEGPA_ERR_INVALID, "pool_stats: null cache");
    if (in_use) *in_use = c->desc.num_pages - c->n_free;
    if (n_free) *n_free = c->n_free;
    return SEGPA_OK;
}

// ---------------------------------------------------------------------------------------------
// Alg. 2 lines 1-14 + the tile scheduler
// ---------------------------------------------------------------------------------------------
segpa_status_t segpa_build_segments(segpa_cache_t* c, int32_t layer, const segpa_segment_req_t* reqs,
                                    int32_t n, segpa_segments_t** out, void* cuda_stream) {
    if (!c || !reqs || !out) return fail(SEGPA_ERR_INVALID, "build_segments: null argument");
    *out = nullptr;
    if (n < 1) return fail(SEGPA_ERR_INVALID, "build_segments: n %d < 1", n);
    if (layer < 0 || layer >= c->desc.num_layers) return fail(SEGPA_ERR_INVALID, "build_segments: layer %d out of range", layer);
    const int P = c->desc.page_size, G = c->G, D = c->desc.head_dim;
    const int ppb = kBlockKeys / P;
    const int32_t zero_page = (int32_t)c->desc.num_pages;
    const int tiles_per_item = (c->kernel_kind == 1) ? c->tiles_per_item : 1;
    const int TT = kTileRows / G;               // tokens per 128-row tile (GQA packing)
    const int item_tok = TT * tiles_per_item;

    segpa_segments* S = nullptr;
    if (!c->free_seg_objs.empty()) {
        S = c->free_seg_objs.back();
        c->free_seg_objs.pop_back();
    } else {
        S = new (std::nothrow) segpa_segments();
        if (!S) return fail(SEGPA_ERR_OOM, "build_segments: host allocation failed");
    }
    S->cache = c;
    S->layer = layer;
    S->tiles_per_item = tiles_per_item;
    using TileTmp = PlanTile;
    PlanScratch& ps = c->plan;
    std::vector<TileTmp>& tiles = ps.tiles;
    tiles.clear();
    int64_t q_rows = 0, pairs = 0, vis_tokens = 0;
    try {
        S->reqs.assign(reqs, reqs + n);
        S->segs.reserve((size_t)n);
        {
            size_t n_tiles_max = 0;
            for (int32_t s = 0; s < n; ++s) n_tiles_max += (size_t)(std::max(reqs[s].q_len, 1) + item_tok - 1) / (size_t)item_tok;
            tiles.reserve(n_tiles_max);
        }
        // validation + per-segment metadata
        using Iv = PlanIv;
        std::vector<Iv>& ivs = ps.ivs;
        ivs.clear();
        for (int32_t s = 0; s < n; ++s) {
            const segpa_segment_req_t& r = reqs[s];
            if (r.kv_head < 0 || r.kv_head >= c->desc.num_kv_heads) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: kv_head %d out of range", s, r.kv_head); }
            auto it = c->streams.find(StreamKey{layer, r.kv_head, r.seq_id});
            if (it == c->streams.end()) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: no stream (layer %d, kv_head %d, seq %lld)", s, layer, r.kv_head, (long long)r.seq_id); }
            const StreamRec& rec = it->second;
            if (r.head_class != SEGPA_GLOBAL && r.head_class != SEGPA_LOCAL) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: bad head_class %d", s, r.head_class); }
            if (r.q_len < 1 || r.q_len > rec.kv_len) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: q_len %d not in [1, kv_len=%lld]", s, r.q_len, (long long)rec.kv_len); }
            if (r.head_class == SEGPA_LOCAL && r.window < 1) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: LOCAL window %d < 1", s, r.window); }
            if (r.q_row_start < 0) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: negative q_row_start", s); }
            if (r.n_sink < 0) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: negative n_sink", s); }
            ivs.push_back(Iv{r.kv_head, r.q_row_start, r.q_row_start + r.q_len});

            const int64_t kv_len = rec.kv_len;
            const int64_t W = (r.head_class == SEGPA_GLOBAL) ? (int64_t)INT32_MAX / 2 : r.window;
            // Positions are token indices; pages and KV blocks are laid out in slot space (slot = token + the unused slots
            // behind earlier head segments' tails; the identity for a dense stream)
            auto slot_of = [&rec](int64_t tok) { return rec.pads.empty() ? tok : rec.slot_of(tok); };
            // Alg. 2 lines 6-10: visible positions of the whole segment
            const int64_t vis_lo = std::max<int64_t>(0, kv_len - r.q_len - W + 1);
            const int64_t vis_lo_slot = slot_of(vis_lo), last_slot = slot_of(kv_len - 1);
            // S_sink: the first n_sink tokens stay visible to a LOCAL head; they matter only when
            // some query's window starts after position 0 (the last query's does iff kv_len > W)
            const int64_t ns = (r.head_class == SEGPA_LOCAL) ? std::min<int64_t>(r.n_sink, kv_len) : 0;
            const bool has_sink = ns > 0 && kv_len > W;
            const int64_t sink_slots = (has_sink && std::min(ns, vis_lo) > 0) ? slot_of(std::min(ns, vis_lo) - 1) + 1 : 0;
            const int64_t sink_pages = has_sink ? std::min(cdiv(sink_slots, P), vis_lo_slot / P) : 0;   // pages wholly before the window's first page
            const int64_t seg_kb_lo = has_sink ? 0 : vis_lo_slot / kBlockKeys;
            const int64_t seg_kb_hi = last_slot / kBlockKeys + 1;
            const int64_t first_vis_page = vis_lo_slot / P;
            const int64_t n_stream_pages = (int64_t)rec.pages.size();
            SegDev sd{};
            sd.q_row_start = r.q_row_start;
            sd.page_off = (long long)S->pages.size();
            sd.q_len = r.q_len;
            sd.kv_len = (int)kv_len;
            sd.head_class = r.head_class;
            sd.window = (int)W;
            sd.n_sink = has_sink ? (int)ns : 0;
            sd.kv_head = r.kv_head;
            sd.first_page = (int)(seg_kb_lo * ppb);
            sd.n_pages_listed = (int)((seg_kb_hi - seg_kb_lo) * ppb);
            sd.pad_off = (int)S->pads.size();
            sd.n_pads = (int)rec.pads.size();
            for (const PadPoint& pp : rec.pads) S->pads.push_back(PadDev{(int)pp.tok, (int)pp.pad});
            if (!rec.pads.empty()) S->has_ragged = true;
            // Alg. 2 line 12: Translate(T_page, U_h): sink pages and recent-window pages (lines 9-10); invisible
            // pages (the evicted middle) and absent ones -> the zero page, never read
            {
                const int64_t lst_lo = sd.first_page, lst_hi = sd.first_page + sd.n_pages_listed;
                const int64_t vis_a = std::max(lst_lo, first_vis_page), vis_b = std::min(lst_hi, n_stream_pages);
                // (holes are negative ids: a branch-free minimum first, the search for the message only on failure)
                int32_t min_id = 0;
                for (int64_t pg = 0; pg < sink_pages; ++pg) min_id = std::min(min_id, rec.pages[(size_t)pg]);
                for (int64_t pg = vis_a; pg < vis_b; ++pg) min_id = std::min(min_id, rec.pages[(size_t)pg]);
                if (min_id < 0) {
                    for (int64_t pg = 0; pg < sink_pages; ++pg)
                        if (rec.pages[(size_t)pg] < 0) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: sink page %lld of the stream was evicted", s, (long long)pg); }
                    for (int64_t pg = vis_a; pg < vis_b; ++pg)
                        if (rec.pages[(size_t)pg] < 0) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: segment %d: visible page %lld of the stream was evicted", s, (long long)pg); }
                }
                S->pages.insert(S->pages.end(), rec.pages.begin(), rec.pages.begin() + sink_pages);
                S->pages.insert(S->pages.end(), (size_t)(vis_a - lst_lo - sink_pages), zero_page);
                S->pages.insert(S->pages.end(), rec.pages.begin() + vis_a, rec.pages.begin() + vis_b);
                S->pages.insert(S->pages.end(), (size_t)(lst_hi - vis_b), zero_page);
            }
            S->segs.push_back(sd);
            if (S->mass_off.empty()) S->mass_off.push_back(0);
            S->mass_off.push_back(S->mass_off.back() + cdiv(kv_len, kBlockKeys) * kBlockKeys);
            vis_tokens += last_slot + 1 - first_vis_page * P + sink_pages * P;
            q_rows = std::max<int64_t>(q_rows, r.q_row_start + r.q_len);
            pairs += visible_pairs(kv_len - r.q_len, kv_len - 1, W);
            if (has_sink) {   // sink keys not already inside the window: sum over the queries i of clamp(i - W + 1, 0, ns)
                const int64_t a = kv_len - r.q_len - W + 1, b = kv_len - W;          // x = i - W + 1 runs over [a, b]
                const int64_t lo = std::max<int64_t>(a, 1), mid = std::min<int64_t>(b, ns);   // x in [lo, mid] contributes x, x > ns contributes ns
                if (mid >= lo) pairs += (lo + mid) * (mid - lo + 1) / 2;
                if (b > ns) pairs += (b - std::max<int64_t>(a, ns + 1) + 1) * ns;
            }
            // tiles: exactly the KV blocks (of slots) the tile's rows attend to
            for (int64_t t0 = 0; t0 < r.q_len; t0 += item_tok) {
                const int64_t n_tok = std::min<int64_t>(item_tok, r.q_len - t0);
                const int64_t i0 = kv_len - r.q_len + t0, i1 = i0 + n_tok - 1;
                const int64_t lo = std::max<int64_t>(0, i0 - W + 1);
                TileTmp tt{s, (int)t0, (int)n_tok, (int)(slot_of(lo) / kBlockKeys), (int)(slot_of(i1) / kBlockKeys + 1), 0, false};
                tt.cost = tt.kb_hi - tt.kb_lo;
                if (has_sink) {
                    // two KV block ranges: sink blocks [0, sb) then the window blocks; one range when they touch
                    const int sb = (int)cdiv(slot_of(std::min(ns, i1 + 1) - 1) + 1, kBlockKeys);
                    tt.cost = (sb >= tt.kb_lo) ? tt.kb_hi : sb + tt.kb_hi - tt.kb_lo;
                    tt.kb_lo = 0;
                    tt.sink = true;
                }
                tiles.push_back(tt);
            }
        }
        // overlap check on (row, head): same kv_head (hence same q heads) and intersecting rows
        std::sort(ivs.begin(), ivs.end(), [](const Iv& a, const Iv& b) { return a.kv_head != b.kv_head ? a.kv_head < b.kv_head : a.lo < b.lo; });
        for (size_t i = 1; i < ivs.size(); ++i)
            if (ivs[i].kv_head == ivs[i - 1].kv_head && ivs[i].lo < ivs[i - 1].hi) { delete S; return fail(SEGPA_ERR_INVALID, "build_segments: two segments of kv_head %d overlap on rows [%lld, %lld)", ivs[i].kv_head, (long long)ivs[i].lo, (long long)std::min(ivs[i].hi, ivs[i - 1].hi)); }

        // scheduler: split long tiles along KV when the grid would be unbalanced (decode-shaped global heads),
        // then assign the items to the CTAs of the persistent grid (LPT, below)
        int64_t total_cost = 0;
        for (auto& t : tiles) total_cost += t.cost;
        const int64_t chunk = std::max<int64_t>(8, cdiv(total_cost, (int64_t)c->num_sms * 4));
        // Decode-shaped tiles (a few rows against a long stream, HBM-bound) are cut coarser: pieces of about one CTA's
        // share of the whole plan.  Every piece costs a Q load, a drain of 2 x 128 TMEM lanes for a handful of valid rows
        // and one more partial for the combine pass to read, and LPT still balances the grid with ~2 pieces per CTA
        // (measured: fig9-decode-128k 92 -> 65 us per layer, cfg4d 99 -> 93 us against pieces of a quarter of that size).
        const int64_t chunk_dec = std::max<int64_t>(8, cdiv(total_cost, (int64_t)c->num_sms));
        int n_split_tiles = 0, n_slots = 0;
        S->items.reserve(tiles.size() + (size_t)c->num_sms * 8);
        S->item_meta.reserve(tiles.size() + (size_t)c->num_sms * 8);
        for (size_t ti = 0; ti < tiles.size(); ++ti) {
            const TileTmp& t = tiles[ti];
            const int cost = t.cost;
            int parts = 1;
            const bool dec = S->reqs[(size_t)t.seg].q_len <= TT;
            const int64_t ch = dec ? chunk_dec : chunk;
            if (cost > (dec ? ch + ch / 8 : ch + ch / 2) && !t.sink) parts = (int)cdiv(cost, ch);   // (sink items are not cut along KV)
            // Decode-shaped segment (all its rows fit the first of the item's two tile slots; the short tail item of a
            // long prefill segment does not count: it is not worth a combine pass): run it STRIDED -- the
            // two slots take alternate KV blocks of the same rows as two independent chains, each writing a
            // partial that the combine kernel merges -- so the second slot is not left idle.
            const bool strided = tiles_per_item == 2 && S->reqs[(size_t)t.seg].q_len <= TT && cost >= 2 && c->kernel_kind == 1;
            if (parts > 1) ++n_split_tiles;
            if (parts > 1 || strided)
                S->combs.push_back(CombDev{t.seg, t.t0, t.n_tok, n_slots, parts, strided ? 1 : 0, 0, 0});
            for (int p = 0; p < parts; ++p) {
                // (parts == 1, nearly every tile: no divisions on this path)
                const int lo = (t.sink || parts == 1) ? t.kb_lo : t.kb_lo + (int)((int64_t)cost * p / parts);
                const int hi = (t.sink || parts == 1) ? t.kb_hi : t.kb_lo + (int)((int64_t)cost * (p + 1) / parts);
                const int slot = (parts > 1 || strided) ? n_slots++ : -1;
                ItemDev itd{t.seg, t.t0, t.n_tok, lo, hi, slot, strided ? 1 : 0, t.sink ? t.cost : hi - lo, {{0, 0, 0}, {0, 0, 0}}, {0, 0}};
                const segpa_segment_req_t& rq = S->reqs[(size_t)t.seg];
                const StreamRec& srec = c->streams.find(StreamKey{layer, rq.kv_head, rq.seq_id})->second;
                if (!srec.pads.empty()) {   // ragged stream: the slots of the tiles' first / last visible key and last sink key
                    const SegDev& sdv = S->segs[(size_t)t.seg];
                    for (int tl = 0; tl < 2; ++tl) {
                        const int64_t tok_lo = t.t0 + (int64_t)tl * TT, tok_hi = std::min<int64_t>(t.t0 + t.n_tok, tok_lo + TT);
                        if (tok_hi <= tok_lo) continue;
                        const int64_t i0 = srec.kv_len - rq.q_len + tok_lo, i1 = srec.kv_len - rq.q_len + tok_hi - 1;
                        itd.slots[tl][0] = (int)srec.slot_of(std::max<int64_t>(0, i0 - sdv.window + 1));
                        itd.slots[tl][1] = (int)srec.slot_of(i1);
                        itd.slots[tl][2] = sdv.n_sink > 0 ? (int)srec.slot_of(std::min<int64_t>(sdv.n_sink, i1 + 1) - 1) : -1;
                    }
                }
                S->items.push_back(itd);
                S->item_meta.push_back(segpa_segments::ItemMeta{(int32_t)ti, parts > 1 ? p : -1, parts});
            }
        }
        const int64_t kv_blocks = lpt_assign(ps, S->items, &S->item_meta, c->num_sms, S->cta_off);
        S->narrow = c->kernel_kind == 1;
        for (const ItemDev& itd : S->items) S->narrow = S->narrow && itd.n_tok * G <= 16;

        segpa_plan_stats_t& stt = S->stats;
        stt.n_segments = n;
        stt.n_tiles = (int32_t)tiles.size();
        stt.n_items = (int32_t)S->items.size();
        stt.n_split_tiles = n_split_tiles;
        stt.tile_tokens = TT;
        stt.block_keys = kBlockKeys;
        stt.kv_blocks = kv_blocks;
        stt.attended_pairs = pairs * G;
        stt.q_rows = q_rows;
        stt.visible_kv_tokens = vis_tokens;
        stt.workspace_bytes = (int64_t)n_slots * kTileRows * tiles_per_item * (D + 2) * 4;
    } catch (const std::bad_alloc&) {
        delete S;
        return fail(SEGPA_ERR_OOM, "build_segments: host allocation failed");
    }

    if (!c->planning_only) {
        DeviceGuard g(c->desc.device);
        cudaStream_t st = (cudaStream_t)cuda_stream;
        auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
        S->off_segs = 0;
        S->off_items = al(S->off_segs + S->segs.size() * sizeof(SegDev));
        S->off_pages = al(S->off_items + S->items.size() * sizeof(ItemDev));
        S->off_combs = al(S->off_pages + S->pages.size() * sizeof(int32_t));
        S->off_cta = al(S->off_combs + std::max<size_t>(1, S->combs.size()) * sizeof(CombDev));
        S->off_pads = al(S->off_cta + S->cta_off.size() * sizeof(int32_t));
        const size_t blob_bytes = al(S->off_pads + std::max<size_t>(1, S->pads.size()) * sizeof(PadDev));
        // device storage: recycled from the cache's free list (no cudaMalloc / cudaMallocHost in steady state)
        // Oldest first, and only one whose last use has completed on the device: a caller that enqueues steps
        // back to back (host planning of step k+1 under the kernels of step k) must not be made to wait here.
        // While none is ready the cache grows, up to twice the live objects + 2; past that the oldest is waited for.
        SegBuf* B = nullptr;
        for (size_t i = 0; i < c->free_bufs.size() && !B; ++i) {
            SegBuf* cand = c->free_bufs[i];
            if (!cand->blob.pending || cudaEventQuery(cand->blob.ev) == cudaSuccess) {
                B = cand;
                c->free_bufs.erase(c->free_bufs.begin() + (long)i);
            }
        }
        cudaGetLastError();   // (cudaErrorNotReady from the queries is not an error)
        if (!B && !c->free_bufs.empty() && c->n_seg_bufs >= 2 * (c->seg_objs.size() + 1) + 2) {
            B = c->free_bufs.front();
            c->free_bufs.erase(c->free_bufs.begin());
        }
        if (!B) {
            B = new (std::nothrow) SegBuf();
            if (!B) { delete S; return fail(SEGPA_ERR_OOM, "build_segments: host allocation failed"); }
            ++c->n_seg_bufs;
        }
        S->buf = B;
        S->last_stream = st;
        cudaError_t e = staging_acquire(B->blob, blob_bytes);
        if (e == cudaSuccess && !B->counter) e = cudaMalloc((void**)&B->counter, 256);
        const size_t ws_rows = (size_t)S->stats.workspace_bytes / ((size_t)(D + 2) * 4);
        if (e == cudaSuccess && ws_rows > B->ws_rows) {
            if (B->ws_o) cudaFree(B->ws_o);
            if (B->ws_ml) cudaFree(B->ws_ml);
            B->ws_o = B->ws_ml = nullptr;
            B->ws_rows = 0;
            e = cudaMalloc((void**)&B->ws_o, ws_rows * D * 4);
            if (e == cudaSuccess) e = cudaMalloc((void**)&B->ws_ml, ws_rows * 2 * 4);
            if (e == cudaSuccess) B->ws_rows = ws_rows;
        }
        if (e != cudaSuccess) {
            cudaGetLastError();
            free_segments_obj(c, S);
            return fail(e == cudaErrorMemoryAllocation ? SEGPA_ERR_OOM : SEGPA_ERR_CUDA, "build_segments: %s", cudaGetErrorString(e));
        }
        uint8_t* hb = (uint8_t*)B->blob.h;
        memcpy(hb + S->off_segs, S->segs.data(), S->segs.size() * sizeof(SegDev));
        memcpy(hb + S->off_items, S->items.data(), S->items.size() * sizeof(ItemDev));
        memcpy(hb + S->off_pages, S->pages.data(), S->pages.size() * sizeof(int32_t));
        if (!S->combs.empty()) memcpy(hb + S->off_combs, S->combs.data(), S->combs.size() * sizeof(CombDev));
        memcpy(hb + S->off_cta, S->cta_off.data(), S->cta_off.size() * sizeof(int32_t));
        if (!S->pads.empty()) memcpy(hb + S->off_pads, S->pads.data(), S->pads.size() * sizeof(PadDev));
        e = staging_upload(B->blob, blob_bytes, c->up_stream, st);
        if (e != cudaSuccess) {
            cudaGetLastError();
            free_segments_obj(c, S);
            return fail(SEGPA_ERR_CUDA, "build_segments: upload failed: %s", cudaGetErrorString(e));
        }
    }
    c->seg_objs.push_back(S);
    *out = S;
    return SEGPA_OK;
}

segpa_status_t segpa_free_segments(segpa_cache_t* c, segpa_segments_t* s) {
    if (!c || !s) return fail(SEGPA_ERR_INVALID, "free_segments: null argument");
    auto it = std::find(c->seg_objs.begin(), c->seg_objs.end(), s);
    if (it == c->seg_objs.end()) return fail(SEGPA_ERR_STATE, "free_segments: not owned by this cache");
    c->seg_objs.erase(it);
    DeviceGuard g(c->desc.device);
    free_segments_obj(c, s);
    return SEGPA_OK;
}

segpa_status_t segpa_segments_stats(const segpa_segments_t* s, segpa_plan_stats_t* out) {
    if (!s || !out) return fail(SEGPA_ERR_INVALID, "segments_stats: null argument");
    *out = s->stats;
    return SEGPA_OK;
}

segpa_status_t segpa_segments_items(const segpa_segments_t* s, segpa_item_t* items_out, int32_t cap, int32_t* n_out) {
    if (!s) return fail(SEGPA_ERR_INVALID, "segments_items: null argument");
    if (n_out) *n_out = (int32_t)s->items.size();
    if (items_out) {
        int32_t cta = 0;
        for (int32_t i = 0; i < cap && i < (int32_t)s->items.size(); ++i) {
            while (cta + 1 < (int32_t)s->cta_off.size() && i >= s->cta_off[(size_t)cta + 1]) ++cta;
            const ItemDev& it = s->items[(size_t)i];
            const segpa_segments::ItemMeta& m = s->item_meta[(size_t)i];
            items_out[i] = segpa_item_t{it.seg, it.t0, it.n_tok, it.kb_lo, it.kb_hi, m.split, m.n_splits, m.tile, cta, 0};
        }
    }
    return SEGPA_OK;
}

segpa_status_t segpa_segments_pages(const segpa_segments_t* s, int32_t segment, int32_t* first_page_index,
                                    int32_t* page_ids_out, int32_t cap, int32_t* n_out) {
    if (!s || segment < 0 || segment >= (int32_t)s->segs.size()) return fail(SEGPA_ERR_INVALID, "segments_pages: bad argument");
    const SegDev& sd = s->segs[(size_t)segment];
    if (first_page_index) *first_page_index = sd.first_page;
    if (n_out) *n_out = sd.n_pages_listed;
    if (page_ids_out)
        for (int32_t i = 0; i < cap && i < sd.n_pages_listed; ++i) page_ids_out[i] = s->pages[(size_t)sd.page_off + i];
    return SEGPA_OK;
}

// ---------------------------------------------------------------------------------------------
// Alg. 2 lines 15-16
// ---------------------------------------------------------------------------------------------
segpa_status_t segpa_attention_fwd(segpa_cache_t* c, const segpa_segments_t* s, const void* q,
                                   int64_t q_row_stride, float scale, void* out, int64_t out_row_stride,
                                   float* lse, int64_t lse_stride, int64_t T, void* cuda_stream) {
    if (!c || !s || !q || !out) return fail(SEGPA_ERR_INVALID, "attention_fwd: null argument");
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "attention_fwd: planning-only cache has no device; there is no CPU fallback");
    if (s->cache != c) return fail(SEGPA_ERR_STATE, "attention_fwd: segments were built by another cache");
    if (std::find(c->seg_objs.begin(), c->seg_objs.end(), s) == c->seg_objs.end()) return fail(SEGPA_ERR_STATE, "attention_fwd: stale segments object");
    const int Hq = c->desc.num_q_heads, D = c->desc.head_dim;
    if (T < s->stats.q_rows) return fail(SEGPA_ERR_INVALID, "attention_fwd: T %lld < rows used by the plan %lld", (long long)T, (long long)s->stats.q_rows);
    if (q_row_stride < (int64_t)Hq * D || out_row_stride < (int64_t)Hq * D) return fail(SEGPA_ERR_INVALID, "attention_fwd: row stride smaller than Hq*D");
    if ((q_row_stride % 8) || (out_row_stride % 8) || ((uintptr_t)q % 16) || ((uintptr_t)out % 16)) return fail(SEGPA_ERR_INVALID, "attention_fwd: q/out must be 16-byte aligned with row strides multiple of 8 elements");
    if (lse && lse_stride < T) return fail(SEGPA_ERR_INVALID, "attention_fwd: lse_stride < T");
    if (!(scale > 0.f) || !(scale < 1e30f)) return fail(SEGPA_ERR_INVALID, "attention_fwd: softmax_scale must be positive and finite");

    DeviceGuard g(c->desc.device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SEGPA_ERR_CUDA, "attention_fwd: earlier asynchronous failure: %s", cudaGetErrorString(e));

    FwdParams p{};
    s->last_stream = st;
    fill_fwd_params(p, c, s);
    p.q = (const uint16_t*)q;
    p.out = (uint16_t*)out;
    p.lse = lse;
    p.q_row_stride = q_row_stride;
    p.out_row_stride = out_row_stride;
    p.lse_stride = lse_stride;
    p.scale = scale;
    if (c->kernel_kind == 1) {
        const char* why = encode_q_map(&p.q_map, q, T, Hq, D, c->G, p.tile_tokens, q_row_stride);
        if (why) return fail(SEGPA_ERR_CUDA, "attention_fwd: %s", why);
    }

#ifdef SEGPA_TRACE
    static unsigned long long* d_trace = nullptr;
    if (!d_trace) cudaMalloc((void**)&d_trace, 16 * kTraceCap * 8);
    cudaMemsetAsync(d_trace, 0, 16 * kTraceCap * 8, st);
    p.trace = d_trace;
#endif
    int launches = 0;
#ifdef SEGPA_BRINGUP
    if (c->kernel_kind == 0) {   // test build only: the SIMT cross-check kernel over the same plan (it pulls items from a cursor)
        e = cudaMemsetAsync(s->buf->counter, 0, 256, st);
        if (e == cudaSuccess) e = launch_attention_simt(p, st);
        ++launches;
    } else
#endif
    if (e == cudaSuccess) {
        e = launch_attention_tc(p, st);
        ++launches;
    }
    if (e == cudaSuccess && p.n_combs > 0) {
        e = launch_combine(p, st);
        ++launches;
    }
#ifdef SEGPA_TRACE
    if (const char* tf = getenv("SEGPA_TRACE_FILE")) {
        std::vector<unsigned long long> h(16 * kTraceCap);
        cudaStreamSynchronize(st);
        cudaMemcpy(h.data(), d_trace, h.size() * 8, cudaMemcpyDeviceToHost);
        if (FILE* f = fopen(tf, "wb")) { fwrite(h.data(), 8, h.size(), f); fclose(f); }
    }
#endif
    c->last_launches = launches;
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(SEGPA_ERR_CUDA, "attention_fwd: launch failed: %s", cudaGetErrorString(e));
    }
    return SEGPA_OK;
}

namespace {

// segpa_attention_fwd_host: cut the plan into chunks of consecutive query rows (about 16 MB of Q each, at most 16),
// each with its own LPT assignment over the persistent grid and its own combine entries, and upload them (once per
// segments object).  An item belongs to the chunk that holds its first row.
segpa_status_t plan_host_chunks(segpa_cache* c, const segpa_segments* s, int64_t T, cudaStream_t st, const bool async) {
    if (s->host_planned) return SEGPA_OK;
    const int Hq = c->desc.num_q_heads, D = c->desc.head_dim;
    const int64_t row_bytes = (int64_t)Hq * D * 2;
    const int64_t rows_used = std::max<int64_t>(1, std::min(T, s->stats.q_rows));
    // ~16 MB of Q per chunk for a synchronous call (whose first chunk goes up and whose last comes down with the link idle
    // the other way: small chunks keep that short), ~32 MB for an asynchronous one (its ends overlap the neighbouring calls,
    // and fewer copies, events and launches pay: cfg5 185 -> 179 ms per step; 8 MB chunks: 200 ms).  The plan is made by the
    // first call on the segments object and kept.
    const int64_t chunk_bytes = async ? (32 << 20) : (16 << 20);
    int64_t n_chunks = std::min<int64_t>(16, std::max<int64_t>(1, (rows_used * row_bytes + chunk_bytes - 1) / chunk_bytes));
    int64_t rows_per = std::max<int64_t>(2 * kTileRows, cdiv(rows_used, n_chunks));   // an item spans < 2 * 128 rows: it reaches into the next chunk at most
    n_chunks = cdiv(rows_used, rows_per);
    std::vector<std::vector<ItemDev>> per((size_t)n_chunks);
    std::vector<int64_t> need((size_t)n_chunks, 0);
    for (const ItemDev& it : s->items) {
        const int64_t r0 = s->segs[(size_t)it.seg].q_row_start + it.t0;
        const size_t ch = (size_t)std::min<int64_t>(n_chunks - 1, r0 / rows_per);
        per[ch].push_back(it);
        need[ch] = std::max(need[ch], r0 + it.n_tok);
    }
    std::vector<std::vector<CombDev>> combs((size_t)n_chunks);
    for (const CombDev& cd : s->combs) {
        const int64_t r0 = s->segs[(size_t)cd.seg].q_row_start + cd.t0;
        combs[(size_t)std::min<int64_t>(n_chunks - 1, r0 / rows_per)].push_back(cd);
    }
    auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
    std::vector<uint8_t> blob;
    std::vector<int32_t> cta_off;
    s->hchunks.clear();
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        segpa_segments::HostChunk hc{};
        hc.row_lo = ch * rows_per;
        hc.row_hi = (ch == n_chunks - 1) ? T : std::min<int64_t>(T, (ch + 1) * rows_per);   // the last chunk carries the rows past the plan's
        hc.need_hi = std::max(need[(size_t)ch], hc.row_lo);
        std::vector<ItemDev>& items = per[(size_t)ch];
        hc.n_items = (int)items.size();
        cta_off.assign(1, 0);
        if (!items.empty()) lpt_assign(c->plan, items, nullptr, c->num_sms, cta_off);
        hc.n_cta = (int)cta_off.size() - 1;
        hc.n_combs = (int)combs[(size_t)ch].size();
        for (const CombDev& cd : combs[(size_t)ch]) hc.comb_max_rows = std::max(hc.comb_max_rows, cd.n_tok * c->G);
        hc.off_items = al(blob.size());
        blob.resize(hc.off_items + items.size() * sizeof(ItemDev));
        if (!items.empty()) memcpy(blob.data() + hc.off_items, items.data(), items.size() * sizeof(ItemDev));
        hc.off_cta = al(blob.size());
        blob.resize(hc.off_cta + cta_off.size() * sizeof(int32_t));
        memcpy(blob.data() + hc.off_cta, cta_off.data(), cta_off.size() * sizeof(int32_t));
        hc.off_combs = al(blob.size());
        blob.resize(hc.off_combs + std::max<size_t>(1, combs[(size_t)ch].size()) * sizeof(CombDev));
        if (hc.n_combs) memcpy(blob.data() + hc.off_combs, combs[(size_t)ch].data(), (size_t)hc.n_combs * sizeof(CombDev));
        s->hchunks.push_back(hc);
    }
    Staging& sg = s->buf->host_blob;
    cudaError_t e = staging_acquire(sg, al(blob.size()));
    if (e == cudaSuccess) {
        memcpy(sg.h, blob.data(), blob.size());
        e = staging_upload(sg, al(blob.size()), c->up_stream, st);
    }
    if (e != cudaSuccess) { cudaGetLastError(); return fail(e == cudaErrorMemoryAllocation ? SEGPA_ERR_OOM : SEGPA_ERR_CUDA, "attention_fwd_host: %s", cudaGetErrorString(e)); }
    s->host_planned = true;
    return SEGPA_OK;
}

}  // namespace

namespace {

segpa_status_t attention_fwd_host_impl(segpa_cache_t* c, const segpa_segments_t* s, const void* q_host, float scale, void* out_host,
                                       float* lse_host, int64_t T, void* cuda_stream, const bool async) {
    if (!c || !s || !q_host || !out_host) return fail(SEGPA_ERR_INVALID, "attention_fwd_host: null argument");
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "attention_fwd_host: planning-only cache has no device; there is no CPU fallback");
    if (s->cache != c || std::find(c->seg_objs.begin(), c->seg_objs.end(), s) == c->seg_objs.end())
        return fail(SEGPA_ERR_STATE, "attention_fwd_host: segments were not built by this cache (or were freed)");
    if (T < 1 || T < s->stats.q_rows) return fail(SEGPA_ERR_INVALID, "attention_fwd_host: T %lld < rows used by the plan %lld", (long long)T, (long long)s->stats.q_rows);
    if (!(scale > 0.f) || !(scale < 1e30f)) return fail(SEGPA_ERR_INVALID, "attention_fwd_host: softmax_scale must be positive and finite");
    const int Hq = c->desc.num_q_heads, D = c->desc.head_dim;
    const size_t row_bytes = (size_t)Hq * D * 2;
    const size_t qb = (size_t)T * row_bytes, lb = (size_t)T * Hq * 4;
    DeviceGuard g(c->desc.device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SEGPA_ERR_CUDA, "attention_fwd_host: earlier asynchronous failure: %s", cudaGetErrorString(e));
    segpa_cache::HostStage& hs = c->hs[async ? (c->hs_turn++ & 1) : 0];
    if (!hs.done && cudaEventCreateWithFlags(&hs.done, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        return fail(SEGPA_ERR_CUDA, "attention_fwd_host: cannot create events");
    }
    if (qb > hs.q_bytes || lb > hs.lse_bytes) {
        // (growing the set: its last user must have finished with it)
        if (hs.pending) { cudaEventSynchronize(hs.done); hs.pending = false; }
        cudaStreamSynchronize(st);
    }
    if (qb > hs.q_bytes) {
        if (hs.q) { cudaFree(hs.q); cudaFree(hs.out); hs.q = hs.out = nullptr; hs.q_bytes = 0; }
        if (cudaMalloc((void**)&hs.q, qb) != cudaSuccess || cudaMalloc((void**)&hs.out, qb) != cudaSuccess) {
            cudaGetLastError();
            if (hs.q) cudaFree(hs.q);
            hs.q = hs.out = nullptr;
            return fail(SEGPA_ERR_OOM, "attention_fwd_host: staging allocation of 2 x %zu bytes failed", qb);
        }
        hs.q_bytes = qb;
    }
    if (lb > hs.lse_bytes) {
        if (hs.lse) { cudaFree(hs.lse); hs.lse = nullptr; hs.lse_bytes = 0; }
        if (cudaMalloc((void**)&hs.lse, lb) != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_OOM, "attention_fwd_host: staging allocation failed"); }
        hs.lse_bytes = lb;
    }
    if (!c->h2d_stream && (cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking) != cudaSuccess ||
                           cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking) != cudaSuccess)) {
        cudaGetLastError();
        return fail(SEGPA_ERR_CUDA, "attention_fwd_host: cannot create the copy streams");
    }
    s->last_stream = st;
    segpa_status_t rc = plan_host_chunks(c, s, T, st, async);
    if (rc != SEGPA_OK) return rc;
    const size_t n_ch = s->hchunks.size();
    while (c->host_events.size() < 2 * n_ch + 1) {
        cudaEvent_t ev = nullptr;
        if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "attention_fwd_host: cannot create events"); }
        c->host_events.push_back(ev);
    }
    cudaEvent_t* ev_in = c->host_events.data();            // [n_ch]: Q rows of chunk k are on the device
    cudaEvent_t* ev_done = c->host_events.data() + n_ch;   // [n_ch]: kernels of chunk k have finished
    cudaEvent_t ev_start = c->host_events[2 * n_ch];

    // Three streams: Q chunks go up on h2d_stream one after the other; the caller's stream runs chunk k's kernels once
    // its rows (and the first rows of chunk k+1 its last items reach into) have arrived; d2h_stream copies chunk k's out /
    // lse rows back while chunk k+1 computes.  PCIe is full duplex, so the call is bounded by the larger direction.
    // (row, head) pairs no segment covers come back as zeros: the staging rows are cleared first.
    FwdParams base{};
    fill_fwd_params(base, c, s);
    const char* why = encode_q_map(&base.q_map, hs.q, T, Hq, D, c->G, base.tile_tokens, (int64_t)Hq * D);
    if (why) return fail(SEGPA_ERR_CUDA, "attention_fwd_host: %s", why);
    base.q = hs.q;
    base.out = hs.out;
    base.lse = hs.lse;
    base.q_row_stride = base.out_row_stride = (int64_t)Hq * D;
    base.lse_stride = T;
    base.scale = scale;
    const uint8_t* hb = (const uint8_t*)s->buf->host_blob.d;
    // the set's previous user (two asynchronous calls ago) must have finished: its kernels with hs.q, its copies back with
    // hs.out / hs.lse; done was recorded behind all of them
    e = cudaSuccess;
    if (hs.pending) {
        e = cudaStreamWaitEvent(st, hs.done, 0);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(c->h2d_stream, hs.done, 0);
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(hs.out, 0, qb, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(hs.lse, 0, lb, st);
    if (!async) {
        if (e == cudaSuccess) e = cudaEventRecord(ev_start, st);                  // earlier work on the caller's stream is ordered before
        if (e == cudaSuccess) e = cudaStreamWaitEvent(c->h2d_stream, ev_start, 0);   // ... the first copy
    }   // (asynchronous calls: the Q rows may go up while the kernels of the call before still run -- they use the other set)
    for (size_t k = 0; k < n_ch && e == cudaSuccess; ++k) {
        const segpa_segments::HostChunk& hc = s->hchunks[k];
        e = cudaMemcpyAsync((uint8_t*)hs.q + (size_t)hc.row_lo * row_bytes, (const uint8_t*)q_host + (size_t)hc.row_lo * row_bytes,
                            (size_t)(hc.row_hi - hc.row_lo) * row_bytes, cudaMemcpyHostToDevice, c->h2d_stream);
        if (e == cudaSuccess) e = cudaEventRecord(ev_in[k], c->h2d_stream);
    }
    int launches = 0;
    for (size_t k = 0; k < n_ch && e == cudaSuccess; ++k) {
        const segpa_segments::HostChunk& hc = s->hchunks[k];
        size_t last_in = k;
        while (last_in + 1 < n_ch && s->hchunks[last_in].row_hi < hc.need_hi) ++last_in;
        e = cudaStreamWaitEvent(st, ev_in[last_in], 0);
        if (e == cudaSuccess && hc.n_items > 0) {
            FwdParams p = base;
            p.items = (const ItemDev*)(hb + hc.off_items);
            p.cta_off = (const int*)(hb + hc.off_cta);
            p.combs = (const CombDev*)(hb + hc.off_combs);
            p.n_items = hc.n_items;
            p.n_cta = hc.n_cta;
            p.n_combs = hc.n_combs;
            p.comb_max_rows = hc.comb_max_rows;
            e = launch_attention_tc(p, st);
            ++launches;
            if (e == cudaSuccess && p.n_combs > 0) { e = launch_combine(p, st); ++launches; }
        }
        if (e == cudaSuccess) e = cudaEventRecord(ev_done[k], st);
        // rows of chunk k are final once the kernels of chunk k have run (items of chunk k-1 that reach into it ran before)
        if (e == cudaSuccess) e = cudaStreamWaitEvent(c->d2h_stream, ev_done[k], 0);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync((uint8_t*)out_host + (size_t)hc.row_lo * row_bytes, (const uint8_t*)hs.out + (size_t)hc.row_lo * row_bytes,
                                (size_t)(hc.row_hi - hc.row_lo) * row_bytes, cudaMemcpyDeviceToHost, c->d2h_stream);
        if (e == cudaSuccess && lse_host)
            e = cudaMemcpy2DAsync(lse_host + hc.row_lo, (size_t)T * 4, hs.lse + hc.row_lo, (size_t)T * 4, (size_t)(hc.row_hi - hc.row_lo) * 4,
                                  (size_t)Hq, cudaMemcpyDeviceToHost, c->d2h_stream);
    }
    c->last_launches = launches;
    if (e == cudaSuccess) e = cudaEventRecord(hs.done, c->d2h_stream);
    if (e == cudaSuccess) hs.pending = true;
    if (!async) {
        // the call is synchronous: wait for the last copy back (and leave the caller's stream ordered after it)
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, hs.done, 0);
        if (e == cudaSuccess) e = cudaEventSynchronize(hs.done);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        hs.pending = false;
    }
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "attention_fwd_host: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}

}  // namespace

segpa_status_t segpa_attention_fwd_host(segpa_cache_t* c, const segpa_segments_t* s, const void* q_host, float scale, void* out_host,
                                        float* lse_host, int64_t T, void* cuda_stream) {
    return attention_fwd_host_impl(c, s, q_host, scale, out_host, lse_host, T, cuda_stream, false);
}

segpa_status_t segpa_attention_fwd_host_async(segpa_cache_t* c, const segpa_segments_t* s, const void* q_host, float scale,
                                              void* out_host, float* lse_host, int64_t T, void* cuda_stream) {
    return attention_fwd_host_impl(c, s, q_host, scale, out_host, lse_host, T, cuda_stream, true);
}

segpa_status_t segpa_host_wait(segpa_cache_t* c) {
    if (!c) return fail(SEGPA_ERR_INVALID, "host_wait: null cache");
    if (c->planning_only) return SEGPA_OK;
    DeviceGuard g(c->desc.device);
    cudaError_t e = cudaSuccess;
    for (auto& h : c->hs)
        if (h.pending) {
            const cudaError_t e2 = cudaEventSynchronize(h.done);
            if (e == cudaSuccess) e = e2;
            h.pending = false;
        }
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "host_wait: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}


segpa_status_t segpa_merge(segpa_cache_t* c, const void* out_a, const float* lse_a, const void* out_b, const float* lse_b,
                           void* out, float* lse, int64_t row_stride, int64_t lse_stride, int64_t T, void* cuda_stream) {
    if (!c || !out_a || !lse_a || !out_b || !lse_b || !out || !lse) return fail(SEGPA_ERR_INVALID, "merge: null argument");
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "merge: planning-only cache has no device");
    const int Hq = c->desc.num_q_heads, D = c->desc.head_dim;
    if (T < 1 || row_stride < (int64_t)Hq * D || lse_stride < T) return fail(SEGPA_ERR_INVALID, "merge: bad T / strides");
    if ((row_stride % 8) || ((uintptr_t)out_a % 16) || ((uintptr_t)out_b % 16) || ((uintptr_t)out % 16))
        return fail(SEGPA_ERR_INVALID, "merge: out_a / out_b / out must be 16-byte aligned with a row stride multiple of 8 elements (as in attention_fwd)");
    DeviceGuard g(c->desc.device);
    cudaError_t e = launch_merge((const uint16_t*)out_a, lse_a, (const uint16_t*)out_b, lse_b, (uint16_t*)out, lse, row_stride,
                                 lse_stride, T, Hq, D, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "merge: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}

segpa_status_t segpa_segments_mass_layout(const segpa_segments_t* s, int64_t* offsets_out, int32_t cap, int32_t* n_out) {
    if (!s) return fail(SEGPA_ERR_INVALID, "segments_mass_layout: null argument");
    if (n_out) *n_out = (int32_t)s->segs.size();
    if (offsets_out)
        for (int32_t i = 0; i < cap && i < (int32_t)s->mass_off.size(); ++i) offsets_out[i] = s->mass_off[(size_t)i];
    return SEGPA_OK;
}

namespace {

// builds and uploads the attention-mass plan of a segments object (once)
segpa_status_t plan_mass(segpa_cache* c, const segpa_segments* s, cudaStream_t st) {
    if (s->mass_planned) {
        // the plan was uploaded by an earlier call, possibly on another stream: order this stream after that copy
        if (s->buf->mass_blob.up && cudaStreamWaitEvent(st, s->buf->mass_blob.up, 0) != cudaSuccess) {
            cudaGetLastError();
            return fail(SEGPA_ERR_CUDA, "attention_mass: cannot order the stream after the plan upload");
        }
        return SEGPA_OK;
    }
    const int TT = kTileRows / c->G;
    std::vector<MassItem> items;
    for (size_t si = 0; si < s->segs.size(); ++si) {
        const SegDev& sg = s->segs[si];
        const int64_t p0 = sg.kv_len - sg.q_len, W = sg.window, ns = sg.n_sink;
        const int ppb = kBlockKeys / c->desc.page_size;
        const int kb_first = sg.first_page / ppb, kb_end = kb_first + sg.n_pages_listed / ppb;
        for (int kb = kb_first; kb < kb_end; ++kb) {
            const int64_t lo_key = (int64_t)kb * kBlockKeys, hi_key = lo_key + kBlockKeys - 1;
            // rows (positions) that see a key of the block: causal p >= lo_key; window p <= hi_key + W - 1, or a sink block
            const int64_t p_first = std::max(p0, lo_key);
            const int64_t p_last = (lo_key < ns) ? (int64_t)sg.kv_len - 1 : std::min<int64_t>(sg.kv_len - 1, hi_key + W - 1);
            if (p_first > p_last) continue;
            items.push_back(MassItem{(int)si, kb, (int)((p_first - p0) / TT), (int)((p_last - p0) / TT + 1)});
        }
    }
    const int n_items = (int)items.size();
    const int n_cta = std::min(n_items, c->num_sms);
    std::vector<int32_t> cta_off((size_t)n_cta + 1, 0);
    std::vector<MassItem> ordered;
    if (n_items > 0) {
        // LPT over the persistent grid, cost = query tiles of the item (+1 for the K block load)
        std::vector<int> order((size_t)n_items);
        for (int i = 0; i < n_items; ++i) order[(size_t)i] = i;
        auto cost = [&](int i) { return items[(size_t)i].t_hi - items[(size_t)i].t_lo + 1; };
        std::sort(order.begin(), order.end(), [&](int a, int b) { return cost(a) != cost(b) ? cost(a) > cost(b) : a < b; });
        std::vector<int64_t> heap((size_t)n_cta);
        for (int q = 0; q < n_cta; ++q) heap[(size_t)q] = q;
        std::vector<std::vector<int>> per((size_t)n_cta);
        auto gt = std::greater<int64_t>();
        for (int idx : order) {
            std::pop_heap(heap.begin(), heap.end(), gt);
            int64_t& top = heap.back();
            per[(size_t)(top & 1023)].push_back(idx);
            top += (int64_t)cost(idx) * 1024;
            std::push_heap(heap.begin(), heap.end(), gt);
        }
        for (int q = 0; q < n_cta; ++q) {
            for (int idx : per[(size_t)q]) ordered.push_back(items[(size_t)idx]);
            cta_off[(size_t)q + 1] = (int32_t)ordered.size();
        }
    }
    std::vector<int32_t> kv_lens(s->segs.size());
    for (size_t i = 0; i < s->segs.size(); ++i) kv_lens[i] = s->segs[i].kv_len;
    auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
    s->m_off_items = 0;
    s->m_off_cta = al(std::max<size_t>(1, ordered.size()) * sizeof(MassItem));
    s->m_off_layout = al(s->m_off_cta + cta_off.size() * sizeof(int32_t));
    s->m_off_kvlen = al(s->m_off_layout + s->mass_off.size() * sizeof(int64_t));
    const size_t bytes = al(s->m_off_kvlen + kv_lens.size() * sizeof(int32_t));
    Staging& sg = s->buf->mass_blob;
    cudaError_t e = staging_acquire(sg, bytes);
    if (e == cudaSuccess) {
        uint8_t* hb = (uint8_t*)sg.h;
        if (!ordered.empty()) memcpy(hb + s->m_off_items, ordered.data(), ordered.size() * sizeof(MassItem));
        memcpy(hb + s->m_off_cta, cta_off.data(), cta_off.size() * sizeof(int32_t));
        memcpy(hb + s->m_off_layout, s->mass_off.data(), s->mass_off.size() * sizeof(int64_t));
        memcpy(hb + s->m_off_kvlen, kv_lens.data(), kv_lens.size() * sizeof(int32_t));
        e = staging_upload(sg, bytes, c->up_stream, st);   // (recorded in sg.up: calls on other streams wait for it, below)
    }
    if (e != cudaSuccess) { cudaGetLastError(); return fail(e == cudaErrorMemoryAllocation ? SEGPA_ERR_OOM : SEGPA_ERR_CUDA, "attention_mass: %s", cudaGetErrorString(e)); }
    s->mass_n_cta = n_cta;
    s->mass_planned = true;
    return SEGPA_OK;
}

}  // namespace

segpa_status_t segpa_attention_mass(segpa_cache_t* c, const segpa_segments_t* s, const void* q, int64_t q_row_stride, float scale,
                                    const float* lse, int64_t lse_stride, int64_t T, float* mass, int64_t mass_len,
                                    void* cuda_stream) {
    if (!c || !s || !q || !lse || !mass) return fail(SEGPA_ERR_INVALID, "attention_mass: null argument");
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "attention_mass: planning-only cache has no device");
    if (s->cache != c || std::find(c->seg_objs.begin(), c->seg_objs.end(), s) == c->seg_objs.end())
        return fail(SEGPA_ERR_STATE, "attention_mass: segments were not built by this cache (or were freed)");
    const int Hq = c->desc.num_q_heads, D = c->desc.head_dim;
    if (T < s->stats.q_rows || lse_stride < T) return fail(SEGPA_ERR_INVALID, "attention_mass: T / lse_stride smaller than the plan's rows");
    if (q_row_stride < (int64_t)Hq * D || (q_row_stride % 8) || ((uintptr_t)q % 16)) return fail(SEGPA_ERR_INVALID, "attention_mass: bad q stride / alignment");
    if (s->has_ragged) return fail(SEGPA_ERR_UNSUPPORTED, "attention_mass: a segment's stream has head segments with partial last pages (ragged chunk tails); the mass kernel works on dense streams only");
    if (mass_len < s->mass_off.back()) return fail(SEGPA_ERR_INVALID, "attention_mass: mass has %lld entries, the layout needs %lld", (long long)mass_len, (long long)s->mass_off.back());
    if (!(scale > 0.f) || !(scale < 1e30f)) return fail(SEGPA_ERR_INVALID, "attention_mass: softmax_scale must be positive and finite");
    DeviceGuard g(c->desc.device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s->last_stream = st;
    segpa_status_t rc = plan_mass(c, s, st);
    if (rc != SEGPA_OK) return rc;
    MassParams p{};
    const char* why = encode_q_map(&p.q_map, q, T, Hq, D, c->G, kTileRows / c->G, q_row_stride);
    if (why) return fail(SEGPA_ERR_CUDA, "attention_mass: %s", why);
    const uint8_t* mb = (const uint8_t*)s->buf->mass_blob.d;
    const uint8_t* db = (const uint8_t*)s->buf->blob.d;
    p.segs = (const SegDev*)(db + s->off_segs);
    p.pages = (const int*)(db + s->off_pages);
    p.items = (const MassItem*)(mb + s->m_off_items);
    p.cta_off = (const int*)(mb + s->m_off_cta);
    p.mass_off = (const long long*)(mb + s->m_off_layout);
    p.k_pool = c->k_pool;
    p.lse = lse;
    p.mass = mass;
    p.lse_stride = lse_stride;
    p.scale = scale;
    p.n_cta = s->mass_n_cta;
    p.G = c->G;
    p.D = D;
    p.P = c->desc.page_size;
    p.tile_tokens = kTileRows / c->G;
    p.page_bytes = c->page_bytes;
#ifdef SEGPA_TRACE
    static unsigned long long* d_mtrace = nullptr;
    if (!d_mtrace) cudaMalloc((void**)&d_mtrace, 32 * kTraceCap * 8);
    cudaMemsetAsync(d_mtrace, 0, 32 * kTraceCap * 8, st);
    p.trace = d_mtrace;
#endif
    cudaError_t e = cudaMemsetAsync(mass, 0, (size_t)s->mass_off.back() * sizeof(float), st);
    if (e == cudaSuccess) e = launch_attention_mass(p, st);
#ifdef SEGPA_TRACE
    if (const char* tf = getenv("SEGPA_MASS_TRACE_FILE")) {
        std::vector<unsigned long long> h(32 * kTraceCap);
        cudaStreamSynchronize(st);
        cudaMemcpy(h.data(), d_mtrace, h.size() * 8, cudaMemcpyDeviceToHost);
        if (FILE* f = fopen(tf, "wb")) { fwrite(h.data(), 8, h.size(), f); fclose(f); }
    }
#endif
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "attention_mass: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}

segpa_status_t segpa_mass_select(segpa_cache_t* c, const segpa_segments_t* s, const float* mass, float tau, uint8_t* selected,
                                 int32_t* n_selected, void* cuda_stream) {
    if (!c || !s || !mass || !selected || !n_selected) return fail(SEGPA_ERR_INVALID, "mass_select: null argument");
    if (c->planning_only) return fail(SEGPA_ERR_STATE, "mass_select: planning-only cache has no device");
    if (s->cache != c || std::find(c->seg_objs.begin(), c->seg_objs.end(), s) == c->seg_objs.end())
        return fail(SEGPA_ERR_STATE, "mass_select: segments were not built by this cache (or were freed)");
    if (!(tau > 0.f) || !(tau <= 1.f)) return fail(SEGPA_ERR_INVALID, "mass_select: tau must be in (0, 1]");
    DeviceGuard g(c->desc.device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s->last_stream = st;
    segpa_status_t rc = plan_mass(c, s, st);
    if (rc != SEGPA_OK) return rc;
    const uint8_t* mb = (const uint8_t*)s->buf->mass_blob.d;
    cudaError_t e = cudaMemsetAsync(selected, 0, (size_t)s->mass_off.back(), st);
    if (e == cudaSuccess)
        e = launch_mass_select(mass, (const long long*)(mb + s->m_off_layout), (const int*)(mb + s->m_off_kvlen), (int)s->segs.size(), tau,
                               selected, n_selected, st);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SEGPA_ERR_CUDA, "mass_select: %s", cudaGetErrorString(e)); }
    return SEGPA_OK;
}

int32_t segpa_last_launch_count(const segpa_cache_t* c) { return c ? c->last_launches : 0; }

#ifdef SEGPA_BRINGUP
// Test build only (libsegpa_bringup.so; not declared in include/segpa.h, not in the product library): run the
// plans of this cache on the SIMT cross-check kernel -- a second opinion on the pool layout, the builder and the
// scheduler that shares no kernel code with the tcgen05 path.  Call before build_segments.
segpa_status_t segpa_bringup_use_simt(segpa_cache_t* c, int32_t on) {
    if (!c) return fail(SEGPA_ERR_INVALID, "bringup_use_simt: null cache");
    if (!c->seg_objs.empty()) return fail(SEGPA_ERR_STATE, "bringup_use_simt: segments objects exist");
    c->kernel_kind = on ? 0 : 1;
    return SEGPA_OK;
}
#endif

}  // extern "C"
