// Plan geometry shared by the attention kernels (segpa_attn_tc.cu: two 128-row tiles per work item; segpa_attn_tc1.cu:
// one tile, two softmax warpgroups that alternate key blocks): which KV blocks and 64-key halves a tile of a work item
// visits.  Included INSIDE `namespace segpa { namespace {` of each kernel file (device-only helpers, internal linkage).
// Needs kHalfKeys defined by the including file.
struct TileRange {
    int n_rows;       // valid rows (0 = tile unused in this item)
    int tok0;         // first token of the tile inside the segment's q range
    int sink64, sb;   // sink part: 64-key halves [0, sink64) in blocks [0, sb), visited before the window part
                      // (0 when the segment has no sinks or the sink blocks touch the window blocks: merged)
    int lo64, hi64;   // window part: 64-key halves [lo64, hi64) that hold keys visible to some row of the tile
    int lo, hi;       // first block of the window part and one past its last block
    int step;         // 1; or 2 for a strided item (the two tiles hold the SAME rows and take alternate blocks)
};

// A strided item (ItemDev::flags & 1, decode-shaped: all its rows fit one tile) runs its KV range as two
// independent chains: tile t takes the blocks kb_lo + t, kb_lo + t + 2, ... and writes its own split-KV
// partial; the combine kernel merges them.  That keeps two QK^T -> softmax -> PV chains in flight where a
// single tile would leave the second tile slot (and half of the latency hiding) unused.
// Sinks (LOCAL segments with n_sink > 0): the visible set is [0, n_sink) U [i - W + 1, i]; a tile
// visits the sink blocks first and then its window blocks (two KV block ranges per item); when the two
// ranges touch they are merged into one and the gap is masked per element.  In a strided item tile 0 takes
// the sink blocks.
// KV blocks, pages and the 64-key halves below are all in SLOT space (head segments start on fresh pages, so
// a ragged stream has unused slots behind a segment's tail; slot = token for a dense stream), positions in token space.
__device__ __forceinline__ TileRange tile_range(const ItemDev& it, const SegDev& sg, const PadDev* __restrict__ pads, int tile, int TT, int G) {
    TileRange r;
    const bool strided = (it.flags & 1) != 0;
    const int tok_lo = it.t0 + (strided ? 0 : tile * TT);
    const int tok_hi = min(it.t0 + it.n_tok, tok_lo + TT);
    r.tok0 = tok_lo;
    r.n_rows = max(0, tok_hi - tok_lo) * G;
    r.sink64 = r.sb = r.lo64 = r.hi64 = r.lo = r.hi = 0;
    r.step = 1;
    if (r.n_rows == 0) return r;
    const int i0 = sg.kv_len - sg.q_len + tok_lo, i1 = sg.kv_len - sg.q_len + tok_hi - 1;
    // slots of the first and the last key the tile's rows see, and of its last sink key
    // (ragged stream: looked up by the host, ItemDev::slots; a strided item's two tile slots hold the same rows)
    int3 sl = make_int3(max(0, i0 - sg.window + 1), i1, min(sg.n_sink, i1 + 1) - 1);
    if (sg.n_pads > 0) {   // (selects, not an indexed access: `it` must stay in registers)
        const bool first = strided || tile == 0;
        sl = make_int3(first ? it.slots[0][0] : it.slots[1][0], first ? it.slots[0][1] : it.slots[1][1], first ? it.slots[0][2] : it.slots[1][2]);
    }
    r.lo64 = max(it.kb_lo * 2, sl.x / kHalfKeys);
    r.hi64 = min(it.kb_hi * 2, sl.y / kHalfKeys + 1);
    if (r.hi64 < r.lo64) r.hi64 = r.lo64;
    if (sg.n_sink > 0 && it.kb_lo == 0) {
        r.sink64 = (sl.z + 1 + kHalfKeys - 1) / kHalfKeys;
        r.sb = (r.sink64 + 1) >> 1;
        if (r.hi64 > r.lo64 && r.sb >= (r.lo64 >> 1)) { r.lo64 = 0; r.sink64 = r.sb = 0; }   // ranges touch: merge
        if (strided && tile != 0) r.sink64 = r.sb = 0;
    }
    r.lo = r.lo64 >> 1;
    r.hi = (r.hi64 == r.lo64) ? r.lo : ((r.hi64 + 1) >> 1);
    if (strided) {
        r.step = 2;
        const int first = r.lo + (((r.lo - it.kb_lo) & 1) != tile ? 1 : 0);       // first block of this parity
        if (first >= r.hi) { r.hi64 = r.lo64; r.lo = r.hi = first; return r; }   // no window block of its own
        r.hi = first + ((r.hi - 1 - first) & ~1) + 1;
        r.lo = first;
    }
    return r;
}

__device__ __forceinline__ bool has_blocks(const TileRange& r) { return r.sb > 0 || r.hi > r.lo; }
__device__ __forceinline__ int first_block(const TileRange& r) { return r.sb > 0 ? 0 : r.lo; }
__device__ __forceinline__ int last_block(const TileRange& r) { return r.hi > r.lo ? r.hi - 1 : r.sb - 1; }
__device__ __forceinline__ int n_blocks(const TileRange& r) { return r.sb + (r.hi - r.lo + r.step - 1) / r.step; }
// k-th block of the tile's sequence (sink blocks, then window blocks)
__device__ __forceinline__ int block_at(const TileRange& r, int k) { return k < r.sb ? k : r.lo + (k - r.sb) * r.step; }

// halves (bit 0 = keys [0, 64), bit 1 = keys [64, 128)) of block j the tile attends to (0: not its block)
__device__ __forceinline__ int half_mask(const TileRange& r, int j) {
    if (j < r.sb) return (2 * j < r.sink64 ? 1 : 0) | (2 * j + 1 < r.sink64 ? 2 : 0);
    if (j < r.lo || j >= r.hi || ((j - r.lo) & (r.step - 1))) return 0;
    return ((2 * j >= r.lo64 && 2 * j < r.hi64) ? 1 : 0) | ((2 * j + 1 >= r.lo64 && 2 * j + 1 < r.hi64) ? 2 : 0);
}

// The blocks the loader puts into the ring for an item: the union of its tiles' sequences, as sink blocks
// [0, sb) followed by window blocks [lo, hi) (one range [0, hi) when they touch).
struct ItemBlocks { int sb, lo, hi; };
template <int NT>
__device__ __forceinline__ ItemBlocks item_blocks(const ItemDev& it, const SegDev& sg, const PadDev* __restrict__ pads, int TT, int G) {
    ItemBlocks b;
    b.sb = 0; b.lo = INT_MAX; b.hi = 0;
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        const TileRange tr = tile_range(it, sg, pads, t, TT, G);
        if (tr.n_rows == 0) continue;
        b.sb = max(b.sb, tr.sb);
        if (tr.hi > tr.lo) { b.lo = min(b.lo, tr.lo); b.hi = max(b.hi, tr.hi); }
    }
    if (b.hi <= b.lo) { b.lo = b.hi = b.sb; }
    else if (b.sb >= b.lo) { b.lo = 0; b.sb = 0; }
    return b;
}

