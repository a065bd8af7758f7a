// Fused variable-length attention over per-head page lists (Alg. 2 line 15) for sm_100a, ONE 128-row
// tile per work item with the softmax of consecutive key blocks on TWO warpgroups (tiles_per_item = 1 plans).
//
// Why a second schedule.  In segpa_attn_tc.cu (two tiles per item) a tile's chain is serial: with S_t, O_t of two tiles in
// the 512 TMEM columns a tile has one score buffer, so QK^T(j+1) cannot start before PV(j) has read P(j), which cannot
// start before softmax(j) has finished; the tensor pipe works on one tile only while the other tile's softmax runs
// (DESIGN.md section 5.2).  Here the 512 columns are spent on ONE tile:
//     S0 S1 S2 [0, 384) (P_b, bf16, overwrites the first 64 columns of S_b in place)   O [384, 384 + D)
// Three score buffers: QK^T(x) only has to wait for PV(x-3) to have read P[x mod 3], so it is issued up to two blocks
// ahead of the softmax and runs UNDER it, and PV(x) has three block-times to finish before its buffer is needed again.
// The softmax of block x is done by warpgroup x mod 2, so two blocks' exponentials are in flight at once and both
// accumulate into the one O.  The two warpgroups share the running reference maximum of a row through shared memory
// (lazy: it moves only when a block's maximum exceeds it by 2^8, and then the warpgroup that moves it rescales O after
// the previous PV has completed); each keeps its own partial row sum, merged by the epilogue.
// Measured: on a par with the two-tile kernel on cfg2 / cfg3, 3-5 % behind on cfg4 / cfg5 (a K/V
// block is loaded per tile instead of per two tiles); the product default stays two tiles per item.
//
// One persistent CTA per SM, 16 warps:
//   warp 0 / 3    K loader / V loader (bulk copy per page; separate K and V rings: V(x) is consumed later than K(x)); warp 0
//                 also loads the Q tiles (TMA, two buffers: the next item's tile is loaded during the current item)
//   warp 1 / 2    QK^T issuer: QK^T(x) -> S[x mod 3] / PV issuer: O (+)= P[x mod 3] V(x).  Independent of each other but for
//                 the barriers (they touch different TMEM columns); both schedules are continuous across items
//   warps 4..7    softmax warpgroup of the even blocks, warps 8..11 of the odd blocks (thread = query row)
//   warps 12..15  epilogue warpgroup: O / l -> bf16, LSE, split-KV partials
// Blocks are numbered by a running counter over the CTA's whole item list (every role counts alike), so an item with an
// odd number of blocks does not leave one warpgroup idle.
#include "segpa_internal.h"
#include "sm100_ptx.cuh"

#include <climits>

namespace segpa {
using namespace ptx;

namespace {

constexpr int kLoaderWarp = 0;
constexpr int kMmaWarp = 1;
constexpr int kPvWarp = 2;
constexpr int kVLoaderWarp = 3;   // (also allocates and frees TMEM)
constexpr int kFirstSoftmaxWarp = 4;
constexpr int kFirstEpilogueWarp = 12;
constexpr int kThreads = 512;
constexpr int kHalfKeys = 64;
// register budgets (setmaxnreg): 128 * 72 + 256 * 192 + 128 * 56 = 65536
constexpr int kRegsLow = 72;
constexpr int kRegsSoftmax = 192;
constexpr int kRegsEpilogue = 56;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: the reference maximum moves only when a block's exceeds it by > 2^8
constexpr int kOutWarpBytes = 32 * 128;

// Pipeline trace (debug builds with -DSEGPA_TRACE only): lane 0 of every warp of CTA 0 logs (tag, arg, SM clock) records.
#ifdef SEGPA_TRACE
#define TRACE(tag, arg)                                                                                          \
    do {                                                                                                         \
        if (blockIdx.x == 0 && (threadIdx.x & 31) == 0 && trace_n < kTraceCap)                                   \
            p.trace[(threadIdx.x >> 5) * kTraceCap + trace_n++] =                                                \
                ((unsigned long long)(tag) << 56) | ((unsigned long long)((arg) & 0xffff) << 40) |               \
                ((unsigned long long)clock64() & 0xffffffffffull);                                               \
    } while (0)
#else
#define TRACE(tag, arg) do { } while (0)
#endif

// TMEM columns
constexpr uint32_t kColS = 0, kColO = 384;   // S0 S1 S2 [0, 384) (P_b, bf16, aliases the first 64 columns of S_b), O [384, 384 + D)
constexpr uint32_t kPBufs = 3;           // S / P buffers: block g uses buffer g mod 3

template <int D>
struct Cfg1 {
    static constexpr int kTileBytes = kTileRows * D * 2;      // Q tile, K block or V block
    static constexpr int kKStages = (D == 128) ? 2 : 4;
    static constexpr int kVStages = (D == 128) ? 2 : 4;
    static constexpr int kSmemQ = 2 * kTileBytes;
    static constexpr int kSmemK = kKStages * kTileBytes;
    static constexpr int kSmemV = kVStages * kTileBytes;
    static constexpr int kSmemOut = 4 * kOutWarpBytes;      // epilogue staging: 32 rows x 64 bf16 columns per warp
    static constexpr int kSmemBytes = kSmemQ + kSmemK + kSmemV + kSmemOut + 1024 /*align slack*/;
    static constexpr int kHalves = D / 64;
    static constexpr uint32_t kSBO = kHalves * kAtomBytes;
};

struct Bars1 {
    uint64_t k_full[4], k_empty[4];
    uint64_t v_full[4], v_empty[4];
    uint64_t q_full[2], q_empty[2];
    uint64_t s_full[3];        // MMA -> softmax: QK^T of a block has completed (S buffer b)
    uint64_t p_full[3][2];     // [P buffer][half]: P columns of keys [0,64) / [64,128) are in TMEM (PV starts on the first half)
    uint64_t pv_done[3];       // MMA -> softmax: PV of the block in P buffer b has completed (P_b reusable; O quiescent for a rescale)
    uint64_t m_pub[2];         // softmax -> softmax: the row maxima reference after the block of buffer b is in mref[]
    uint64_t o_final;          // MMA -> epilogue: last PV of the item has completed
    uint64_t o_free;           // epilogue -> MMA: O has been read out, the next item may overwrite it
    uint64_t stat_full;        // softmax (both warpgroups) -> epilogue: (m, l) parts of the finished item are in smem
    uint64_t stat_free;        // epilogue -> softmax
    uint32_t tmem_base;
};

#include "segpa_attn_common.cuh"  // (inside namespace segpa { namespace { : TileRange, tile_range, n_blocks, block_at, half_mask, ...)

}  // namespace

// RG: the plan has ragged streams (head segments with partial last pages in mid-stream).
template <int D, bool RG>
__global__ void __launch_bounds__(kThreads, 1) attention_tc1_kernel(const __grid_constant__ FwdParams p) {
    using C = Cfg1<D>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ Bars1 bars;
    __shared__ float mref[kTileRows];        // running reference maximum of each row (log2 units), handed from block to block
    __shared__ float2 stats[2][kTileRows];   // (scale m, partial row sum l) of each softmax warpgroup for the finished item
    __shared__ int out_row16[kTileRows];     // epilogue: where each row of the tile goes in `out` (16-byte units, -1: nowhere)
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~static_cast<uintptr_t>(1023));
    const uint32_t sQ = smem_u32(smem);
    const uint32_t sK = sQ + C::kSmemQ;
    const uint32_t sV = sK + C::kSmemK;
    const uint32_t sOut = sV + C::kSmemV;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // this CTA's work items: a contiguous, cost-descending slice of the list (host-side LPT assignment)
    const int i_lo = p.cta_off[blockIdx.x], i_hi = p.cta_off[blockIdx.x + 1];
    const int G = p.G, TT = p.tile_tokens, ppb = kBlockKeys / p.P;
    const int rows_per_slot = kTileRows * p.tiles_per_item;
#ifdef SEGPA_TRACE
    int trace_n = 0;
#endif

    if (threadIdx.x == 0) {
        for (int s = 0; s < 4; ++s) {
            mbar_init(smem_u32(&bars.k_full[s]), 1);
            mbar_init(smem_u32(&bars.k_empty[s]), 1);
            mbar_init(smem_u32(&bars.v_full[s]), 1);
            mbar_init(smem_u32(&bars.v_empty[s]), 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(smem_u32(&bars.q_full[b]), 1);
            mbar_init(smem_u32(&bars.q_empty[b]), 1);
            mbar_init(smem_u32(&bars.m_pub[b]), 128);
        }
        for (int b = 0; b < 3; ++b) {
            mbar_init(smem_u32(&bars.s_full[b]), 1);
            mbar_init(smem_u32(&bars.p_full[b][0]), 128);
            mbar_init(smem_u32(&bars.p_full[b][1]), 128);
            mbar_init(smem_u32(&bars.pv_done[b]), 1);
        }
        mbar_init(smem_u32(&bars.o_final), 1);
        mbar_init(smem_u32(&bars.o_free), 128);
        mbar_init(smem_u32(&bars.stat_full), 256);
        mbar_init(smem_u32(&bars.stat_free), 128);
        fence_mbar_init();
    }
    if (warp == 3) {
        tmem_alloc(smem_u32(&bars.tmem_base), 512);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = bars.tmem_base;
    // everything above overlapped the tail of the previous kernel of the stream (programmatic dependent launch)
    pdl_launch_dependents();
    pdl_wait();

    if (warp == kLoaderWarp || warp == kVLoaderWarp) {
        // ------------------------------------------------------------------ K loader (warp 0) / V loader (warp 3)
        // Separate rings: K(x) is consumed by QK^T(x), V(x) one step later by PV(x).
        reg_dec<kRegsLow>();
        const bool is_v = warp == kVLoaderWarp;
        const uint8_t* pool = is_v ? p.v_pool : p.k_pool;
        const uint32_t ring = is_v ? sV : sK;
        const uint32_t n_stages = is_v ? C::kVStages : C::kKStages;
        uint64_t* full = is_v ? bars.v_full : bars.k_full;
        uint64_t* empty = is_v ? bars.v_empty : bars.k_empty;
        uint32_t n_blk = 0;  // blocks filled so far
        // The K loader also loads the Q tiles (TMA, two buffers: the next item's tile is loaded during the current item).
        // Q tile image: [D/64 halves][128 rows][128 B], SWIZZLE_128B; row r = (token, group head) as the TMA box
        // {64 elements, G heads, tile_tokens tokens} lays it out.  Rows >= G*tile_tokens are never written (their scores
        // are garbage and never stored); tokens past T are zero-filled by TMA.
        const uint32_t box_bytes = (uint32_t)(64 * 2 * G * TT);
        uint32_t n_fill = 0;
        if (!is_v && lane == 0) prefetch_tmap(&p.q_map);
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const TileRange tr = tile_range(it, sg, p.pads, 0, TT, G);
            if (!is_v && tr.n_rows > 0) {
                const uint32_t qb = n_fill & 1;
                mbar_wait(smem_u32(&bars.q_empty[qb]), ((n_fill >> 1) & 1) ^ 1);   // last QK^T on this buffer's old Q is done
                ++n_fill;
                if (elect_one()) {
                    mbar_arrive_expect_tx(smem_u32(&bars.q_full[qb]), box_bytes * C::kHalves);
#pragma unroll
                    for (int h = 0; h < C::kHalves; ++h)
                        tma_load_3d(sQ + qb * C::kTileBytes + h * (kTileRows * 128), &p.q_map, h * 64, sg.kv_head * G,
                                    (int)(sg.q_row_start + tr.tok0), smem_u32(&bars.q_full[qb]));
                }
                __syncwarp();
            }
            const int n_steps = tr.n_rows > 0 ? n_blocks(tr) : 0;
            // page ids are fetched one block ahead: the dependent global load of the next block is in flight
            // while this block's copies are issued
            const int* pg = p.pages + sg.page_off - sg.first_page + lane;
            int page_next = (lane < ppb && n_steps > 0) ? pg[(long long)block_at(tr, 0) * ppb] : 0;
            for (int x = 0; x < n_steps; ++x) {
                const int page = page_next;
                if (lane < ppb && x + 1 < n_steps) page_next = pg[(long long)block_at(tr, x + 1) * ppb];
                const uint32_t st = n_blk % n_stages, ph = (n_blk / n_stages) & 1;
                if (lane == 0) {
                    mbar_wait(smem_u32(&empty[st]), ph ^ 1);
                    mbar_arrive_expect_tx(smem_u32(&full[st]), C::kTileBytes);
                }
                __syncwarp();
                if (lane < ppb)
                    bulk_g2s(ring + st * C::kTileBytes + lane * p.page_bytes, pool + (size_t)page * p.page_bytes, p.page_bytes,
                             smem_u32(&full[st]));
                ++n_blk;
            }
        }
    } else if (warp == kMmaWarp) {
        // ------------------------------------------------------------------ QK^T issuer
        // Two issuer warps: QK^T(x) -> S[x & 1] here, PV(x) below.  They touch different TMEM columns and meet only through
        // the barriers, so QK^T runs ahead of PV as far as the two S buffers allow (a single issuer spent ~2 300 cycles per
        // block in serial barrier waits and MMA issue: pipeline trace).  The whole warp walks the schedule and waits on the
        // barriers (warp-uniform control flow); one elected lane issues the tcgen05 instructions.
        reg_dec<kRegsLow>();
        constexpr uint32_t idesc_qk = make_idesc_bf16(128, 128, 0, 0);
        constexpr uint32_t idesc_qk64 = make_idesc_bf16(128, kHalfKeys, 0, 0);   // edge blocks: one 64-key half only
        // descriptors differ from a base only in the start-address field: add (bytes >> 4)
        const uint64_t dq0 = make_desc_sw128(sQ, 16, kAtomBytes);
        const uint64_t dk0 = make_desc_sw128(sK, 16, C::kSBO);
        uint32_t gb = 0;                       // running block number
        uint32_t nk = 0, n_q = 0;              // K stage reads, Q buffers consumed so far
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const TileRange tr = tile_range(it, sg, p.pads, 0, TT, G);
            if (tr.n_rows == 0) continue;
            const uint32_t qb = n_q & 1, qph = (n_q >> 1) & 1;
            ++n_q;
            const int nb = n_blocks(tr);
            if (nb == 0) {
                // tile present but no block of its own in this (split) item: hand Q straight back
                mbar_wait(smem_u32(&bars.q_full[qb]), qph);
                if (elect_one()) tc_commit(smem_u32(&bars.q_empty[qb]));
                __syncwarp();
                continue;
            }
            const uint64_t dq = dq0 + (uint64_t)((qb * C::kTileBytes) >> 4);
            for (int kb = 0; kb < nb; ++kb, ++gb) {
                const int j = block_at(tr, kb);
                const int am = half_mask(tr, j);           // never 0: the tile's own block sequence
                const uint32_t b = gb % kPBufs;
                const uint32_t tS = tmem + kColS + b * 128;
                // K stage landed, S_b / P_b free (PV of block gb - 3 has read P_b), Q landed (first block)
                const uint32_t st_k = nk % C::kKStages;
                TRACE(10, j);
                mbar_wait(smem_u32(&bars.k_full[st_k]), (nk / C::kKStages) & 1);
                ++nk;
                TRACE(11, j);
                if (gb >= kPBufs) mbar_wait(smem_u32(&bars.pv_done[b]), ((gb / kPBufs) - 1) & 1);
                if (kb == 0) mbar_wait(smem_u32(&bars.q_full[qb]), qph);
                tc_fence_after();
                TRACE(12, j);
                if (elect_one()) {
                    const uint64_t dk = dk0 + (uint64_t)((st_k * C::kTileBytes) >> 4);
                    if (am == 3) {
#pragma unroll
                        for (int kk = 0; kk < D / 16; ++kk) {
                            const uint32_t oq = ((kk / 4) * (kTileRows * 128) + (kk % 4) * 32) >> 4;
                            const uint32_t ok = ((kk / 4) * kAtomBytes + (kk % 4) * 32) >> 4;
                            mma_ss(tS, dq + oq, dk + ok, idesc_qk, kk > 0 ? 1u : 0u);
                        }
                    } else {
                        const int hb = (am == 2) ? 1 : 0;
                        const uint64_t dkh = dk + (uint64_t)((hb * 8 * C::kSBO) >> 4);
#pragma unroll
                        for (int kk = 0; kk < D / 16; ++kk) {
                            const uint32_t oq = ((kk / 4) * (kTileRows * 128) + (kk % 4) * 32) >> 4;
                            const uint32_t ok = ((kk / 4) * kAtomBytes + (kk % 4) * 32) >> 4;
                            mma_ss(tS + hb * kHalfKeys, dq + oq, dkh + ok, idesc_qk64, kk > 0 ? 1u : 0u);
                        }
                    }
                    tc_commit(smem_u32(&bars.s_full[b]));
                    tc_commit(smem_u32(&bars.k_empty[st_k]));
                    if (kb == nb - 1) tc_commit(smem_u32(&bars.q_empty[qb]));   // this Q buffer may be refilled
                }
                __syncwarp();
                TRACE(13, j);
            }
        }
    } else if (warp == kPvWarp) {
        // ------------------------------------------------------------------ PV issuer: O (+)= P[x & 1] V(x)
        reg_dec<kRegsLow>();
        constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, 0, 1);
        const uint64_t dv0 = make_desc_sw128(sV, kAtomBytes, C::kSBO);
        const uint32_t tO = tmem + kColO;
        uint32_t pv_g = 0;                     // running block number
        uint32_t nv = 0, n_of = 0;             // V stage reads, first-PV-of-an-item waits so far
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const TileRange tr = tile_range(it, sg, p.pads, 0, TT, G);
            if (tr.n_rows == 0) continue;
            const int nb = n_blocks(tr);
            for (int kb = 0; kb < nb; ++kb, ++pv_g) {
                const int pv_mask = half_mask(tr, block_at(tr, kb));   // halves of the block that hold visible keys
                const bool pv_first = kb == 0, pv_last = kb == nb - 1;
                const uint32_t b = pv_g % kPBufs, ph = (pv_g / kPBufs) & 1;
                const uint32_t tP = tmem + kColS + b * 128;   // P_b: the first 64 columns of S_b
                const uint32_t st_v = nv % C::kVStages;
                TRACE(14, pv_g);
                mbar_wait(smem_u32(&bars.v_full[st_v]), (nv / C::kVStages) & 1);
                ++nv;
                TRACE(15, pv_g);
                const uint64_t dv = dv0 + (uint64_t)((st_v * C::kTileBytes) >> 4);
                const uint32_t acc0 = pv_first ? 0u : 1u;
                // PV starts as soon as the first 64 keys of P are in TMEM; the softmax warpgroup is still working on the other 64
                mbar_wait(smem_u32(&bars.p_full[b][0]), ph);
                if (pv_first) {   // first PV of an item overwrites O: the epilogue must have read the previous item's out
                    mbar_wait(smem_u32(&bars.o_free), (n_of & 1) ^ 1);
                    ++n_of;
                }
                tc_fence_after();
                if ((pv_mask & 1) && elect_one()) {
#pragma unroll
                    for (int kk = 0; kk < kHalfKeys / 16; ++kk)
                        mma_ts(tO, tP + kk * 8, dv + (uint64_t)((kk * 2 * C::kSBO) >> 4), idesc_pv, kk > 0 ? 1u : acc0);
                }
                __syncwarp();
                TRACE(16, pv_g);
                mbar_wait(smem_u32(&bars.p_full[b][1]), ph);
                tc_fence_after();
                TRACE(17, pv_g);
                if (elect_one()) {
                    if (pv_mask & 2) {   // (a half without visible keys is skipped: its P is zero anyway)
                        const uint32_t acc1 = (pv_mask & 1) ? 1u : acc0;
#pragma unroll
                        for (int kk = kHalfKeys / 16; kk < kBlockKeys / 16; ++kk)
                            mma_ts(tO, tP + kk * 8, dv + (uint64_t)((kk * 2 * C::kSBO) >> 4), idesc_pv, kk > kHalfKeys / 16 ? 1u : acc1);
                    }
                    tc_commit(smem_u32(&bars.pv_done[b]));
                    tc_commit(smem_u32(&bars.v_empty[st_v]));
                    if (pv_last) tc_commit(smem_u32(&bars.o_final));
                }
                __syncwarp();
            }
        }
    } else if (warp < kFirstEpilogueWarp) {
        // ------------------------------------------------------------------ softmax warpgroups (w = 0: even blocks, 1: odd)
        reg_inc<kRegsSoftmax>();
        const int w = (warp - kFirstSoftmaxWarp) >> 2;
        const int wq = warp & 3;                       // TMEM lane quadrant this warp may access
        const int r = wq * 32 + lane;                  // row inside the tile
        const uint32_t lane_base = (uint32_t)(wq * 32) << 16;
        const uint32_t tO = tmem + lane_base + kColO;
        const float sl2 = p.scale * 1.4426950408889634f;
        uint32_t gb = 0;                               // running block number of the item's first block
        uint32_t n_st = 0;
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const TileRange tr = tile_range(it, sg, p.pads, 0, TT, G);
            if (tr.n_rows == 0) continue;

            const int rc = min(r, tr.n_rows - 1);            // rows past the end mirror the last valid row
            const int tok = tr.tok0 + rc / G;
            const int pos = sg.kv_len - sg.q_len + tok;      // query position i
            const int key_lo = max(0, pos - sg.window + 1);  // visible keys [key_lo, pos]
            const bool warp_has_rows = wq * 32 < tr.n_rows;  // decode-shaped tiles: most warps hold no row
            // positions are non-decreasing along the lanes, so the warp-wide extremes of the visible column range
            // are those of the first and the last lane: formed once per item, no votes or reductions per block
            const int pos_w0 = __shfl_sync(0xffffffffu, pos, 0), pos_w1 = __shfl_sync(0xffffffffu, pos, 31);
            const int klo_w0 = __shfl_sync(0xffffffffu, key_lo, 0), klo_w1 = __shfl_sync(0xffffffffu, key_lo, 31);
            float m_l = -INFINITY, l = 0.f;   // this warpgroup's part of the row sum, expressed against the reference m_l

            const int nb = n_blocks(tr);
            for (int kb = 0; kb < nb; ++kb) {
                const uint32_t g = gb + (uint32_t)kb;
                if ((int)(g & 1) != w) continue;
                const int j = block_at(tr, kb);
                const uint32_t pb = g % kPBufs;                              // this block's S / P buffer
                const uint32_t tS = tmem + lane_base + kColS + pb * 128;
                const uint32_t tP = tS;                                      // P overwrites S in place (bf16: its first 64 columns)
                TRACE(20, j);
                mbar_wait(smem_u32(&bars.s_full[pb]), (g / kPBufs) & 1);
                tc_fence_after();
                TRACE(21, j);
                if (!warp_has_rows) {
                    // no row in this warp: keep the barriers' arrival counts.  (Their order is safe: S(g) ready means QK^T(g)
                    // was issued, which waited for PV(g - 3), which waited for p_full of block g - 3: an arrival for block g
                    // cannot land in that block's phase.  m_pub is chained explicitly.)
                    if (g > 0) mbar_wait(smem_u32(&bars.m_pub[w ^ 1]), ((g - 1) >> 1) & 1);
                    mbar_arrive(smem_u32(&bars.m_pub[w]));
                    mbar_arrive(smem_u32(&bars.p_full[pb][0]));
                    mbar_arrive(smem_u32(&bars.p_full[pb][1]));
                    continue;
                }
                // Column c of block j is slot 128 j + c.  In a dense stream that is token 128 j + c; in a ragged one
                // (head segments on their own pages) the block either lies inside one head segment
                // (token = slot - pad, same form) or holds a segment tail: unused slots and a change of pad (ragged_blk)
                int tokb = j * kBlockKeys;      // token of column 0
                bool ragged_blk = false;
                if (RG && sg.n_pads > 0) {
                    int padv = 0, prev = 0;
                    for (int k = 0; k < sg.n_pads; ++k) {
                        const PadDev pd = p.pads[sg.pad_off + k];
                        const int seg0 = pd.tok + pd.pad, tail = pd.tok + prev;   // unused slots [tail, seg0)
                        if (seg0 <= j * kBlockKeys) padv = pd.pad;
                        else if (tail < (j + 1) * kBlockKeys) ragged_blk = true;
                        prev = pd.pad;
                    }
                    tokb -= padv;
                }
                // visible columns of this block: c <= cmax and (c >= cmin or c < csink)
                const int cmin = key_lo - tokb, cmax = pos - tokb;
                const int csink = sg.n_sink - tokb;        // same for every row of the segment
                const int mn_cmin = klo_w0 - tokb, mx_cmin = klo_w1 - tokb;   // over the warp's rows
                const int mn_cmax = pos_w0 - tokb, mx_cmax = pos_w1 - tokb;
                const bool need_mask = mn_cmax < kBlockKeys - 1 || (mx_cmin > 0 && csink < kBlockKeys);
                // the whole score row of this thread: 128 fp32 columns -> registers, one wait
                uint32_t s[kBlockKeys];
#pragma unroll
                for (int c = 0; c < 4; ++c) tmem_ld32(tS + c * 32, s + c * 32);
                // under the latency of those loads: the wait for the row's reference after block g - 1 (normally satisfied
                // long before, the other warpgroup is half a block ahead, but even a satisfied mbarrier wait costs ~100 cycles)
                if (g > 0) mbar_wait(smem_u32(&bars.m_pub[w ^ 1]), ((g - 1) >> 1) & 1);
                const float m_prev = (kb == 0) ? -INFINITY : mref[r];
                tmem_wait_ld();
                TRACE(22, j);
                bool dead[4] = {false, false, false, false};   // 32-column chunk masked for every row of the warp
                if (RG && ragged_blk) {
                    // The block holds the tail of a head segment.  Visible columns as a 128-bit set, built from
                    // intervals: for every head segment that reaches into the block, its columns [ra, rb) hold the
                    // tokens c + off; of those, the window [key_lo, pos] and the sinks [0, n_sink) are visible.
                    uint32_t vis[4] = {0u, 0u, 0u, 0u};
                    auto add_bits = [&vis](int a, int b) {
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const int lo = min(max(a - 32 * q, 0), 32), hi = min(max(b - 32 * q, 0), 32);
                            if (hi > lo) vis[q] |= (hi == 32 ? 0xffffffffu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
                        }
                    };
                    const int B = j * kBlockKeys;
                    int start = 0, pad_c = 0;
                    for (int k = 0; k <= sg.n_pads; ++k) {
                        int end = INT_MAX, nstart = 0, npad = 0;
                        if (k < sg.n_pads) {
                            const PadDev pd = p.pads[sg.pad_off + k];
                            end = pd.tok + pad_c;
                            nstart = pd.tok + pd.pad;
                            npad = pd.pad;
                        }
                        const int ra = max(start, B) - B, rb = min(end, B + kBlockKeys) - B;
                        if (ra < rb) {
                            const int off = B - pad_c;
                            add_bits(max(ra, key_lo - off), min(rb, pos - off + 1));
                            add_bits(ra, min(rb, min(sg.n_sink, pos + 1) - off));
                        }
                        start = nstart;
                        pad_c = npad;
                    }
#pragma unroll
                    for (int c = 0; c < 4; ++c) dead[c] = __all_sync(0xffffffffu, vis[c] == 0u);
#pragma unroll
                    for (int e = 0; e < kBlockKeys; ++e)
                        if (!((vis[e >> 5] >> (e & 31)) & 1u)) s[e] = 0xff800000u;   // -inf
                } else if (need_mask) {
                    // boundary block (causal diagonal / window edge / sink edge).  Per 32-column chunk, warp-uniformly:
                    // all visible -> untouched; all masked -> no exp at all; ragged -> element mask in registers
                    if (sg.n_sink == 0) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const int c0 = 32 * c, c1 = 32 * c + 31;
                            dead[c] = c0 > mx_cmax || c1 < mn_cmin;
                            if (!dead[c] && !(c1 <= mn_cmax && c0 >= mx_cmin)) {
#pragma unroll
                                for (int e = 0; e < 32; ++e)
                                    if (c0 + e > cmax || c0 + e < cmin) s[c0 + e] = 0xff800000u;   // -inf
                            }
                        }
                    } else {   // with sinks the visible columns are two intervals: [0, csink) and [cmin, cmax]
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const int c0 = 32 * c, c1 = 32 * c + 31;
                            dead[c] = c0 > mx_cmax || (c1 < mn_cmin && c0 >= csink);
                            if (!dead[c] && !(c1 <= mn_cmax && (c0 >= mx_cmin || c1 < csink))) {
#pragma unroll
                                for (int e = 0; e < 32; ++e)
                                    if (c0 + e > cmax || (c0 + e < cmin && c0 + e >= csink)) s[c0 + e] = 0xff800000u;
                            }
                        }
                    }
                }
                // row max: one pair of chains per 32-column chunk, no branches; a dead chunk (left holding raw,
                // possibly stale scores) is dropped by a select.  max.f32 returns the non-NaN operand.
                float mc[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    float ma = -INFINITY, mb = -INFINITY;
#pragma unroll
                    for (int e = 32 * c; e < 32 * c + 32; e += 4) {
                        ma = max3(ma, __uint_as_float(s[e + 0]), __uint_as_float(s[e + 1]));
                        mb = max3(mb, __uint_as_float(s[e + 2]), __uint_as_float(s[e + 3]));
                    }
                    mc[c] = dead[c] ? -INFINITY : fmaxf(ma, mb);
                }
                const float mx2 = fmaxf(fmaxf(mc[0], mc[1]), fmaxf(mc[2], mc[3])) * sl2;
                // ---- the row's reference maximum, handed from block to block (the other warpgroup did block g - 1)
                TRACE(23, j);
                // lazy: it moves only when this block's maximum exceeds it by 2^8 (P then stays <= 2^8: exact after the
                // final O / l, because every row sum uses the same reference)
                const bool grow = mx2 > m_prev + kRescaleThreshold;
                const float m_new = grow ? mx2 : m_prev;
                mref[r] = m_new;
                mbar_arrive(smem_u32(&bars.m_pub[w]));   // (release: orders the store before the arrive)
                if (m_l != m_new) {                      // this warpgroup's row sum follows the reference
                    l *= (m_l == -INFINITY) ? 0.f : fast_exp2(m_l - m_new);
                    m_l = m_new;
                }
                // (warp-uniform decision: tcgen05.ld/st are warp-collective)
                if (__any_sync(0xffffffffu, grow) && kb > 0) {
                    // O holds the blocks up to g - 1 against m_prev: wait until PV(g - 1) has completed (nothing else can
                    // touch O before this warpgroup hands over P(g)), then rescale the row
                    mbar_wait(smem_u32(&bars.pv_done[(g - 1) % kPBufs]), ((g - 1) / kPBufs) & 1);
                    tc_fence_after();
                    const float corr = !grow ? 1.f : ((m_prev == -INFINITY) ? 0.f : fast_exp2(m_prev - m_new));
#pragma unroll 1
                    for (int c = 0; c < D / 16; ++c) {
                        uint32_t v[16];
                        tmem_ld16(tO + c * 16, v);
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 16; ++e) v[e] = __float_as_uint(__uint_as_float(v[e]) * corr);
                        tmem_st16(tO + c * 16, v);
                    }
                }
                tc_fence_after();
                const float mref_v = (m_new == -INFINITY) ? 0.f : m_new;
                // p = 2^(s*scale*log2e - m) (masked columns: 2^-inf = 0), row sum, bf16 P -> TMEM
                const uint64_t sl2x2 = pack2(sl2, sl2), nmx2 = pack2(-mref_v, -mref_v);
                uint64_t rsa = pack2(0.f, 0.f), rsb = pack2(0.f, 0.f);
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t pk[16];
                    if (dead[c]) {
#pragma unroll
                        for (int q = 0; q < 16; ++q) pk[q] = 0u;
                    } else {
#pragma unroll
                        for (int q = 0; q < 16; ++q) {
                            const int e = c * 32 + 2 * q;
                            const uint64_t x = ffma2(pack2(__uint_as_float(s[e]), __uint_as_float(s[e + 1])), sl2x2, nmx2);
                            float x0, x1;
                            unpack2(x, x0, x1);
                            const float p0 = fast_exp2(x0), p1 = fast_exp2(x1);
                            if (q & 1) rsb = fadd2(rsb, pack2(p0, p1)); else rsa = fadd2(rsa, pack2(p0, p1));
                            pk[q] = pack_bf16x2(p0, p1);
                        }
                    }
                    tmem_st16(tP + c * 16, pk);
                    if (c == 1) {   // keys [0, 64) done: let their PV start
                        tmem_wait_st();
                        tc_fence_before();
                        mbar_arrive(smem_u32(&bars.p_full[pb][0]));
                    }
                }
                float rs0, rs1, rs2, rs3;
                unpack2(rsa, rs0, rs1);
                unpack2(rsb, rs2, rs3);
                l += (rs0 + rs1) + (rs2 + rs3);
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(smem_u32(&bars.p_full[pb][1]));
                TRACE(26, j);
            }
            gb += (uint32_t)nb;
            // hand this warpgroup's (reference, partial row sum) to the epilogue warpgroup and go on to the next item
            mbar_wait(smem_u32(&bars.stat_free), (n_st & 1) ^ 1);
            ++n_st;
            stats[w][r] = make_float2(m_l, l);
            mbar_arrive(smem_u32(&bars.stat_full));   // release: orders the store before the arrive
        }
    } else {
        // ------------------------------------------------------------------ epilogue warpgroup
        reg_dec<kRegsEpilogue>();
        const int wq = warp & 3;
        const int r = wq * 32 + lane;
        const uint32_t lane_base = (uint32_t)(wq * 32) << 16;
        const uint32_t tO = tmem + lane_base + kColO;
        uint32_t n_o = 0, n_st = 0;
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const TileRange tr = tile_range(it, sg, p.pads, 0, TT, G);
            if (tr.n_rows == 0) continue;
            const bool has_blk = has_blocks(tr);
            const int rc = min(r, tr.n_rows - 1);
            const int tok = tr.tok0 + rc / G;
            const bool valid = r < tr.n_rows;
            const int head = sg.kv_head * G + rc % G;
            const long long row = sg.q_row_start + tok;
            mbar_wait(smem_u32(&bars.stat_full), n_st & 1);
            ++n_st;
            // the row's reference is the later (larger) of the two warpgroups'; each partial sum is brought to it
            const float2 sa = stats[0][r], sb = stats[1][r];
            mbar_arrive(smem_u32(&bars.stat_free));
            float2 ml;
            ml.x = fmaxf(sa.x, sb.x);
            ml.y = ((sa.x == -INFINITY) ? 0.f : sa.y * fast_exp2(sa.x - ml.x)) + ((sb.x == -INFINITY) ? 0.f : sb.y * fast_exp2(sb.x - ml.x));
            if (has_blk) {
                mbar_wait(smem_u32(&bars.o_final), n_o & 1);
                ++n_o;
                tc_fence_after();
            }
            if (it.partial_slot >= 0) {
                const size_t base = (size_t)it.partial_slot * rows_per_slot + (size_t)(tr.tok0 - it.t0) * G + r;
#pragma unroll 1
                for (int c = 0; c < D / 16; ++c) {
                    uint32_t v[16];
                    if (has_blk) { tmem_ld16(tO + c * 16, v); tmem_wait_ld(); }
                    else {
#pragma unroll
                        for (int e = 0; e < 16; ++e) v[e] = 0u;
                    }
                    if (valid) {
                        float4* dst = reinterpret_cast<float4*>(p.ws_o + base * D + c * 16);
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            dst[e] = make_float4(__uint_as_float(v[4 * e]), __uint_as_float(v[4 * e + 1]),
                                                 __uint_as_float(v[4 * e + 2]), __uint_as_float(v[4 * e + 3]));
                    }
                }
                if (valid) { p.ws_ml[base * 2] = ml.x; p.ws_ml[base * 2 + 1] = ml.y; }
                if (has_blk) {
                    tc_fence_before();
                    mbar_arrive(smem_u32(&bars.o_free));   // O may be overwritten by the next item
                }
            } else {
                // Row r of the tile is one contiguous D-element row of `out`, but consecutive rows are far apart:
                // a store straight from the TMEM layout (lane = row) touches 32 lines per instruction.  So each
                // warp transposes its 32 rows through shared memory, 64 columns at a time (16-byte chunks
                // XOR-swizzled by row, conflict-free both ways), and stores 4 full 128-byte lines per instruction.
                const float inv = 1.f / ml.y;
                const long long off16 = (row * p.out_row_stride + (long long)head * D) >> 3;
                out_row16[r] = valid ? (int)off16 : -1;
                const uint32_t stg = sOut + wq * kOutWarpBytes;
                uint4* out16 = reinterpret_cast<uint4*>(p.out);
#pragma unroll 1
                for (int h = 0; h < D / 64; ++h) {
#pragma unroll 2
                    for (int c = 0; c < 4; ++c) {
                        uint32_t v[16];
                        tmem_ld16(tO + h * 64 + c * 16, v);
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            uint4 o;
                            o.x = pack_bf16x2(__uint_as_float(v[8 * e + 0]) * inv, __uint_as_float(v[8 * e + 1]) * inv);
                            o.y = pack_bf16x2(__uint_as_float(v[8 * e + 2]) * inv, __uint_as_float(v[8 * e + 3]) * inv);
                            o.z = pack_bf16x2(__uint_as_float(v[8 * e + 4]) * inv, __uint_as_float(v[8 * e + 5]) * inv);
                            o.w = pack_bf16x2(__uint_as_float(v[8 * e + 6]) * inv, __uint_as_float(v[8 * e + 7]) * inv);
                            sts128(stg + lane * 128 + (((2 * c + e) ^ (lane & 7)) << 4), o);
                        }
                    }
                    if (h == D / 64 - 1 && has_blk) {   // O is in registers / shared memory now: the next item may overwrite it
                        tc_fence_before();
                        mbar_arrive(smem_u32(&bars.o_free));
                    }
                    __syncwarp();
#pragma unroll 4
                    for (int i = 0; i < 8; ++i) {
                        const int rr = i * 4 + (lane >> 3);
                        const int ro = out_row16[wq * 32 + rr];
                        const uint4 o = lds128(stg + rr * 128 + (((lane & 7) ^ (rr & 7)) << 4));
                        if (ro >= 0) out16[(long long)ro + h * 8 + (lane & 7)] = o;
                    }
                    __syncwarp();
                }
                if (valid && p.lse) p.lse[(long long)head * p.lse_stride + row] = (ml.x + log2f(ml.y)) * 0.6931471805599453f;
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 3) tmem_dealloc(tmem, 512);
}

// ---------------------------------------------------------------------------------------------
template <int D, bool RG>
static cudaError_t launch_one1(const FwdParams& p, cudaStream_t st) {
    using C = Cfg1<D>;
    // the opt-in to > 48 KB of dynamic shared memory is per device: remember which devices have it
    static bool configured[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        cudaError_t e = cudaFuncSetAttribute(attention_tc1_kernel<D, RG>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    return launch_pdl(attention_tc1_kernel<D, RG>, dim3((unsigned)p.n_cta), dim3(kThreads), (size_t)C::kSmemBytes, st, p);
}

// tiles_per_item == 1 plans that are not decode-shaped
cudaError_t launch_attention_tc1(const FwdParams& p, cudaStream_t st) {
    if (p.n_items == 0) return cudaSuccess;
    if (p.has_ragged) return p.D == 128 ? launch_one1<128, true>(p, st) : launch_one1<64, true>(p, st);
    return p.D == 128 ? launch_one1<128, false>(p, st) : launch_one1<64, false>(p, st);
}

}  // namespace segpa
