// Fused variable-length attention over per-head page lists (Alg. 2 line 15) for
// sm_100a: cp.async.bulk (TMA) page gather -> shared memory, TMA tensor-map loads of Q, tcgen05.mma
// with TMEM accumulators for S = Q K^T and O += P V, fp32 online softmax, bf16 output + fp32 LSE.
// See DESIGN.md section 5.2.
//
// One persistent CTA per SM, 16 warps, warp-specialised:
//   warp 0 / 3    K loader / V loader: one bulk copy per physical page into a ring of K/V stages
//   warp 1        MMA issuer (whole warp walks the schedule, one elected lane issues)
//   warp 2        Q loader: two TMA boxes per 128-row tile, next item's Q prefetched into L2
//                 (warp 3 also allocates TMEM)
//   warps 4..7    softmax warpgroup of tile 0 (thread = query row)
//   warps 8..11   softmax warpgroup of tile 1 (NT = 2: two 128-row tiles of adjacent tokens share
//                 every K/V stage and ping-pong on the tensor pipe)
//   warps 12..15  epilogue warpgroup: O / l -> bf16, LSE, split-KV partials, for both tiles
// The MMA schedule is one continuous sequence of steps across work items: step (item, block j) issues
// for each tile PV of the PREVIOUS step's block (possibly the last block of the previous item) and
// QK^T of block j, so the tensor pipe does not drain at item boundaries; the epilogue of item i runs
// beside the first blocks of item i+1.
// A tile row r is (token t0 + r / G, query head kv_head*G + r % G): the G heads of a KV head share
// each K/V page load (GQA packing).
//
// TMEM (512 columns): S_t at [128 t, 128 t + 128) (P_t, bf16, aliases its first 64 columns),
// O_t at [256 + 128 t, +D).
#include "segpa_internal.h"
#include "sm100_ptx.cuh"

#include <climits>
#include <cstdlib>
#include <type_traits>

namespace segpa {
using namespace ptx;

namespace {

constexpr int kLoaderWarp = 0;
constexpr int kMmaWarp = 1;
constexpr int kQWarp = 2;
constexpr int kVLoaderWarp = 3;   // (also allocates and frees TMEM)
constexpr int kFirstSoftmaxWarp = 4;
constexpr int kFirstEpilogueWarp = 12;
constexpr int kThreads = 512;
constexpr int kHalfKeys = 64;
// register budgets (setmaxnreg): 128 * 72 + 256 * 192 + 128 * 56 = 65536
constexpr int kRegsLow = 72;
constexpr int kRegsSoftmax = 192;
constexpr int kRegsEpilogue = 56;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: O is rescaled only when the max grows by > 2^8

// Pipeline trace (debug builds with -DSEGPA_TRACE only): lane 0 of every warp of CTA 0 logs
// (tag, arg, SM clock) records that _work scripts turn into a timeline.
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

constexpr int kOutWarpBytes = 32 * 128;

template <int D, int NT>
struct Cfg {
    static constexpr int kTileBytes = kTileRows * D * 2;      // Q tile, K block or V block
    static constexpr int kStages = (D == 128) ? 4 : 8;   // > 114 KB of smem either way: one CTA per SM (it owns all of TMEM)
    static constexpr int kSmemQ = NT * kTileBytes;
    static constexpr int kSmemKV = kStages * kTileBytes;
    static constexpr int kSmemOut = 4 * kOutWarpBytes;      // epilogue staging: 32 rows x 64 bf16 columns per warp
    static constexpr int kSmemBytes = kSmemQ + kSmemKV + kSmemOut + 1024 /*align slack*/;
    static constexpr int kHalves = D / 64;
    static constexpr uint32_t kSBO = kHalves * kAtomBytes;
};

struct Bars {
    uint64_t kv_full[8];
    uint64_t kv_empty[8];
    uint64_t q_full[2];
    uint64_t q_empty[2];
    uint64_t s_full[2];
    uint64_t p_full[2][2];     // [tile][half]: P columns of keys [0,64) / [64,128) are in TMEM (PV starts on the first half)
    uint64_t o_final[2];    // MMA -> epilogue: last PV of the item's tile has completed
    uint64_t o_free[2];     // epilogue -> MMA: O_t has been read out, the next item may overwrite it
    uint64_t stat_full[2];  // softmax -> epilogue: (m, l) of the finished tile are in smem
    uint64_t stat_free[2];  // epilogue -> softmax
    uint32_t tmem_base;
};

#include "segpa_attn_common.cuh"  // (inside namespace segpa { namespace { : TileRange, tile_range, item_blocks, ...)

// ---------------------------------------------------------------------------------------------
// Softmax of a decode-shaped plan (instantiation NARROW: every tile of the plan holds <= 16 valid rows).
// With one thread per query row the exponentials of a 4-row tile cost as much as those of a 128-row tile
// (MUFU.EX2 occupies its pipe 8 cycles per warp instruction whatever the number of active lanes: measured), and the
// chain QK^T -> softmax -> PV of a decode step was bound by them (1 500 of ~2 500 cycles per block), not by HBM.
// Here a row is spread over FOUR threads: warp 0 of the tile's softmax warpgroup reads S with the 16x256b shape
// (thread t: rows t/4 and t/4 + 8, columns 8i + 2(t%4), +1 of every 8), so a thread holds 32 columns of a row (64 with
// rows 8..15 in use), reduces max / sum over its group of four with two shuffles, and writes bf16 P back with the
// 16x128b shape, whose column 4i + t%4 is exactly the pair it has just packed.  Warps 1..3 of the warpgroup hold no row.
// ---------------------------------------------------------------------------------------------
template <int D, bool RG>
__device__ __forceinline__ void softmax_narrow(const FwdParams& p, Bars& bars, float2 (&stats)[2][kTileRows], const uint32_t tmem,
                                               const int tile, const int wq, const int lane, const int i_lo, const int i_hi,
                                               const int TT, const int G) {
    const uint32_t tS = tmem + tile * 128;            // lanes 0..15 of quadrant 0
    const uint32_t tO = tmem + 256 + tile * 128;
    const float sl2 = p.scale * 1.4426950408889634f;
    const int g = lane >> 2, q = lane & 3;
    uint32_t n_s = 0, n_st = 0;
    for (int ii = i_lo; ii < i_hi; ++ii) {
        const ItemDev it = p.items[ii];
        const SegDev sg = p.segs[it.seg];
        const TileRange tr = tile_range(it, sg, p.pads, tile, TT, G);
        if (tr.n_rows == 0) continue;
        const int nb = n_blocks(tr);
        if (wq != 0) {   // no rows in this warp: keep the barriers' arrival counts
            for (int kb = 0; kb < nb; ++kb) {
                mbar_wait(smem_u32(&bars.s_full[tile]), n_s & 1);
                ++n_s;
                mbar_arrive(smem_u32(&bars.p_full[tile][0]));
                mbar_arrive(smem_u32(&bars.p_full[tile][1]));
            }
            mbar_wait(smem_u32(&bars.stat_free[tile]), (n_st & 1) ^ 1);
            ++n_st;
            mbar_arrive(smem_u32(&bars.stat_full[tile]));
            continue;
        }
        // rows X = 0: g, X = 1: g + 8 (rows past the end mirror the last valid row)
        const bool useB = tr.n_rows > 8;
        int pos[2], klo[2];
        bool live[2];
#pragma unroll
        for (int X = 0; X < 2; ++X) {
            const int row = g + 8 * X;
            live[X] = row < tr.n_rows;
            pos[X] = sg.kv_len - sg.q_len + tr.tok0 + min(row, tr.n_rows - 1) / G;
            klo[X] = max(0, pos[X] - sg.window + 1);
        }
        const int pos_min = sg.kv_len - sg.q_len + tr.tok0, pos_max = pos_min + (tr.n_rows - 1) / G;
        const int klo_max = max(0, pos_max - sg.window + 1);
        float m[2] = {-INFINITY, -INFINITY}, l[2] = {0.f, 0.f};   // l: this thread's part of the row sum
        for (int kb = 0; kb < nb; ++kb) {
            const int j = block_at(tr, kb);
            mbar_wait(smem_u32(&bars.s_full[tile]), n_s & 1);
            ++n_s;
            tc_fence_after();
            int tokb = j * kBlockKeys;      // token of column 0 (see the one-thread-per-row path)
            bool ragged_blk = false;
            if (RG && sg.n_pads > 0) {
                int padv = 0, prev = 0;
                for (int k = 0; k < sg.n_pads; ++k) {
                    const PadDev pd = p.pads[sg.pad_off + k];
                    const int seg0 = pd.tok + pd.pad, tail = pd.tok + prev;
                    if (seg0 <= j * kBlockKeys) padv = pd.pad;
                    else if (tail < (j + 1) * kBlockKeys) ragged_blk = true;
                    prev = pd.pad;
                }
                tokb -= padv;
            }
            // element (row X, repeat i, e) = s[4 i + 2 X + e], column 8 i + 2 q + e
            uint32_t s[64];
            tmem_ld_16x256b_x16(tS, s);
            tmem_wait_ld();
            const int csink = sg.n_sink - tokb;
            const bool need_mask = pos_min - tokb < kBlockKeys - 1 || (klo_max - tokb > 0 && csink < kBlockKeys);
            if (RG && ragged_blk) {
#pragma unroll
                for (int X = 0; X < 2; ++X) {
                    uint32_t vis[4] = {0u, 0u, 0u, 0u};
                    auto add_bits = [&vis](int a, int b) {
#pragma unroll
                        for (int w = 0; w < 4; ++w) {
                            const int lo = min(max(a - 32 * w, 0), 32), hi = min(max(b - 32 * w, 0), 32);
                            if (hi > lo) vis[w] |= (hi == 32 ? 0xffffffffu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
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
                            add_bits(max(ra, klo[X] - off), min(rb, pos[X] - off + 1));
                            add_bits(ra, min(rb, min(sg.n_sink, pos[X] + 1) - off));
                        }
                        start = nstart;
                        pad_c = npad;
                    }
#pragma unroll
                    for (int i = 0; i < 16; ++i)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int c = 8 * i + 2 * q + e;
                            if (!((vis[c >> 5] >> (c & 31)) & 1u)) s[4 * i + 2 * X + e] = 0xff800000u;   // -inf
                        }
                }
            } else if (need_mask) {
                // visible columns of row X: c <= cmax and (c >= cmin or c < csink); also drops whatever a half of S that
                // this block's QK^T did not write still holds
#pragma unroll
                for (int X = 0; X < 2; ++X) {
                    const int cmin = klo[X] - tokb, cmax = pos[X] - tokb;
#pragma unroll
                    for (int i = 0; i < 16; ++i)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int c = 8 * i + 2 * q + e;
                            if (c > cmax || (c < cmin && c >= csink)) s[4 * i + 2 * X + e] = 0xff800000u;
                        }
                }
            }
            // row max over the thread's columns, then over its group of four
            float mx[2];
#pragma unroll
            for (int X = 0; X < 2; ++X) {
                float ma = -INFINITY, mb = -INFINITY;
#pragma unroll
                for (int i = 0; i < 16; i += 2) {
                    ma = max3(ma, __uint_as_float(s[4 * i + 2 * X]), __uint_as_float(s[4 * i + 2 * X + 1]));
                    mb = max3(mb, __uint_as_float(s[4 * i + 4 + 2 * X]), __uint_as_float(s[4 * i + 4 + 2 * X + 1]));
                }
                float v = fmaxf(ma, mb);
                v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
                v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
                mx[X] = v * sl2;
            }
            // lazy rescale, as in the one-thread-per-row path (rows that hold nothing never ask for one)
            const bool growA = live[0] && mx[0] > m[0] + kRescaleThreshold, growB = live[1] && mx[1] > m[1] + kRescaleThreshold;
            if (__any_sync(0xffffffffu, growA || growB)) {
                float corr[2] = {1.f, 1.f};
                if (growA) { corr[0] = (m[0] == -INFINITY) ? 0.f : fast_exp2(m[0] - mx[0]); m[0] = mx[0]; l[0] *= corr[0]; }
                if (growB) { corr[1] = (m[1] == -INFINITY) ? 0.f : fast_exp2(m[1] - mx[1]); m[1] = mx[1]; l[1] *= corr[1]; }
                if (kb > 0) {
                    uint32_t o[D / 2];
                    if (D == 128) tmem_ld_16x256b_x16(tO, o); else tmem_ld_16x256b_x8(tO, o);
                    tmem_wait_ld();
#pragma unroll
                    for (int i = 0; i < D / 8; ++i)
#pragma unroll
                        for (int e = 0; e < 4; ++e) o[4 * i + e] = __float_as_uint(__uint_as_float(o[4 * i + e]) * corr[e >> 1]);
                    if (D == 128) tmem_st_16x256b_x16(tO, o); else tmem_st_16x256b_x8(tO, o);
                }
            }
            const float mref[2] = {(m[0] == -INFINITY) ? 0.f : m[0], (m[1] == -INFINITY) ? 0.f : m[1]};
            // p = 2^(s*scale*log2e - m), bf16 pairs -> P (aliases S[0, 64)); keys [0, 64) first so that their PV can start
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t pk[16];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int ib = 8 * h + i;
#pragma unroll
                    for (int X = 0; X < 2; ++X) {
                        if (X == 1 && !useB) { pk[2 * i + 1] = 0u; continue; }
                        const float p0 = fast_exp2(fmaf(__uint_as_float(s[4 * ib + 2 * X]), sl2, -mref[X]));
                        const float p1 = fast_exp2(fmaf(__uint_as_float(s[4 * ib + 2 * X + 1]), sl2, -mref[X]));
                        l[X] += p0 + p1;
                        pk[2 * i + X] = pack_bf16x2(p0, p1);
                    }
                }
                tmem_st_16x128b_x8(tS + 32 * h, pk);
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(smem_u32(&bars.p_full[tile][h]));
            }
        }
        // row sums over the groups of four (butterflies: every thread of a group ends with the same bits), then hand (m, l)
        // of rows g and g + 8 to the epilogue warpgroup
#pragma unroll
        for (int X = 0; X < 2; ++X) {
            l[X] += __shfl_xor_sync(0xffffffffu, l[X], 1);
            l[X] += __shfl_xor_sync(0xffffffffu, l[X], 2);
        }
        mbar_wait(smem_u32(&bars.stat_free[tile]), (n_st & 1) ^ 1);
        ++n_st;
        if (q == 0) {
            stats[tile][g] = make_float2(m[0], l[0]);
            stats[tile][g + 8] = make_float2(m[1], l[1]);
        }
        mbar_arrive(smem_u32(&bars.stat_full[tile]));
    }
}

}  // namespace

// RG: the plan has ragged streams (head segments with partial last pages in mid-stream).  The dense
// instantiation carries none of that code: inlined into the softmax loop it cost cfg2 3 % even when never taken.
// NARROW: every tile of the plan holds <= 16 valid rows (a decode-shaped plan): the softmax spreads a row over four threads.
template <int D, int NT, bool RG, bool NARROW>
__global__ void __launch_bounds__(kThreads, 1) attention_tc_kernel(const __grid_constant__ FwdParams p) {
    using C = Cfg<D, NT>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ Bars bars;
    __shared__ float2 stats[2][kTileRows];   // (m in log2 units, l) of a finished tile, softmax -> epilogue
    __shared__ int out_row16[kTileRows];     // epilogue: where each row of the tile goes in `out` (16-byte units, -1: nowhere)
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~static_cast<uintptr_t>(1023));
    const uint32_t sQ = smem_u32(smem);
    const uint32_t sKV = sQ + C::kSmemQ;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // this CTA's work items: a contiguous, cost-descending slice of the list (host-side LPT assignment)
    const int i_lo = p.cta_off[blockIdx.x], i_hi = p.cta_off[blockIdx.x + 1];
    const int G = p.G, TT = p.tile_tokens, ppb = kBlockKeys / p.P;
    const int rows_per_slot = kTileRows * p.tiles_per_item;
#ifdef SEGPA_TRACE
    int trace_n = 0;
#endif

    if (threadIdx.x == 0) {
        for (int s = 0; s < C::kStages; ++s) {
            mbar_init(smem_u32(&bars.kv_full[s]), 1);
            mbar_init(smem_u32(&bars.kv_empty[s]), 1);
        }
        for (int t = 0; t < 2; ++t) {
            mbar_init(smem_u32(&bars.q_full[t]), 1);
            mbar_init(smem_u32(&bars.q_empty[t]), 1);
            mbar_init(smem_u32(&bars.s_full[t]), 1);
            mbar_init(smem_u32(&bars.p_full[t][0]), 128);
            mbar_init(smem_u32(&bars.p_full[t][1]), 128);
            mbar_init(smem_u32(&bars.o_final[t]), 1);
            mbar_init(smem_u32(&bars.o_free[t]), 128);
            mbar_init(smem_u32(&bars.stat_full[t]), 128);
            mbar_init(smem_u32(&bars.stat_free[t]), 128);
        }
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
    // everything above overlapped the tail of the previous kernel of the stream (programmatic dependent launch); from
    // here on this kernel reads what that kernel wrote (K/V pages, partials' workspace, out)
    pdl_launch_dependents();
    pdl_wait();

    if (warp == kLoaderWarp || warp == kVLoaderWarp) {
        // ------------------------------------------------------------------ K/V loaders
        // Two warps: warp 0 fills the K stages, warp 3 the V stages (ring order K(j), V(j): even fills are K, odd
        // fills are V, and kStages is even, so a stage always belongs to the same warp).  The stages of K(j+1) and
        // V(j) are freed by the same step and both are needed by the next one; one warp issuing them one after the
        // other (about 600 cycles per stage of bulk copies plus the page-id fetch) put the second on the critical
        // path of every step (pipeline trace).
        reg_dec<kRegsLow>();
        const int kv = (warp == kLoaderWarp) ? 0 : 1;
        const uint8_t* pool = (kv == 0) ? p.k_pool : p.v_pool;
        uint32_t n_blk = 0;  // blocks filled so far (this warp's fill number is 2 * n_blk + kv)
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const ItemBlocks ib = item_blocks<NT>(it, sg, p.pads, TT, G);
            const int n_steps = ib.sb + ib.hi - ib.lo;
            // page ids are fetched one block ahead: the dependent global load of the next block is in flight
            // while this block's copies are issued (decode-shaped items consume a block every ~1500 cycles)
            const int* pg = p.pages + sg.page_off - sg.first_page + lane;
            auto blk = [&](int x) { return x < ib.sb ? x : ib.lo + (x - ib.sb); };
            int page_next = (lane < ppb && n_steps > 0) ? pg[(long long)blk(0) * ppb] : 0;
            for (int x = 0; x < n_steps; ++x) {
                const int j = blk(x);
                const int page = page_next;
                if (lane < ppb && x + 1 < n_steps) page_next = pg[(long long)blk(x + 1) * ppb];
                const uint32_t fill = 2 * n_blk + kv;
                const uint32_t st = fill % C::kStages, ph = (fill / C::kStages) & 1;
                TRACE(1, j * 2 + kv);
                if (lane == 0) {
                    mbar_wait(smem_u32(&bars.kv_empty[st]), ph ^ 1);
                    mbar_arrive_expect_tx(smem_u32(&bars.kv_full[st]), C::kTileBytes);
                }
                TRACE(2, j * 2 + kv);
                __syncwarp();
                if (lane < ppb)
                    bulk_g2s(sKV + st * C::kTileBytes + lane * p.page_bytes, pool + (size_t)page * p.page_bytes, p.page_bytes,
                             smem_u32(&bars.kv_full[st]));
                ++n_blk;
            }
        }
    } else if (warp == kMmaWarp) {
        // ------------------------------------------------------------------ MMA issuer
        // The whole warp walks the schedule and waits on the barriers (warp-uniform control flow);
        // one elected lane issues the tcgen05 instructions.
        reg_dec<kRegsLow>();
        constexpr uint32_t idesc_qk = make_idesc_bf16(128, 128, 0, 0);
        constexpr uint32_t idesc_qk64 = make_idesc_bf16(128, kHalfKeys, 0, 0);   // edge blocks: one 64-key half only
        constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, 0, 1);
        // descriptors differ from a base only in the start-address field: add (bytes >> 4)
        const uint64_t dq0 = make_desc_sw128(sQ, 16, kAtomBytes);
        const uint64_t dk0 = make_desc_sw128(sKV, 16, C::kSBO);
        const uint64_t dv0 = make_desc_sw128(sKV, kAtomBytes, C::kSBO);
        uint32_t rd = 0;                       // stage reads so far
        uint32_t n_q[2] = {0, 0}, n_p[2] = {0, 0}, n_of[2] = {0, 0};
        // the block whose PV is still to be issued, per tile (it may belong to the previous item)
        bool pv_valid[2] = {false, false}, pv_first[2] = {false, false}, pv_last[2] = {false, false};
        int pv_mask[2] = {0, 0};   // halves of the pending block that hold visible keys
        TileRange tr[2];
        tr[1].n_rows = 0; tr[1].lo = tr[1].hi = 0; tr[1].tok0 = 0;

        // One step of the continuous schedule: per tile, PV of the pending block, then QK^T of block j.
        // Ring order is K(j), V(j); V of the pending block was filled before K(j).
        auto step = [&](const bool have_k, const int j) {
            const bool have_v = pv_valid[0] || pv_valid[1];
            uint32_t st_v = 0, st_k = 0;
            TRACE(10, j);
            if (have_v) {
                st_v = rd % C::kStages;
                mbar_wait(smem_u32(&bars.kv_full[st_v]), (rd / C::kStages) & 1);
                ++rd;
            }
            if (have_k) {
                st_k = rd % C::kStages;
                mbar_wait(smem_u32(&bars.kv_full[st_k]), (rd / C::kStages) & 1);
                ++rd;
            }
            // per-tile part of the step (t is a compile-time constant so the per-tile state stays in registers)
            auto tile_part = [&](auto tile_c) {
                constexpr int t = decltype(tile_c)::value;
                const uint32_t tS = tmem + t * 128, tO = tmem + 256 + t * 128;
                const bool do_pv = pv_valid[t];
                const int am = (have_k && tr[t].n_rows > 0) ? half_mask(tr[t], j) : 0;
                const bool do_qk = am != 0;
                TRACE(11 + t * 4, j);
                const uint64_t dv = dv0 + (uint64_t)((st_v * C::kTileBytes) >> 4);
                const uint32_t acc0 = pv_first[t] ? 0u : 1u;
                if (do_pv) {
                    // PV starts as soon as the first 64 keys of P are in TMEM; the softmax warpgroup is still
                    // working on the other 64
                    mbar_wait(smem_u32(&bars.p_full[t][0]), n_p[t] & 1);
                    if (pv_first[t]) {   // first PV of an item overwrites O_t: the epilogue must have read it out
                        mbar_wait(smem_u32(&bars.o_free[t]), (n_of[t] & 1) ^ 1);
                        ++n_of[t];
                    }
                    tc_fence_after();
                    if ((pv_mask[t] & 1) && elect_one()) {
#pragma unroll
                        for (int kk = 0; kk < kHalfKeys / 16; ++kk)
                            mma_ts(tO, tS + kk * 8, dv + (uint64_t)((kk * 2 * C::kSBO) >> 4), idesc_pv, kk > 0 ? 1u : acc0);
                    }
                    __syncwarp();
                    mbar_wait(smem_u32(&bars.p_full[t][1]), n_p[t] & 1);
                    ++n_p[t];
                }
                if (do_qk && j == first_block(tr[t])) {
                    mbar_wait(smem_u32(&bars.q_full[t]), n_q[t] & 1);
                    ++n_q[t];
                }
                tc_fence_after();
                TRACE(12 + t * 4, j);
                if (elect_one()) {
                    if (do_pv) {
                        if (pv_mask[t] & 2) {   // (a half without visible keys is skipped: its P is zero anyway)
                            const uint32_t acc1 = (pv_mask[t] & 1) ? 1u : acc0;
#pragma unroll
                            for (int kk = kHalfKeys / 16; kk < kBlockKeys / 16; ++kk)
                                mma_ts(tO, tS + kk * 8, dv + (uint64_t)((kk * 2 * C::kSBO) >> 4), idesc_pv, kk > kHalfKeys / 16 ? 1u : acc1);
                        }
                        if (pv_last[t]) tc_commit(smem_u32(&bars.o_final[t]));
                    }
                    if (do_qk) {
                        const uint64_t dq = dq0 + (uint64_t)((t * C::kTileBytes) >> 4);
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
                        tc_commit(smem_u32(&bars.s_full[t]));
                        if (j == last_block(tr[t])) tc_commit(smem_u32(&bars.q_empty[t]));   // Q_t may be refilled
                    }
                }
                __syncwarp();
                TRACE(13 + t * 4, j);
                pv_valid[t] = do_qk;
                pv_mask[t] = am;
                pv_first[t] = do_qk && j == first_block(tr[t]);
                pv_last[t] = do_qk && j == last_block(tr[t]);
            };
            // A tile with no pending PV can have its QK^T issued at once; one with a pending PV first waits
            // for its softmax warpgroup.  Serve the former first (strided items: the two tiles alternate blocks,
            // so this is what lets the two chains overlap instead of waiting on each other).
            if (NT == 2) {
                const bool t1_first = pv_valid[0] && !pv_valid[1];
                if (t1_first) { tile_part(std::integral_constant<int, 1>{}); tile_part(std::integral_constant<int, 0>{}); }
                else { tile_part(std::integral_constant<int, 0>{}); tile_part(std::integral_constant<int, 1>{}); }
            } else {
                tile_part(std::integral_constant<int, 0>{});
            }
            if (elect_one()) {
                if (have_v) tc_commit(smem_u32(&bars.kv_empty[st_v]));
                if (have_k) tc_commit(smem_u32(&bars.kv_empty[st_k]));
            }
            __syncwarp();
        };

        // (one pass more than there are items: the last one only flushes the PV of the very last block; `step`
        // has a single call site on purpose -- it is large and every copy costs instruction-cache space)
        for (int ii = i_lo; ii <= i_hi; ++ii) {
            const bool flush = ii == i_hi;
            ItemBlocks ib;
            ib.sb = 0; ib.lo = 0; ib.hi = 1;
            if (!flush) {
                const ItemDev it = p.items[ii];
                const SegDev sg = p.segs[it.seg];
                ib = item_blocks<NT>(it, sg, p.pads, TT, G);
#pragma unroll
                for (int t = 0; t < NT; ++t) tr[t] = tile_range(it, sg, p.pads, t, TT, G);
#pragma unroll
                for (int t = 0; t < NT; ++t)
                    if (tr[t].n_rows > 0 && !has_blocks(tr[t])) {
                        // tile present but no block of its own in this (split) item: hand Q straight back
                        mbar_wait(smem_u32(&bars.q_full[t]), n_q[t] & 1);
                        ++n_q[t];
                        if (elect_one()) tc_commit(smem_u32(&bars.q_empty[t]));
                        __syncwarp();
                    }
            }
            const int n_steps = ib.sb + ib.hi - ib.lo;
            for (int x = 0; x < n_steps; ++x) step(!flush, x < ib.sb ? x : ib.lo + (x - ib.sb));
        }
    } else if (warp == kQWarp) {
        // ------------------------------------------------------------------ Q loader (TMA)
        // Q tile image: [D/64 halves][128 rows][128 B], SWIZZLE_128B; row r = (token, group head) as the
        // TMA box {64 elements, G heads, tile_tokens tokens} lays it out.  Rows >= G*tile_tokens are never
        // written (their scores are garbage and never stored); tokens past T are zero-filled by TMA.
        reg_dec<kRegsLow>();
        const uint32_t box_bytes = (uint32_t)(64 * 2 * G * TT);
        uint32_t n_fill[2] = {0, 0};
        if (lane == 0) prefetch_tmap(&p.q_map);
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            // pull the next item's Q tiles towards L2 while this one is computed
            const int in = ii + 1;
            if (in < i_hi && elect_one()) {
                const ItemDev itn = p.items[in];
                const SegDev sgn = p.segs[itn.seg];
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                    const TileRange trn = tile_range(itn, sgn, p.pads, t, TT, G);
                    if (trn.n_rows == 0) continue;
#pragma unroll
                    for (int h = 0; h < C::kHalves; ++h)
                        tma_prefetch_3d(&p.q_map, h * 64, sgn.kv_head * G, (int)(sgn.q_row_start + trn.tok0));
                }
            }
            __syncwarp();
#pragma unroll
            for (int t = 0; t < NT; ++t) {
                const TileRange tr = tile_range(it, sg, p.pads, t, TT, G);
                if (tr.n_rows == 0) continue;
                TRACE(40, t);
                mbar_wait(smem_u32(&bars.q_empty[t]), (n_fill[t] & 1) ^ 1);   // last QK^T on the old Q is done
                ++n_fill[t];
                TRACE(41, t);
                if (elect_one()) {
                    mbar_arrive_expect_tx(smem_u32(&bars.q_full[t]), box_bytes * C::kHalves);
#pragma unroll
                    for (int h = 0; h < C::kHalves; ++h)
                        tma_load_3d(sQ + t * C::kTileBytes + h * (kTileRows * 128), &p.q_map, h * 64, sg.kv_head * G,
                                    (int)(sg.q_row_start + tr.tok0), smem_u32(&bars.q_full[t]));
                }
                __syncwarp();
            }
        }
    } else if (warp < kFirstEpilogueWarp) {
        // ------------------------------------------------------------------ softmax warpgroups
        reg_inc<kRegsSoftmax>();
        const int tile = (warp - kFirstSoftmaxWarp) >> 2;
        if (NARROW) {
            if (tile < NT) softmax_narrow<D, RG>(p, bars, stats, tmem, tile, warp & 3, lane, i_lo, i_hi, TT, G);
        } else if (tile < NT) {
            const int wq = warp & 3;                       // TMEM lane quadrant this warp may access
            const int r = wq * 32 + lane;                  // row inside the tile
            const uint32_t lane_base = (uint32_t)(wq * 32) << 16;
            const uint32_t tS = tmem + lane_base + tile * 128;
            const uint32_t tO = tmem + lane_base + 256 + tile * 128;
            const float sl2 = p.scale * 1.4426950408889634f;
            uint32_t n_s = 0, n_st = 0;
            for (int ii = i_lo; ii < i_hi; ++ii) {
                const ItemDev it = p.items[ii];
                const SegDev sg = p.segs[it.seg];
                const TileRange tr = tile_range(it, sg, p.pads, tile, TT, G);
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
                float m_used = -INFINITY, l = 0.f;

                const int nb = n_blocks(tr);
                for (int kb = 0; kb < nb; ++kb) {
                    const int j = block_at(tr, kb);
                    TRACE(20, j);
                    mbar_wait(smem_u32(&bars.s_full[tile]), n_s & 1);
                    ++n_s;
                    tc_fence_after();
                    TRACE(21, j);
                    if (warp_has_rows) {
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
                                for (int w = 0; w < 4; ++w) {
                                    const int lo = min(max(a - 32 * w, 0), 32), hi = min(max(b - 32 * w, 0), 32);
                                    if (hi > lo) vis[w] |= (hi == 32 ? 0xffffffffu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
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
                        const float mx = fmaxf(fmaxf(mc[0], mc[1]), fmaxf(mc[2], mc[3]));
                        const float mx2 = mx * sl2;
                        // lazy rescale (warp-uniform decision: tcgen05.ld/st are warp-collective)
                        const bool grow = mx2 > m_used + kRescaleThreshold;
                        if (__any_sync(0xffffffffu, grow)) {
                            float corr = 1.f;
                            if (grow) {
                                corr = (m_used == -INFINITY) ? 0.f : fast_exp2(m_used - mx2);
                                m_used = mx2;
                                l *= corr;
                            }
                            if (kb > 0) {
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
                        }
                        TRACE(23, j);
                        const float mref = (m_used == -INFINITY) ? 0.f : m_used;
                        // p = 2^(s*scale*log2e - m) (masked columns: 2^-inf = 0), row sum, bf16 P -> TMEM (aliases S[0, 64))
                        const uint64_t sl2x2 = pack2(sl2, sl2), nmx2 = pack2(-mref, -mref);
                        uint64_t rsa = pack2(0.f, 0.f), rsb = pack2(0.f, 0.f);
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            uint32_t pk[16];
                            if (dead[c]) {
#pragma unroll
                                for (int q = 0; q < 16; ++q) pk[q] = 0u;
                                tmem_st16(tS + c * 16, pk);
                                if (c == 1) {
                                    tmem_wait_st();
                                    tc_fence_before();
                                    mbar_arrive(smem_u32(&bars.p_full[tile][0]));
                                }
                                continue;
                            }
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
                            tmem_st16(tS + c * 16, pk);
                            if (c == 1) {   // keys [0, 64) done: let their PV start
                                tmem_wait_st();
                                tc_fence_before();
                                mbar_arrive(smem_u32(&bars.p_full[tile][0]));
                            }
                        }
                        float rs0, rs1, rs2, rs3;
                        unpack2(rsa, rs0, rs1);
                        unpack2(rsb, rs2, rs3);
                        l += (rs0 + rs1) + (rs2 + rs3);
                        tmem_wait_st();
                    } else {
                        mbar_arrive(smem_u32(&bars.p_full[tile][0]));
                    }
                    tc_fence_before();
                    mbar_arrive(smem_u32(&bars.p_full[tile][1]));
                    TRACE(24, j);
                }
                // hand (m, l) to the epilogue warpgroup and go straight on to the next item
                mbar_wait(smem_u32(&bars.stat_free[tile]), (n_st & 1) ^ 1);
                ++n_st;
                stats[tile][r] = make_float2(m_used, l);
                mbar_arrive(smem_u32(&bars.stat_full[tile]));   // release: orders the store before the arrive
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue warpgroup
        reg_dec<kRegsEpilogue>();
        const int wq = warp & 3;
        const int r = wq * 32 + lane;
        const uint32_t lane_base = (uint32_t)(wq * 32) << 16;
        uint32_t n_o[2] = {0, 0}, n_st[2] = {0, 0};
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const ItemDev it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
#pragma unroll 1
            for (int tile = 0; tile < NT; ++tile) {
                const TileRange tr = tile_range(it, sg, p.pads, tile, TT, G);
                if (tr.n_rows == 0) continue;
                const uint32_t tO = tmem + lane_base + 256 + tile * 128;
                const bool has_blk = has_blocks(tr);
                const int rc = min(r, tr.n_rows - 1);
                const int tok = tr.tok0 + rc / G;
                const bool valid = r < tr.n_rows;
                const int head = sg.kv_head * G + rc % G;
                const long long row = sg.q_row_start + tok;
                TRACE(30, tile);
                mbar_wait(smem_u32(&bars.stat_full[tile]), n_st[tile] & 1);
                ++n_st[tile];
                const float2 ml = stats[tile][r];
                mbar_arrive(smem_u32(&bars.stat_free[tile]));
                if (has_blk) {
                    mbar_wait(smem_u32(&bars.o_final[tile]), n_o[tile] & 1);
                    ++n_o[tile];
                    tc_fence_after();
                }
                TRACE(31, tile);
                if (it.partial_slot >= 0) {
                    const size_t base = (size_t)it.partial_slot * rows_per_slot +
                                        ((it.flags & 1) ? (size_t)tile * kTileRows : (size_t)(tr.tok0 - it.t0) * G) + r;
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
                } else {
                    // Row r of the tile is one contiguous D-element row of `out`, but consecutive rows are far apart:
                    // a store straight from the TMEM layout (lane = row) touches 32 lines per instruction.  So each
                    // warp transposes its 32 rows through shared memory, 64 columns at a time (16-byte chunks
                    // XOR-swizzled by row, conflict-free both ways), and stores 4 full 128-byte lines per instruction.
                    const float inv = 1.f / ml.y;
                    const long long off16 = (row * p.out_row_stride + (long long)head * D) >> 3;
                    out_row16[r] = valid ? (int)off16 : -1;
                    const uint32_t stg = sKV + C::kSmemKV + wq * kOutWarpBytes;
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
                        if (h == D / 64 - 1 && has_blk) {   // O_t is in registers / shared memory now: the next item may overwrite it
                            tc_fence_before();
                            mbar_arrive(smem_u32(&bars.o_free[tile]));
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
                if (has_blk && it.partial_slot >= 0) {
                    tc_fence_before();
                    mbar_arrive(smem_u32(&bars.o_free[tile]));   // O_t may be overwritten by the next item
                }
                TRACE(32, tile);
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 3) tmem_dealloc(tmem, 512);
}

// ---------------------------------------------------------------------------------------------
template <int D, int NT, bool RG, bool NARROW>
static cudaError_t launch_one(const FwdParams& p, cudaStream_t st) {
    using C = Cfg<D, NT>;
    // the opt-in to > 48 KB of dynamic shared memory is per device: remember which devices have it
    static bool configured[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        cudaError_t e = cudaFuncSetAttribute(attention_tc_kernel<D, NT, RG, NARROW>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemBytes);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    return launch_pdl(attention_tc_kernel<D, NT, RG, NARROW>, dim3((unsigned)p.n_cta), dim3(kThreads), (size_t)C::kSmemBytes, st, p);
}

template <int D, int NT>
static cudaError_t launch_shape(const FwdParams& p, cudaStream_t st) {
    if (p.narrow) return p.has_ragged ? launch_one<D, NT, true, true>(p, st) : launch_one<D, NT, false, true>(p, st);
    return p.has_ragged ? launch_one<D, NT, true, false>(p, st) : launch_one<D, NT, false, false>(p, st);
}

cudaError_t launch_attention_tc(const FwdParams& p, cudaStream_t st) {
    if (p.n_items == 0) return cudaSuccess;
    if (p.tiles_per_item == 2) return p.D == 128 ? launch_shape<128, 2>(p, st) : launch_shape<64, 2>(p, st);
    // one tile per item: the schedule with two softmax warpgroups per tile (segpa_attn_tc1.cu), except for decode-shaped
    // plans, which keep this file's kernel (NARROW instantiation)
    if (!p.narrow) return launch_attention_tc1(p, st);
    if (p.has_ragged) return p.D == 128 ? launch_one<128, 1, true, true>(p, st) : launch_one<64, 1, true, true>(p, st);
    return p.D == 128 ? launch_one<128, 1, false, true>(p, st) : launch_one<64, 1, false, true>(p, st);
}

}  // namespace segpa
