// Attention mass per key (by-product for SelectImportantTokens, Alg. 1 line 19):
//     mass[s][j] = sum over the query rows t and query heads g of segment s of p(t, g, j),
//     p(t, g, j) = exp(scale * q . k_j - LSE(t, g)) for visible j, 0 otherwise,
// recomputed from Q, the paged K and the LSE the fused attention wrote (the probabilities themselves never
// exist in memory).  Transposed formulation so that the sum over queries is an in-thread sum:
//     S^T = K_block Q_tile^T    (M = 128 keys = TMEM lanes, N = 128 query rows = columns)
// tcgen05.mma, B (the Q tile, by TMA) K-major from shared memory and A (the K block) from TENSOR MEMORY: the block is the
// same for every tile of an item, so it is copied once per item from its shared-memory page image into TMEM
// (tcgen05.cp.128x256b with the same SWIZZLE_128B descriptors an SS-mode MMA would read it through, one copy per 16
// head-dim columns; in order with the MMAs in the tensor pipe, so no barrier sits between copy and use and the copy of
// item i + 2 cannot overtake item i's MMAs) and the MMAs read half as much from shared memory.  TMEM: two K-block
// buffers [0, 128), three accumulator stages [128, 512).  One thread per key applies the visibility rule and ex2 to
// its 128 columns and keeps the running sum in a register.  A CTA owns a (segment, key block) item and loops over the
// query tiles that can see it: every mass entry is written exactly once, by one thread (deterministic, no atomics).
// Bound: the dense contraction is half of the attention kernel's (no PV) and the exponentials are the same, so the
// MUFU pipe (16 ex2 / clk / SM = 1024 clk per 128x128 tile) limits it at twice the MMA time.
//
// 16 warps: 0 loader (K block, Q tiles), 1 MMA issuer (and the K-block copies), 2-3 per-column LSE / position arrays (3
// also owns TMEM), 4-15 three exp warpgroups, warpgroup g on the tiles whose running number in the CTA's tile sequence
// is g mod 3 (accumulator stage g), all 128 query columns of a key in one thread, in four chunks of 32 with the TMEM
// load of the next chunk under the exponentials of the current one.
// Why several tiles in flight (round 2; ncu source page and the -DSEGPA_TRACE timeline): a tile costs an
// exp warp ~450-1100 cycles of serial latency around its exponentials (two mbarrier waits, the per-tile flags, the
// first TMEM load, the drain -- each a round trip through the instruction queue the other warps' ex2 sit in).  With
// two warpgroups that each took half of the columns of EVERY tile (round 1), all eight warps sat in that prologue
// together and the MUFU pipe idled (56 % busy, 1850 cycles per tile); with the warpgroups on different tiles one's
// prologue runs under the others' exponentials.  What was tried on top and did not pay is listed in DESIGN.md 5.7.
#include "segpa_internal.h"
#include "sm100_ptx.cuh"

namespace segpa {
using namespace ptx;

namespace {

constexpr int kExpGroups = 3;        // exp warpgroups = accumulator stages
constexpr int kMassThreads = 128 + 128 * kExpGroups;   // 4 service warps + the exp warpgroups
// register budgets (setmaxnreg): 128 * 56 + 384 * 144 = 62464 <= 512 * 128, the launch allocation
constexpr int kRegsService = 56, kRegsExp = 144;
// TMEM columns: the K block of the current and the next item as the MMA's A operand (bf16, D / 2 columns each), then the
// accumulator stages
constexpr uint32_t kColA = 0, kColS = 128;

struct alignas(16) MassAux {
    float lse2[kTileRows];   // LSE of column c in log2 units
    int pos[kTileRows];      // query position of column c; -1: no such row
    int pmin, pmax;          // over the valid columns
    int all_rows;            // every column has a row
    int pad;
};

constexpr int kQStages = 4;   // Q tiles in flight
constexpr int kSStages = kExpGroups;   // S accumulators in TMEM (128 columns each), one per exp warpgroup
constexpr int kKStages = 2;   // K blocks: the next item's block is loaded under the current item's last tiles
constexpr int kAuxStages = 8; // per-column arrays: an exp warpgroup needs those of its next tile (three on) the moment it
                              // finishes one, so the LSE warps must be able to run more than three tiles ahead

struct MassBars {
    uint64_t k_full[kKStages], k_empty[kKStages];
    uint64_t q_full[kQStages], q_empty[kQStages];
    uint64_t aux_full[kAuxStages], aux_empty[kAuxStages];
    uint64_t s_full[kSStages], s_empty[kSStages];
    uint32_t tmem_base;
};

}  // namespace

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

template <int D>
__global__ void __launch_bounds__(kMassThreads, 1) attention_mass_kernel(const __grid_constant__ MassParams p) {
    constexpr int kTileBytes = kTileRows * D * 2;
    constexpr int kHalves = D / 64;
    constexpr uint32_t kSBO = kHalves * kAtomBytes;
    extern __shared__ uint8_t smem_raw[];
    __shared__ MassBars bars;
    __shared__ MassAux aux[kAuxStages];
    __shared__ float part_sum[kExpGroups - 1][kTileRows];   // partial masses of the other three exp warpgroups, added by the first in a fixed order
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~static_cast<uintptr_t>(1023));
    const uint32_t sK = smem_u32(smem);           // kKStages K blocks
    const uint32_t sQ = sK + kKStages * kTileBytes;   // kQStages Q stages
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = p.G, TT = p.tile_tokens, ppb = kBlockKeys / p.P;
    const int i_lo = p.cta_off[blockIdx.x], i_hi = p.cta_off[blockIdx.x + 1];
#ifdef SEGPA_TRACE
    int trace_n = 0;
#endif

    if (threadIdx.x == 0) {
        for (int s = 0; s < kKStages; ++s) {
            mbar_init(smem_u32(&bars.k_full[s]), 1);
            mbar_init(smem_u32(&bars.k_empty[s]), 1);
        }
        for (int s = 0; s < kQStages; ++s) {
            mbar_init(smem_u32(&bars.q_full[s]), 1);
            mbar_init(smem_u32(&bars.q_empty[s]), 1);
        }
        for (int s = 0; s < kAuxStages; ++s) {
            mbar_init(smem_u32(&bars.aux_full[s]), 1);
            mbar_init(smem_u32(&bars.aux_empty[s]), 128);      // the one exp warpgroup that takes the tile
        }
        for (int s = 0; s < kSStages; ++s) {
            mbar_init(smem_u32(&bars.s_full[s]), 1);
            mbar_init(smem_u32(&bars.s_empty[s]), 128);
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

    if (warp == 0) {
        // ------------------------------------------------------------------ loader
        reg_dec<kRegsService>();
        uint32_t n_k = 0, n_t = 0;      // K fills, tile fills so far
        if (lane == 0) prefetch_tmap(&p.q_map);
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const MassItem it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const uint32_t ks = n_k % kKStages, kph = (n_k / kKStages) & 1;
            if (lane == 0) {
                mbar_wait(smem_u32(&bars.k_empty[ks]), kph ^ 1);
                mbar_arrive_expect_tx(smem_u32(&bars.k_full[ks]), kTileBytes);
            }
            __syncwarp();
            if (lane < ppb) {
                const int page = p.pages[sg.page_off + (long long)(it.kb * ppb - sg.first_page) + lane];
                bulk_g2s(sK + ks * kTileBytes + lane * p.page_bytes, p.k_pool + (size_t)page * p.page_bytes, p.page_bytes,
                         smem_u32(&bars.k_full[ks]));
            }
            ++n_k;
            for (int ti = it.t_lo; ti < it.t_hi; ++ti, ++n_t) {
                const uint32_t st = n_t % kQStages, ph = (n_t / kQStages) & 1;
                const int tok0 = ti * TT;
                if (lane == 0) {
                    mbar_wait(smem_u32(&bars.q_empty[st]), ph ^ 1);
                    mbar_arrive_expect_tx(smem_u32(&bars.q_full[st]), (uint32_t)(64 * 2 * G * TT) * kHalves);
#pragma unroll
                    for (int h = 0; h < kHalves; ++h)
                        tma_load_3d(sQ + st * kTileBytes + h * (kTileRows * 128), &p.q_map, h * 64, sg.kv_head * G,
                                    (int)(sg.q_row_start + tok0), smem_u32(&bars.q_full[st]));
                }
                __syncwarp();
            }
        }
    } else if (warp == 2 || warp == 3) {
        // ------------------------------------------------------------------ per-column LSE / position arrays of each tile
        // (two warps, one per stage: warp 2 serves the even tiles, warp 3 the odd ones -- a tile costs one
        // round trip to L2 for the LSE values, which one warp alone cannot hide)
        reg_dec<kRegsService>();
        // One tile ahead: the LSE loads of this warp's next tile are issued before the current tile's values are used,
        // so the round trip to L2 runs under the current tile's work (without it each of the two warps was busy ~95 %
        // of the time once the exp warps stopped being the limit).  cur / nxt walk the CTA's (item, tile) sequence,
        // taking the tiles whose running number has this warp's parity.
        struct Cursor {
            int ii, ti, t_hi;
            uint32_t n_t;
            int q_len, p0, head0;          // of the item's segment: rows, position of row 0, first query head
            long long row0;
            bool valid;
        };
        const int par = warp - 2;
        auto open_item = [&](Cursor& c) {
            const MassItem it = p.items[c.ii];
            const SegDev sg = p.segs[it.seg];
            c.ti = it.t_lo; c.t_hi = it.t_hi;
            c.q_len = sg.q_len; c.p0 = sg.kv_len - sg.q_len; c.head0 = sg.kv_head * G; c.row0 = sg.q_row_start;
        };
        auto step = [&](Cursor& c) {       // to the next tile of the sequence
            ++c.n_t;
            if (++c.ti == c.t_hi) {
                if (++c.ii == i_hi) { c.valid = false; return; }
                open_item(c);
            }
        };
        // column c of a full tile is token c / G, head c % G: per lane, once
        int ctok[4], chead[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { ctok[u] = (lane + 32 * u) / G; chead[u] = (lane + 32 * u) % G; }
        auto issue = [&](const Cursor& c, float (&l2)[4], int (&pos)[4]) {
            const int tok0 = c.ti * TT;
            const int n_rows = min(TT, c.q_len - tok0) * G;
            // the four LSE loads of a lane are issued together (clamped to a valid row)
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                int tk = ctok[u], hd = chead[u];
                if (lane + 32 * u >= n_rows) { tk = (n_rows - 1) / G; hd = (n_rows - 1) % G; }   // ragged last tile only
                pos[u] = c.p0 + tok0 + tk;
                l2[u] = p.lse[(long long)(c.head0 + hd) * p.lse_stride + c.row0 + tok0 + tk];
            }
        };
        Cursor cur;
        cur.ii = i_lo; cur.n_t = 0; cur.valid = i_lo < i_hi;
        if (cur.valid) {
            open_item(cur);
            if (par == 1) step(cur);
        }
        float l2[4] = {0.f, 0.f, 0.f, 0.f};
        int pos[4] = {0, 0, 0, 0};
        if (cur.valid) issue(cur, l2, pos);
        while (cur.valid) {
            Cursor nxt = cur;
            step(nxt);
            if (nxt.valid) step(nxt);
            float l2n[4] = {0.f, 0.f, 0.f, 0.f};
            int posn[4] = {0, 0, 0, 0};
            if (nxt.valid) issue(nxt, l2n, posn);
            const uint32_t st = cur.n_t % kAuxStages, ph = (cur.n_t / kAuxStages) & 1;
            const int n_rows = min(TT, cur.q_len - cur.ti * TT) * G;
            // columns past the segment's rows: position -1 (their scores are garbage and never counted)
            int pmin = INT32_MAX, pmax = -1;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (lane + 32 * u < n_rows) {
                    l2[u] *= 1.4426950408889634f;
                    pmin = min(pmin, pos[u]);
                    pmax = max(pmax, pos[u]);
                } else {
                    pos[u] = -1;
                    l2[u] = 0.f;
                }
            }
            pmin = __reduce_min_sync(0xffffffffu, pmin);
            pmax = __reduce_max_sync(0xffffffffu, pmax);
            TRACE(30, cur.n_t);
            if (lane == 0) mbar_wait(smem_u32(&bars.aux_empty[st]), ph ^ 1);
            __syncwarp();
            TRACE(31, cur.n_t);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                aux[st].pos[lane + 32 * u] = pos[u];
                aux[st].lse2[lane + 32 * u] = l2[u];
            }
            if (lane == 0) { aux[st].pmin = pmin; aux[st].pmax = pmax; aux[st].all_rows = n_rows == kTileRows; }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&bars.aux_full[st]));
            TRACE(32, cur.n_t);
            cur = nxt;
#pragma unroll
            for (int u = 0; u < 4; ++u) { l2[u] = l2n[u]; pos[u] = posn[u]; }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer: S^T = K Q^T
        reg_dec<kRegsService>();
        constexpr uint32_t idesc = make_idesc_bf16(128, 128, 0, 0);
        const uint64_t dk0 = make_desc_sw128(sK, 16, kSBO);             // A: K block image (page layout)
        const uint64_t dq0 = make_desc_sw128(sQ, 16, kAtomBytes);       // B: Q tile image (TMA box layout)
        uint32_t n_k = 0, n_t = 0;
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const MassItem it = p.items[ii];
            const uint32_t ks = n_k % kKStages;
            mbar_wait(smem_u32(&bars.k_full[ks]), (n_k / kKStages) & 1);
            ++n_k;
            const uint64_t dk = dk0 + (uint64_t)((ks * kTileBytes) >> 4);
            // The K block is the A operand of every tile of the item: copied once into TMEM (tcgen05.cp, in order with the
            // MMAs in the tensor pipe: no barrier between them, and the copy for item i + 2 cannot overtake item i's MMAs),
            // so that the MMAs read only the Q tile from shared memory -- half of the operand traffic.
            const uint32_t tA = tmem + kColA + ((n_k - 1) & 1) * 64;
            if (elect_one()) {
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t ok = ((kk / 4) * kAtomBytes + (kk % 4) * 32) >> 4;
                    tmem_cp_128x256b(tA + kk * 8, dk + ok);
                }
                tc_commit(smem_u32(&bars.k_empty[ks]));      // the K stage is free as soon as the copies have completed
            }
            __syncwarp();
            for (int ti = it.t_lo; ti < it.t_hi; ++ti, ++n_t) {
                const uint32_t qs = n_t % kQStages, qph = (n_t / kQStages) & 1;
                const uint32_t st = n_t % kSStages, ph = (n_t / kSStages) & 1;
                TRACE(10, n_t);
                mbar_wait(smem_u32(&bars.q_full[qs]), qph);
                TRACE(11, n_t);
                mbar_wait(smem_u32(&bars.s_empty[st]), ph ^ 1);
                TRACE(12, n_t);
                tc_fence_after();
                if (elect_one()) {
                    const uint64_t dq = dq0 + (uint64_t)((qs * kTileBytes) >> 4);
#pragma unroll
                    for (int kk = 0; kk < D / 16; ++kk) {
                        const uint32_t oq = ((kk / 4) * (kTileRows * 128) + (kk % 4) * 32) >> 4;
                        mma_ts(tmem + kColS + st * 128, tA + kk * 8, dq + oq, idesc, kk > 0 ? 1u : 0u);
                    }
                    tc_commit(smem_u32(&bars.s_full[st]));
                    tc_commit(smem_u32(&bars.q_empty[qs]));
                }
                __syncwarp();
            }
        }
    } else if (warp >= 4) {
        // ------------------------------------------------------------------ exp warpgroups: thread = (key, every third tile)
        // Warpgroup g (warps 4 + 4g ...) takes the tiles with running number = g mod 3: accumulator stage g.  A thread
        // walks its key's 128 query columns in four chunks of 32, the TMEM load of the next chunk in flight under the
        // exponentials of the current one; the accumulator stage goes back to the MMA issuer as soon as the last
        // chunk is in registers.  The partial sums of a key are added in a fixed order.
        reg_inc<kRegsExp>();
        const int wq = warp & 3;
        const int grp = (warp - 4) >> 2;
        const int kr = wq * 32 + lane;                                   // key row inside the block
        const uint32_t t_base = tmem + ((uint32_t)(wq * 32) << 16) + kColS + grp * 128;
        const float sl2 = p.scale * 1.4426950408889634f;
        uint32_t n_t = 0;
        for (int ii = i_lo; ii < i_hi; ++ii) {
            const MassItem it = p.items[ii];
            const SegDev sg = p.segs[it.seg];
            const int key = it.kb * kBlockKeys + kr;
            const int blk_lo = it.kb * kBlockKeys, blk_hi = blk_lo + kBlockKeys - 1;
            const bool is_sink_key = key < sg.n_sink;
            float acc = 0.f;
            for (int ti = it.t_lo; ti < it.t_hi; ++ti, ++n_t) {
                if ((int)(n_t % kExpGroups) != grp) continue;
                static_assert(kSStages == kExpGroups, "accumulator stage = exp warpgroup");
                const uint32_t ph = (n_t / kSStages) & 1;
                const uint32_t as = n_t % kAuxStages, aph = (n_t / kAuxStages) & 1;
                TRACE(20, n_t);
                mbar_wait(smem_u32(&bars.aux_full[as]), aph);
                TRACE(21, n_t);
                mbar_wait(smem_u32(&bars.s_full[grp]), ph);
                TRACE(22, n_t);
                tc_fence_after();
                uint32_t sa[32], sb[32];
                tmem_ld32(t_base, sa);
                const MassAux& ax = aux[as];
                // the whole block is visible to every valid column of the tile: causal (blk_hi <= pmin) and inside
                // the window of the latest query (blk_lo > pmax - W); columns without a row have position -1
                const int4 fl = *reinterpret_cast<const int4*>(&ax.pmin);
                const bool full = fl.z != 0 && blk_hi <= fl.x && blk_lo > fl.y - sg.window;
                float pa = 0.f, pb = 0.f, pc = 0.f, pd = 0.f;
                auto chunk = [&](const uint32_t (&s)[32], const int c0) {
                    if (full) {
#pragma unroll
                        for (int e = 0; e < 32; e += 4) {
                            const float4 l4 = *reinterpret_cast<const float4*>(&ax.lse2[c0 + e]);
                            pa += fast_exp2(fmaf(__uint_as_float(s[e + 0]), sl2, -l4.x));
                            pb += fast_exp2(fmaf(__uint_as_float(s[e + 1]), sl2, -l4.y));
                            pc += fast_exp2(fmaf(__uint_as_float(s[e + 2]), sl2, -l4.z));
                            pd += fast_exp2(fmaf(__uint_as_float(s[e + 3]), sl2, -l4.w));
                        }
                    } else {
#pragma unroll
                        for (int e = 0; e < 32; e += 4) {
                            const float4 l4 = *reinterpret_cast<const float4*>(&ax.lse2[c0 + e]);
                            const int4 p4 = *reinterpret_cast<const int4*>(&ax.pos[c0 + e]);
                            const float e0 = fast_exp2(fmaf(__uint_as_float(s[e + 0]), sl2, -l4.x));
                            const float e1 = fast_exp2(fmaf(__uint_as_float(s[e + 1]), sl2, -l4.y));
                            const float e2 = fast_exp2(fmaf(__uint_as_float(s[e + 2]), sl2, -l4.z));
                            const float e3 = fast_exp2(fmaf(__uint_as_float(s[e + 3]), sl2, -l4.w));
                            pa += (key <= p4.x && (key > p4.x - sg.window || is_sink_key)) ? e0 : 0.f;
                            pb += (key <= p4.y && (key > p4.y - sg.window || is_sink_key)) ? e1 : 0.f;
                            pc += (key <= p4.z && (key > p4.z - sg.window || is_sink_key)) ? e2 : 0.f;
                            pd += (key <= p4.w && (key > p4.w - sg.window || is_sink_key)) ? e3 : 0.f;
                        }
                    }
                };
                tmem_wait_ld();
                TRACE(23, n_t);
                tmem_ld32(t_base + 32, sb);
                chunk(sa, 0);
                tmem_wait_ld();
                tmem_ld32(t_base + 64, sa);
                chunk(sb, 32);
                tmem_wait_ld();
                tmem_ld32(t_base + 96, sb);
                // the accumulator stage goes back at the half-way point, at the price of one exposed TMEM load (the
                // other warps of the scheduler fill it): the MMA of the stage's next tile takes ~1500 cycles from this
                // arrive to a visible s_full (wait latency + the MMAs + commit + wait latency), more than one chunk
                tmem_wait_ld();
                tc_fence_before();
                mbar_arrive(smem_u32(&bars.s_empty[grp]));
                chunk(sa, 64);
                chunk(sb, 96);
                acc += (pa + pb) + (pc + pd);
                TRACE(24 + (full ? 0 : 1), n_t);
                mbar_arrive(smem_u32(&bars.aux_empty[as]));
            }
            // mass = ((tiles 0 mod 3) + (1 mod 3)) + (2 mod 3), added by the first warpgroup: one writer per entry, one order
            if (grp > 0) part_sum[grp - 1][kr] = acc;
            asm volatile("bar.sync 1, 384;" ::: "memory");
            if (grp == 0 && key < sg.kv_len)
                p.mass[p.mass_off[it.seg] + key] = (acc + part_sum[0][kr]) + part_sum[1][kr];
            asm volatile("bar.sync 2, 384;" ::: "memory");
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 3) tmem_dealloc(tmem, 512);
}

template <int D>
static cudaError_t launch_mass_one(const MassParams& p, cudaStream_t st) {
    constexpr int smem = (kKStages + kQStages) * kTileRows * D * 2 + 1024;
    // the opt-in to > 48 KB of dynamic shared memory is per device: remember which devices have it
    static bool configured[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        cudaError_t e = cudaFuncSetAttribute(attention_mass_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    attention_mass_kernel<D><<<p.n_cta, kMassThreads, smem, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_attention_mass(const MassParams& p, cudaStream_t st) {
    if (p.n_cta == 0) return cudaSuccess;
    return p.D == 128 ? launch_mass_one<128>(p, st) : launch_mass_one<64>(p, st);
}

// ---------------------------------------------------------------------------------------------
// Selection: per segment, the smallest set of keys whose cumulative mass reaches tau * (total mass)
// ("the smallest set of tokens whose cumulative attention mass exceeds a threshold tau").
// One block per segment; bisection over the bit pattern of the (non-negative) fp32 masses finds the largest
// threshold t with sum{m >= t} >= tau * total; keys with m > t are selected, and of the keys with m == t as
// many (lowest positions first) as are still needed.  Sums run in a fixed order (deterministic).
// ---------------------------------------------------------------------------------------------
__device__ float block_sum(float v, float* red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    float t = 0.f;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
    return t;
}

__global__ void mass_select_kernel(const float* __restrict__ mass, const long long* __restrict__ mass_off, const int* __restrict__ kv_len,
                                   float tau, unsigned char* __restrict__ selected, int* __restrict__ n_selected) {
    __shared__ float red[32];
    const int seg = blockIdx.x, n = kv_len[seg];
    const float* m = mass + mass_off[seg];
    unsigned char* sel = selected + mass_off[seg];
    float tot = 0.f;
    for (int j = threadIdx.x; j < n; j += blockDim.x) tot += m[j];
    tot = block_sum(tot, red);
    const float need = tau * tot;
    // largest bit pattern t with sum{m >= t} >= need (masses are >= 0: their bit patterns order like the values)
    unsigned lo = 0u, hi = 0x7f800000u;
    while (lo < hi) {
        const unsigned mid = lo + (hi - lo + 1) / 2;
        float sum = 0.f;
        for (int j = threadIdx.x; j < n; j += blockDim.x) sum += (__float_as_uint(m[j]) >= mid) ? m[j] : 0.f;
        sum = block_sum(sum, red);
        if (sum >= need) lo = mid; else hi = mid - 1;
    }
    float above = 0.f;
    for (int j = threadIdx.x; j < n; j += blockDim.x) above += (__float_as_uint(m[j]) > lo) ? m[j] : 0.f;
    above = block_sum(above, red);
    const float tval = __uint_as_float(lo);
    // ties at the threshold: take the lowest positions until the mass is reached
    int ties_needed = 0;
    if (tval > 0.f) {
        const float rest = need - above;
        ties_needed = rest > 0.f ? (int)ceilf(rest / tval) : 0;
    }
    __syncthreads();
    // The tie rule is positional: key j at the threshold is taken when fewer than ties_needed threshold keys lie before
    // it.  Every thread takes a contiguous range of positions, counts the threshold keys in it, a block-wide exclusive
    // scan of those counts gives the number before the range, and the thread then walks its range.  (One thread walking
    // the whole stream took ~80 us of the kernel's 190 on cfg2's 4 800-key segments.)
    __shared__ int wsum[32];
    const int per = (n + (int)blockDim.x - 1) / (int)blockDim.x;
    const int j0 = min(n, (int)threadIdx.x * per), j1 = min(n, j0 + per);
    int mine = 0;
    for (int j = j0; j < j1; ++j) mine += __float_as_uint(m[j]) == lo;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = mine;
    for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    int before = incl - mine;
    for (int w2 = 0; w2 < warp; ++w2) before += wsum[w2];
    int taken = before, cnt = 0;
    for (int j = j0; j < j1; ++j) {
        const unsigned b = __float_as_uint(m[j]);
        unsigned char sv = 0;
        if (b > lo) sv = 1;
        else if (b == lo && taken < ties_needed) sv = 1;
        taken += b == lo;
        sel[j] = sv;
        cnt += sv;
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    __syncthreads();
    if (lane == 0) wsum[warp] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot_sel = 0;
        for (int w2 = 0; w2 < (int)(blockDim.x >> 5); ++w2) tot_sel += wsum[w2];
        n_selected[seg] = tot_sel;
    }
}

cudaError_t launch_mass_select(const float* mass, const long long* mass_off_dev, const int* kv_len_dev, int n_segments, float tau,
                               unsigned char* selected, int* n_selected, cudaStream_t st) {
    if (n_segments <= 0) return cudaSuccess;
    mass_select_kernel<<<n_segments, 1024, 0, st>>>(mass, mass_off_dev, kv_len_dev, tau, selected, n_selected);
    return cudaGetLastError();
}

}  // namespace segpa
