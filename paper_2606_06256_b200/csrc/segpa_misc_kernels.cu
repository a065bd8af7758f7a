// Small kernels of libsegpa.so: page scatter (append), RoPEAlign, row gather, split-KV combine, LSE merge; and,
// in the test build only (-DSEGPA_BRINGUP -> libsegpa_bringup.so), the SIMT cross-check attention kernel.
#include "segpa_internal.h"
#include "sm100_ptx.cuh"

#include <type_traits>

#include <cuda_bf16.h>

namespace segpa {

// ---------------------------------------------------------------------------------------------
// a1: write K/V rows into the per-head page images.
// One launch serves a whole batch of streams: one thread per (slot, 16-byte chunk); the job a chunk
// belongs to is found by binary search over the jobs' chunk prefix.  Slots past the last new token of
// a job's last page are zeroed (masked probabilities multiply them, so they must stay finite).
// ---------------------------------------------------------------------------------------------
__global__ void scatter_pages_kernel(uint8_t* __restrict__ k_pool, uint8_t* __restrict__ v_pool,
                                     const ScatterJob* __restrict__ jobs, int n_jobs,
                                     const int* __restrict__ page_ids, long long total_chunks, int D, int P) {
    const int cpr = D >> 3;  // 16-byte chunks per row
    ptx::pdl_launch_dependents();
    ptx::pdl_wait();         // the pool pages may still be read by the previous kernel of the stream
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total_chunks;
         idx += (long long)gridDim.x * blockDim.x) {
        int lo = 0, hi = n_jobs - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (jobs[mid].chunk_begin <= idx) lo = mid; else hi = mid - 1;
        }
        const ScatterJob jb = jobs[lo];
        const long long local = idx - jb.chunk_begin;
        const long long n = local / cpr;
        const int c = (int)(local % cpr);
        const long long gs = jb.first_slot + n;
        const int page = page_ids[jb.page_off + gs / P];
        const int slot = (int)(gs % P);
        const size_t dst = (size_t)page * ((size_t)P * D * 2) + page_elem_offset_bytes(D, slot, c * 8);
        if (n >= jb.n_write) continue;   // tail slots that a later job of this batch fills (same stream, same page)
        uint4 kv = make_uint4(0, 0, 0, 0), vv = make_uint4(0, 0, 0, 0);
        if (n < jb.n_tokens) {
            kv = *reinterpret_cast<const uint4*>(jb.k_src + n * jb.src_stride + c * 8);
            vv = *reinterpret_cast<const uint4*>(jb.v_src + n * jb.src_stride + c * 8);
        }
        *reinterpret_cast<uint4*>(k_pool + dst) = kv;
        *reinterpret_cast<uint4*>(v_pool + dst) = vv;
    }
}

cudaError_t launch_scatter_pages(uint8_t* k_pool, uint8_t* v_pool, const ScatterJob* jobs_dev, int n_jobs,
                                 const int* page_ids_dev, long long total_chunks, int D, int P, cudaStream_t st) {
    if (total_chunks <= 0 || n_jobs <= 0) return cudaSuccess;
    const int threads = 256;
    long long blocks = (total_chunks + threads - 1) / threads;
    if (blocks > 148 * 64) blocks = 148 * 64;   // grid-stride beyond 64 CTAs per SM
    return launch_pdl(scatter_pages_kernel, dim3((unsigned)blocks), dim3(threads), 0, st, k_pool, v_pool, jobs_dev, n_jobs, page_ids_dev,
                      total_chunks, D, P);
}

// ---------------------------------------------------------------------------------------------
// RoPEAlign: K <- R(delta) K in place on the page images.  One thread per (token,
// 16-byte chunk of the first half of the head dim): it holds the 8 pairs (d, d + D/2), d = 8c .. 8c+7.
// HBM-bound: 2 * D * 2 bytes read + written per token.
// ---------------------------------------------------------------------------------------------
// One CTA per unit of kRopeUnitChunks chunks of one job (4 per thread, all eight loads of a thread in flight
// together).  Its prologue, before the wait on the preceding kernel, forms the job's cos / sin of
// delta * base^(-2d/D) in shared memory, in double precision (delta can be 10^5 and more: fp32 argument reduction
// would cost ~1e-3 rad), rounded once to fp32.  Index arithmetic is shifts and masks on 32-bit values (D / 16 and P
// are powers of two); round 2's first version (one chunk per thread, a binary search over the jobs and two 64-bit
// divisions per chunk, a separate table kernel) was bound by instruction issue at 0.66 of the HBM rate.
__global__ void __launch_bounds__(256, 4) rope_align_kernel(uint8_t* __restrict__ k_pool, const RopeJob* __restrict__ jobs, int n_jobs,
                                                         const int* __restrict__ page_ids, double rope_base, int D, int p_shift) {
    __shared__ float cs_s[64], sn_s[64];
    const int cph = D >> 4;                        // 16-byte chunks per half row: 4 or 8
    const int c_shift = cph == 8 ? 3 : 2;
    int lo = 0, hi = n_jobs - 1;                   // this CTA's job (uniform)
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (jobs[mid].unit_begin <= (int)blockIdx.x) lo = mid; else hi = mid - 1;
    }
    const RopeJob jb = jobs[lo];
    ptx::pdl_launch_dependents();
    if ((int)threadIdx.x < D / 2) {
        // theta_d = base^(-2d/D) = 2^(-(2d/D) log2 base); the angle is brought into [-pi, pi] first (2 pi in two
        // pieces: |delta * theta| < 2^40 leaves the reduced angle good to ~1e-9 rad) so that sincos takes its short path
        const double theta = exp2(-2.0 * (int)threadIdx.x / D * log2(rope_base));
        const double ang = (double)jb.delta_pos * theta;
        const double k = rint(ang * 0.15915494309189535);                    // 1 / (2 pi)
        const double r = fma(-k, 2.4492935982947064e-16, fma(-k, 6.283185307179586, ang));
        double sn, cs;
        sincos(r, &sn, &cs);
        cs_s[threadIdx.x] = (float)cs;
        sn_s[threadIdx.x] = (float)sn;
    }
    __syncthreads();
    const int c = (int)threadIdx.x & (cph - 1);    // the same for the four chunks of a thread: 256 is a multiple of cph
    float csv[8], snv[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { csv[i] = cs_s[c * 8 + i]; snv[i] = sn_s[c * 8 + i]; }
    const unsigned job_chunks = (unsigned)jb.n_tokens << c_shift;
    static_assert(kRopeUnitChunks == 4 * 256, "four chunks per thread");
    const unsigned local0 = (unsigned)((int)blockIdx.x - jb.unit_begin) * kRopeUnitChunks + threadIdx.x;
    const size_t page_bytes = ((size_t)D * 2) << p_shift;
    ptx::pdl_wait();                               // the K pages may still be read or written by the kernel before this one
    uint4* pa[4];
    uint4* pb[4];
    uint4 a4[4], b4[4];
    bool ok[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const unsigned local = local0 + i * 256;
        ok[i] = local < job_chunks;
        const unsigned gs = (unsigned)jb.first_slot + (local >> c_shift);
        if (ok[i]) {
            const size_t page = (size_t)page_ids[jb.page_off + (gs >> p_shift)] * page_bytes;
            const int slot = (int)(gs & ((1u << p_shift) - 1));
            pa[i] = reinterpret_cast<uint4*>(k_pool + page + page_elem_offset_bytes(D, slot, c * 8));
            pb[i] = reinterpret_cast<uint4*>(k_pool + page + page_elem_offset_bytes(D, slot, c * 8 + D / 2));
            a4[i] = *pa[i];
            b4[i] = *pb[i];
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (!ok[i]) continue;
        uint32_t* aw = reinterpret_cast<uint32_t*>(&a4[i]);
        uint32_t* bw = reinterpret_cast<uint32_t*>(&b4[i]);
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            uint32_t ra = 0, rb = 0;
#pragma unroll
            for (int hlf = 0; hlf < 2; ++hlf) {
                const float a = __uint_as_float(((aw[w] >> (16 * hlf)) & 0xffffu) << 16);
                const float b = __uint_as_float(((bw[w] >> (16 * hlf)) & 0xffffu) << 16);
                const float cs = csv[w * 2 + hlf], sn = snv[w * 2 + hlf];
                const float na = a * cs - b * sn, nb = a * sn + b * cs;
                ra |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(na)) << (16 * hlf);
                rb |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(nb)) << (16 * hlf);
            }
            aw[w] = ra;
            bw[w] = rb;
        }
        *pa[i] = a4[i];
        *pb[i] = b4[i];
    }
}

cudaError_t launch_rope_align(uint8_t* k_pool, const RopeJob* jobs_dev, int n_jobs, const int* page_ids_dev, int total_units,
                              double rope_base, int D, int P, cudaStream_t st) {
    if (total_units <= 0 || n_jobs <= 0) return cudaSuccess;
    return launch_pdl(rope_align_kernel, dim3((unsigned)total_units), dim3(256), 0, st, k_pool, jobs_dev, n_jobs, page_ids_dev,
                      rope_base, D, P == 32 ? 5 : 4);
}

// ---------------------------------------------------------------------------------------------
// Inverse of the scatter: page images -> rows [n][D] (export / read-back).  One thread per 16-byte chunk.
// ---------------------------------------------------------------------------------------------
__global__ void gather_rows_kernel(const uint8_t* __restrict__ k_pool, const uint8_t* __restrict__ v_pool,
                                   const int* __restrict__ page_ids, int first_slot, long long n_tokens,
                                   uint16_t* __restrict__ k_dst, uint16_t* __restrict__ v_dst, long long dst_stride,
                                   int D, int P) {
    const int cpr = D >> 3;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n_tokens * cpr;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long n = idx / cpr;
        const int c = (int)(idx % cpr);
        const long long gs = first_slot + n;
        const size_t src = (size_t)page_ids[gs / P] * ((size_t)P * D * 2) + page_elem_offset_bytes(D, (int)(gs % P), c * 8);
        if (k_dst) *reinterpret_cast<uint4*>(k_dst + n * dst_stride + c * 8) = *reinterpret_cast<const uint4*>(k_pool + src);
        if (v_dst) *reinterpret_cast<uint4*>(v_dst + n * dst_stride + c * 8) = *reinterpret_cast<const uint4*>(v_pool + src);
    }
}

cudaError_t launch_gather_rows(const uint8_t* k_pool, const uint8_t* v_pool, const int* page_ids_dev, int first_slot,
                               long long n_tokens, uint16_t* k_dst, uint16_t* v_dst, long long dst_stride, int D, int P,
                               cudaStream_t st) {
    const long long total = n_tokens * (D >> 3);
    if (total <= 0) return cudaSuccess;
    long long blocks = (total + 255) / 256;
    if (blocks > 148 * 32) blocks = 148 * 32;
    gather_rows_kernel<<<(unsigned)blocks, 256, 0, st>>>(k_pool, v_pool, page_ids_dev, first_slot, n_tokens, k_dst, v_dst,
                                                         dst_stride, D, P);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// segpa_gather_rows_noalloc: the same gather with its scratch -- the device copy of the page ids the range covers --
// in a fixed file-scope array instead of a staging buffer that grows with cudaMalloc.  For callers that may not
// allocate (code under CUDA graph capture, tight serving loops).  Every GPU that loads the library holds the array
// (kNoAllocMaxPages x 4 B = 64 KB) until the process exits.  All calls share it and it keeps the last call's ids: a call
// overwrites the entries it uses (nothing has to start at zero) in stream order, so calls on ONE stream are safe back to
// back, while calls that overlap on the GPU (different streams, no dependency between them) race on it.
// In host code `g_noalloc_page_ids` is a host-side stand-in for the symbol, not a device address: the address the kernel
// gets comes from cudaGetSymbolAddress, asked once per device with that device current.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) int g_noalloc_page_ids[kNoAllocMaxPages];

static cudaError_t noalloc_page_ids_ptr(int** out) {
    static int* ptr_of_device[64] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!ptr_of_device[dev]) {
        int* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_page_ids);
        if (e != cudaSuccess) return e;
        ptr_of_device[dev] = ptr;
    }
    *out = ptr_of_device[dev];
    return cudaSuccess;
}

// ids_host[0 .. n_ids): the page ids of the range (ordinary host memory: the copy stages them before it returns).
// No allocation: one stream-ordered copy into the fixed array; *ids_dev is what the gather kernel is then given.
cudaError_t noalloc_stage_page_ids(const int* ids_host, int n_ids, cudaStream_t st, const int** ids_dev) {
    if (n_ids < 1 || n_ids > kNoAllocMaxPages) return cudaErrorInvalidValue;   // (the entry point has already refused it with a message)
    int* ptr = nullptr;
    cudaError_t e = noalloc_page_ids_ptr(&ptr);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(ptr, ids_host, (size_t)n_ids * sizeof(int), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    *ids_dev = ptr;
    return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------
// a7: split-KV combine.  Partials hold unnormalised O, running max m (log2 units) and sum l;
// merged in ascending split order (deterministic).  Exactness of the merge: PAPER.md:302.
// One warp per row.
// ---------------------------------------------------------------------------------------------
// One warp folds partials s0, s0 + NW, ... (NB of them at a time, all loads issued before the first use) of a row into
// its running state (M, L, acc): fixed order, so the result does not depend on timing.
template <int D, int NB, int NW, class PartRow>
__device__ __forceinline__ void fold_partials(const FwdParams& p, PartRow part_row, int warp, int lane, int n_part, float& M, float& L,
                                              float (&acc)[D / 32]) {
    constexpr int EPL = D / 32;
    for (int s0 = warp; s0 < n_part; s0 += NW * NB) {
        float2 ml[NB];
        float ov[NB][EPL];
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int s = s0 + i * NW;
            const bool ok = s < n_part;
            const size_t base = part_row(ok ? s : s0);
            ml[i] = ok ? *reinterpret_cast<const float2*>(p.ws_ml + base * 2) : make_float2(-INFINITY, 0.f);
#pragma unroll
            for (int k = 0; k < EPL; ++k) ov[i][k] = ok ? p.ws_o[base * D + lane + 32 * k] : 0.f;
        }
        float mb = M;
#pragma unroll
        for (int i = 0; i < NB; ++i) mb = fmaxf(mb, ml[i].x);
        const float corr = (M == -INFINITY) ? 0.f : exp2f(M - mb);   // (mb = -inf only while every partial so far is empty)
        L *= corr;
#pragma unroll
        for (int k = 0; k < EPL; ++k) acc[k] *= corr;
        M = mb;
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const float w = (ml[i].x == -INFINITY) ? 0.f : exp2f(ml[i].x - M);
            L += w * ml[i].y;
#pragma unroll
            for (int k = 0; k < EPL; ++k) acc[k] += w * ov[i][k];
        }
    }
}

template <int D, int NW>
__global__ void __launch_bounds__(NW * 32) combine_kernel(const __grid_constant__ FwdParams p) {
    constexpr int EPL = D / 32;   // elements per lane
    // NW warps per block: warp w merges partials w, w + NW, ... of the block's row (8 when some tile has many
    // partials, a long decode context cut over the whole grid; 2 when every tile has a few)
    constexpr int NB = 12;        // partials a warp has in flight: all their loads are issued before the first is used
    __shared__ float s_acc[NW][D];
    __shared__ float2 s_ml[NW];
    const int rows_per_slot = kTileRows * p.tiles_per_item;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    ptx::pdl_launch_dependents();
    // block (x, y): comb x, rows y, y + gridDim.y, ...  One block per row.  Each warp folds its share of the row's
    // partials into a state (M, L, acc) of its own -- no pass over all the maxima first, so a row with up to 96 partials
    // costs ONE round trip to memory -- and warp 0 merges the NW states.  Every sum runs in a fixed order.
    // The descriptors were uploaded before the attention kernel started: their two dependent loads run while this
    // block still waits for that kernel (a decode-shaped layer is ~60 us, this kernel ~6 of them, all latency).
    const CombDev c = p.combs[blockIdx.x];
    const SegDev sg = p.segs[c.seg];
    ptx::pdl_wait();         // the partials are the attention kernel's
    const int rows = c.n_tok * p.G;
    // partials of row r: slot first_slot + s at row r; strided items hold a second one at row r + 128
    const int per_slot = (c.flags & 1) ? 2 : 1;
    const int n_part = c.n_splits * per_slot;
    for (int r = blockIdx.y; r < rows; r += gridDim.y) {
        auto part_row = [&](int s) {
            return (size_t)(c.first_slot + s / per_slot) * rows_per_slot + (size_t)(s % per_slot) * kTileRows + r;
        };
        float M = -INFINITY, L = 0.f;
        float acc[EPL];
#pragma unroll
        for (int k = 0; k < EPL; ++k) acc[k] = 0.f;
        if (n_part <= 2 * NW) fold_partials<D, 2, NW>(p, part_row, warp, lane, n_part, M, L, acc);   // (most tiles: a strided item or two)
        else fold_partials<D, NB, NW>(p, part_row, warp, lane, n_part, M, L, acc);
#pragma unroll
        for (int k = 0; k < EPL; ++k) s_acc[warp][lane + 32 * k] = acc[k];
        if (lane == 0) s_ml[warp] = make_float2(M, L);
        __syncthreads();
        if (warp == 0) {
            float Mt = -INFINITY;
#pragma unroll
            for (int w2 = 0; w2 < NW; ++w2) Mt = fmaxf(Mt, s_ml[w2].x);
            float Lt = 0.f;
            float tot[EPL];
#pragma unroll
            for (int k = 0; k < EPL; ++k) tot[k] = 0.f;
#pragma unroll
            for (int w2 = 0; w2 < NW; ++w2) {     // fixed order
                const float2 ml = s_ml[w2];
                const float w = (ml.x == -INFINITY) ? 0.f : exp2f(ml.x - Mt);
                Lt += w * ml.y;
#pragma unroll
                for (int k = 0; k < EPL; ++k) tot[k] += w * s_acc[w2][lane + 32 * k];
            }
            const int t = c.t0 + r / p.G, head = sg.kv_head * p.G + r % p.G;
            const long long row = sg.q_row_start + t;
            const float inv = 1.f / Lt;
#pragma unroll
            for (int k = 0; k < EPL; ++k)
                p.out[row * p.out_row_stride + (long long)head * D + lane + 32 * k] =
                    __bfloat16_as_ushort(__float2bfloat16_rn(tot[k] * inv));
            if (p.lse && lane == 0) p.lse[(long long)head * p.lse_stride + row] = (Mt + log2f(Lt)) * 0.6931471805599453f;
        }
        __syncthreads();
    }
}

cudaError_t launch_combine(const FwdParams& p, cudaStream_t st) {
    if (p.n_combs == 0) return cudaSuccess;
    const dim3 grid((unsigned)p.n_combs, (unsigned)(p.comb_max_rows < 1 ? 1 : (p.comb_max_rows > 256 ? 256 : p.comb_max_rows)));
    if (p.comb_max_parts <= 24)
        return p.D == 128 ? launch_pdl(combine_kernel<128, 2>, grid, dim3(64), 0, st, p) : launch_pdl(combine_kernel<64, 2>, grid, dim3(64), 0, st, p);
    return p.D == 128 ? launch_pdl(combine_kernel<128, 8>, grid, dim3(256), 0, st, p) : launch_pdl(combine_kernel<64, 8>, grid, dim3(256), 0, st, p);
}

// ---------------------------------------------------------------------------------------------
// LSE merge of two results over disjoint key sets.  One warp per (row, head), lanes over D.
// HBM-bound: 2 * D * 2 bytes read + D * 2 written per (row, head).
// ---------------------------------------------------------------------------------------------
// A warp takes 32 consecutive (row, head) units at a time: lane i loads the two LSE values of unit i and forms its
// weights (one load instruction per side for the 32 scattered values, lse being [Hq][T]), then the warp walks the units
// two at a time, every lane moving its D / 32 consecutive elements of the unit's rows with one load per side (8 bytes at
// D = 128).  The rows do not wait for the LSE values: a side whose weight turns out to be 0 is loaded and dropped.
template <int EPL>   // elements per lane: D / 32 = 2 or 4
__global__ void __launch_bounds__(256) merge_kernel(const uint16_t* __restrict__ out_a, const float* __restrict__ lse_a,
                                                    const uint16_t* __restrict__ out_b, const float* __restrict__ lse_b, uint16_t* out,
                                                    float* lse, long long row_stride, long long lse_stride, long long T, int Hq) {
    constexpr int D = EPL * 32;
    using Vec = typename std::conditional<EPL == 4, uint2, uint32_t>::type;
    const int lane = threadIdx.x & 31;
    const long long wid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    const long long n_units = T * Hq;
    for (long long g0 = wid * 32; g0 < n_units; g0 += nw * 32) {
        // this lane's unit: weights and merged LSE
        const long long um = g0 + lane;
        const bool okm = um < n_units;
        const long long rowm = okm ? um / Hq : 0;
        const int headm = okm ? (int)(um - rowm * Hq) : 0;
        const long long lidx = (long long)headm * lse_stride + rowm;
        const float la = okm ? lse_a[lidx] : -INFINITY, lb = okm ? lse_b[lidx] : -INFINITY;
        const long long basem = rowm * row_stride + (long long)headm * D;
        const float m = fmaxf(la, lb);
        float wam = 0.f, wbm = 0.f, l = -INFINITY;
        if (m != -INFINITY) {
            const float ea = expf(la - m), eb = expf(lb - m);     // exp(-inf) = 0
            wam = ea / (ea + eb);
            wbm = eb / (ea + eb);
            l = m + logf(ea + eb);
        }
        if (okm) lse[lidx] = l;
        const int n_here = (int)min((long long)32, n_units - g0);
#pragma unroll 1
        for (int i0 = 0; i0 < n_here; i0 += 2) {
            float wa[2], wb[2];
            long long base[2];
            Vec va[2], vb[2];
            bool ok[2];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int src = min(i0 + i, 31);
                ok[i] = i0 + i < n_here;
                base[i] = __shfl_sync(0xffffffffu, basem, src) + lane * EPL;
                wa[i] = __shfl_sync(0xffffffffu, wam, src);
                wb[i] = __shfl_sync(0xffffffffu, wbm, src);
                va[i] = *reinterpret_cast<const Vec*>(out_a + base[i]);      // (unit min(i, last): always inside the arrays)
                vb[i] = *reinterpret_cast<const Vec*>(out_b + base[i]);
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                if (!ok[i]) continue;
                // a side with weight 0 (lse = -inf) may hold anything, NaN included: it is not read into the sum
                if (wa[i] == 0.f) va[i] = Vec{};
                if (wb[i] == 0.f) vb[i] = Vec{};
                const uint32_t* pa = reinterpret_cast<const uint32_t*>(&va[i]);
                const uint32_t* pb = reinterpret_cast<const uint32_t*>(&vb[i]);
                Vec vo;
                uint32_t* po = reinterpret_cast<uint32_t*>(&vo);
#pragma unroll
                for (int w = 0; w < EPL / 2; ++w) {
                    const float a0 = __uint_as_float(pa[w] << 16), a1 = __uint_as_float(pa[w] & 0xffff0000u);
                    const float b0 = __uint_as_float(pb[w] << 16), b1 = __uint_as_float(pb[w] & 0xffff0000u);
                    const uint32_t r0 = __bfloat16_as_ushort(__float2bfloat16_rn(wa[i] * a0 + wb[i] * b0));
                    const uint32_t r1 = __bfloat16_as_ushort(__float2bfloat16_rn(wa[i] * a1 + wb[i] * b1));
                    po[w] = r0 | (r1 << 16);
                }
                *reinterpret_cast<Vec*>(out + base[i]) = vo;
            }
        }
    }
}

cudaError_t launch_merge(const uint16_t* out_a, const float* lse_a, const uint16_t* out_b, const float* lse_b, uint16_t* out,
                         float* lse, long long row_stride, long long lse_stride, long long T, int Hq, int D, cudaStream_t st) {
    const long long warps = (T * Hq + 31) / 32;
    if (warps <= 0) return cudaSuccess;
    long long blocks = (warps + 7) / 8;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (D == 128) merge_kernel<4><<<(unsigned)blocks, 256, 0, st>>>(out_a, lse_a, out_b, lse_b, out, lse, row_stride, lse_stride, T, Hq);
    else merge_kernel<2><<<(unsigned)blocks, 256, 0, st>>>(out_a, lse_a, out_b, lse_b, out, lse, row_stride, lse_stride, T, Hq);
    return cudaGetLastError();
}

#ifdef SEGPA_BRINGUP
// ---------------------------------------------------------------------------------------------
// SIMT cross-check attention (test build only): same plan, same outputs, no tensor cores.  One warp per query row;
// lanes split the head dim; keys visited one at a time.  Exists to validate the pool layout, the
// builder and the scheduler independently of the tcgen05 kernel.
// ---------------------------------------------------------------------------------------------
__device__ inline float bf16_bits_to_float(uint32_t b) { return __uint_as_float(b << 16); }

__global__ void attention_simt_kernel(FwdParams p) {
    __shared__ int s_item;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const int epl = p.D / 32;  // elements per lane (2 or 4)
    const float sl2 = p.scale * 1.4426950408889634f;
    const int rows_per_slot = kTileRows * p.tiles_per_item;
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(p.counter, 1);
        __syncthreads();
        const int ii = s_item;
        if (ii >= p.n_items) break;
        const ItemDev it = p.items[ii];
        const SegDev sg = p.segs[it.seg];
        const int rows = it.n_tok * p.G;
        for (int r = warp; r < rows; r += nw) {
            const int t = it.t0 + r / p.G, head = sg.kv_head * p.G + r % p.G;
            const long long row = sg.q_row_start + t;
            const int i = sg.kv_len - sg.q_len + t;
            float qv[4], acc[4] = {0.f, 0.f, 0.f, 0.f};
            for (int k = 0; k < epl; ++k)
                qv[k] = bf16_bits_to_float(p.q[row * p.q_row_stride + (long long)head * p.D + lane * epl + k]);
            float m = -INFINITY, l = 0.f;
            // the item's KV blocks are ranges of SLOTS (head segments start on fresh pages): first token at
            // or after a slot, and the slot of a token
            auto tok_at = [&](int u) {
                int start = 0, pad_c = 0;
                for (int k = 0; k < sg.n_pads; ++k) {
                    const PadDev pd = p.pads[sg.pad_off + k];
                    if (u < pd.tok + pad_c) return max(u, start) - pad_c;
                    start = pd.tok + pd.pad;
                    pad_c = pd.pad;
                }
                return max(u, start) - pad_c;
            };
            auto slot_of = [&](int j) {
                int pad = 0;
                for (int k = 0; k < sg.n_pads; ++k) {
                    const PadDev pd = p.pads[sg.pad_off + k];
                    if (pd.tok <= j) pad = pd.pad;
                }
                return j + pad;
            };
            int jlo = max(tok_at(it.kb_lo * kBlockKeys), i - sg.window + 1);
            int jhi = min(tok_at(it.kb_hi * kBlockKeys) - 1, i);
            // visible keys: sink tokens [0, n_sink) not already inside the window, then the window
            const int n_sink_keys = (it.kb_lo == 0) ? min(sg.n_sink, jlo) : 0;
            for (int jj = 0; jj < n_sink_keys + max(0, jhi - jlo + 1); ++jj) {
                const int j = jj < n_sink_keys ? jj : jlo + (jj - n_sink_keys);
                const int u = slot_of(j);
                const int pg = u / p.P, slot = u % p.P;
                const int page = p.pages[sg.page_off + (pg - sg.first_page)];
                const size_t off = (size_t)page * p.page_bytes;
                float dot = 0.f;
                float vv[4];
                for (int k = 0; k < epl; ++k) {
                    const uint32_t eo = page_elem_offset_bytes(p.D, slot, lane * epl + k);
                    dot += qv[k] * bf16_bits_to_float(*reinterpret_cast<const uint16_t*>(p.k_pool + off + eo));
                    vv[k] = bf16_bits_to_float(*reinterpret_cast<const uint16_t*>(p.v_pool + off + eo));
                }
                for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
                const float s2 = dot * sl2;
                const float mn = fmaxf(m, s2);
                const float corr = exp2f(m - mn);   // m = -inf first time: exp2(-inf) = 0
                const float pj = exp2f(s2 - mn);
                l = l * corr + pj;
                for (int k = 0; k < epl; ++k) acc[k] = acc[k] * corr + pj * vv[k];
                m = mn;
            }
            if (it.partial_slot >= 0) {
                const size_t base = (size_t)it.partial_slot * rows_per_slot + r;
                for (int k = 0; k < epl; ++k) p.ws_o[base * p.D + lane * epl + k] = acc[k];
                if (lane == 0) { p.ws_ml[base * 2] = m; p.ws_ml[base * 2 + 1] = l; }
            } else {
                const float inv = 1.f / l;
                for (int k = 0; k < epl; ++k)
                    p.out[row * p.out_row_stride + (long long)head * p.D + lane * epl + k] =
                        __bfloat16_as_ushort(__float2bfloat16_rn(acc[k] * inv));
                if (p.lse && lane == 0) p.lse[(long long)head * p.lse_stride + row] = (m + log2f(l)) * 0.6931471805599453f;
            }
        }
    }
}

cudaError_t launch_attention_simt(const FwdParams& p, cudaStream_t st) {
    attention_simt_kernel<<<p.num_sms * 4, 256, 0, st>>>(p);
    return cudaGetLastError();
}
#endif  // SEGPA_BRINGUP

}  // namespace segpa
