// Internal structures shared by the host runtime and the CUDA kernels of libsegpa.so.
// Not part of the ABI (include/segpa.h is).  Nothing here is used by oracle/.
#pragma once

#include <cstdint>
#include <cuda_runtime.h>
#include <utility>

namespace segpa {

constexpr int kBlockKeys = 128;   // KV block (keys per MMA tile column block)
constexpr int kTileRows = 128;    // query rows per tile (UMMA M)
constexpr int kAtomBytes = 1024;  // one swizzle-128B atom: 8 rows x 128 B

// ---------------------------------------------------------------------------------------------
// Page image.  A physical page holds P tokens x D bf16 of ONE KV head,
// stored as the exact shared-memory image tcgen05.mma consumes, so one cp.async.bulk moves it:
//   for g in [0, P/8)          group of 8 tokens
//     for h in [0, D/64)       64-element (128-byte) half of the head dim
//       atom: 8 rows x 128 B; the 16-byte chunk c of row r is stored at chunk (c ^ r)   (SW128)
// byte offset of (slot s, element d):
//   (s/8)*(D/64)*1024 + (d/64)*1024 + (s%8)*128 + ((((d%64)/8) ^ (s%8)) * 16) + (d%8)*2
// The same image serves K (K-major B operand of S = Q K^T; SBO = (D/64)*1024) and V (MN-major B
// operand of O = P V; SBO = (D/64)*1024, LBO = 1024).
// ---------------------------------------------------------------------------------------------
__host__ __device__ inline uint32_t page_elem_offset_bytes(int D, int slot, int d) {
    const int halves = D >> 6;
    const int r = slot & 7;
    return (uint32_t)((slot >> 3) * halves * kAtomBytes + (d >> 6) * kAtomBytes + r * 128 +
                      ((((d & 63) >> 3) ^ r) << 4) + ((d & 7) << 1));
}

struct SegDev {
    long long q_row_start;
    long long page_off;     // index into the page-id array of this segment's first listed page
    int q_len;
    int kv_len;
    int head_class;         // 0 GLOBAL, 1 LOCAL
    int window;             // W (keys incl. self); large for GLOBAL
    int n_sink;
    int kv_head;
    int first_page;         // absolute page index (slot / P) of page_off
    int n_pages_listed;
    int pad_off;            // ragged streams (head segments with partial last pages): index of the stream's
    int n_pads;             //   first PadDev and their number (0: token j sits at slot j)
};

// Token -> slot map of a ragged stream: tokens >= tok (up to the next entry) sit at slot token + pad; the slots
// [tok + previous pad, tok + pad) behind the previous head segment's tail hold no token.
struct PadDev {
    int tok;
    int pad;
};

struct ItemDev {
    int seg;
    int t0;                 // first token of the item inside the segment's query range
    int n_tok;              // tokens (rows = n_tok * G), <= tiles_per_item * tile_tokens
    int kb_lo;              // visited KV blocks [kb_lo, kb_hi)
    int kb_hi;
    int partial_slot;       // -1: final result written to out/lse; else split-KV partial slot
    int flags;              // bit 0: strided (both tiles hold the same rows and take alternate KV blocks)
    int cost;               // KV blocks the item visits (scheduling only; < kb_hi - kb_lo for sink segments)
    // Ragged streams only (SegDev::n_pads > 0; zero otherwise): per tile slot t of the item, the slots of the first key
    // any of its rows sees, of the last one, and of its last sink key (a dense stream has slot = token and the kernel
    // forms them itself).  Looked up on the host so that no role of the kernel walks the token -> slot map per item.
    int slots[2][3];
    int pad_[2];
};
static_assert(sizeof(ItemDev) == 64, "ItemDev is read as four 16-byte words");

struct CombDev {
    int seg;
    int t0;
    int n_tok;
    int first_slot;
    int n_splits;
    int flags;              // bit 0: strided items: every slot holds two partials of the same rows (at +0 and +128)
    int pad1, pad2;
};

// 128-byte TMA descriptor (CUtensorMap) of Q viewed as [T][Hq][D]; encoded per attention_fwd call.
struct alignas(64) TensorMap {
    unsigned long long opaque[16];
};

struct FwdParams {
    TensorMap q_map;             // box {64 elements, G heads, tile_tokens tokens}, SWIZZLE_128B
    const SegDev* segs;
    const ItemDev* items;
    const int* pages;            // translated physical page ids (zero page = num_pages)
    const PadDev* pads;          // token -> slot maps of the ragged streams (SegDev::pad_off)
    const CombDev* combs;
    const int* cta_off;          // [n_cta + 1]: CTA c of the attention kernel owns items [cta_off[c], cta_off[c+1])
    int n_cta;
    int n_items;
    int n_combs;
    int comb_max_rows;           // most rows (tokens x G) any combine entry has
    int comb_max_parts;          // most partials any combine entry merges
    int* counter;                // dynamic scheduler cursor (zeroed before launch)
    const uint8_t* k_pool;
    const uint8_t* v_pool;
    const uint16_t* q;
    uint16_t* out;
    float* lse;                  // may be null
    float* ws_o;                 // split-KV partial O  [slot][rows_per_item][D]  (unnormalised)
    float* ws_ml;                // split-KV partial (m, l) [slot][rows_per_item][2], m in log2 units
    long long q_row_stride;      // elements
    long long out_row_stride;
    long long lse_stride;
    float scale;
    int Hq, Hkv, G, D, P;
    int tile_tokens;             // floor(128 / G)
    int tiles_per_item;
    int page_bytes;
    int num_sms;
    int narrow;                  // every tile of the plan holds <= 16 rows (decode-shaped plan): the instantiation whose softmax
                                 // spreads a row over four threads
    int has_ragged;              // some segment's stream is ragged (SegDev::n_pads > 0): the kernel instantiation with that code
#ifdef SEGPA_TRACE
    unsigned long long* trace;   // [16 warps][kTraceCap] (tag << 56 | arg << 40 | clock) of CTA 0; debug builds only
#endif
};
#ifdef SEGPA_TRACE
constexpr int kTraceCap = 8192;
#endif

// one COPY-mode append of a batch (a1): rows [n_tokens][D] -> the page images listed at page_off
struct ScatterJob {
    const uint16_t* k_src;
    const uint16_t* v_src;
    long long src_stride;        // elements
    long long n_tokens;
    long long chunk_begin;       // first 16-byte chunk of this job in the batch-wide chunk index
    long long page_off;          // index of this job's first touched page id in the batch's id array
    int first_slot;              // slot of the first new token inside the first touched page
    int n_pages;                 // touched pages (the partial last page of the stream + new pages)
    long long n_write;           // slots written from first_slot on: n_tokens rows, then zeros; = n_tokens when a later
                                 // job of the same batch continues the stream inside this job's last page
};

// One job = a run of tokens contiguous in slot space, moved by one delta.  The rotation kernel runs one CTA per
// unit of kRopeUnitChunks 16-byte half-row chunks of one job.
constexpr int kRopeUnitChunks = 1024;   // (2048 in two rounds per CTA measured 10 % slower)
struct RopeJob {
    long long page_off;          // index of its first page id in the batch's id array
    long long n_tokens;
    long long delta_pos;         // p_on - p_off of the chunk
    int first_slot;              // slot of its first token inside its first page
    int unit_begin;              // first CTA (unit) of this job in the grid
};
cudaError_t launch_rope_align(uint8_t* k_pool, const RopeJob* jobs_dev, int n_jobs, const int* page_ids_dev, int total_units,
                              double rope_base, int D, int P, cudaStream_t st);
cudaError_t launch_gather_rows(const uint8_t* k_pool, const uint8_t* v_pool, const int* page_ids_dev, int first_slot,
                               long long n_tokens, uint16_t* k_dst, uint16_t* v_dst, long long dst_stride, int D, int P,
                               cudaStream_t st);

// segpa_gather_rows_noalloc (segpa_misc_kernels.cu): page ids in a fixed device array of kNoAllocMaxPages entries
constexpr int kNoAllocMaxPages = 16384;   // 64 KB per GPU; = SEGPA_NOALLOC_MAX_PAGES of include/segpa.h
cudaError_t noalloc_stage_page_ids(const int* ids_host, int n_ids, cudaStream_t st, const int** ids_dev);

cudaError_t launch_merge(const uint16_t* out_a, const float* lse_a, const uint16_t* out_b, const float* lse_b, uint16_t* out,
                         float* lse, long long row_stride, long long lse_stride, long long T, int Hq, int D, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Attention mass (SelectImportantTokens by-product): one work item = one 128-key block of a
// segment and the range of query tiles that can see it.
// ---------------------------------------------------------------------------------------------
struct MassItem {
    int seg;
    int kb;                 // 128-key block of the segment's stream
    int t_lo, t_hi;         // query tiles [t_lo, t_hi) (tile = tile_tokens tokens x G heads) with a row that sees a key of the block
};

struct MassParams {
    TensorMap q_map;             // same map as FwdParams::q_map
    const SegDev* segs;
    const MassItem* items;
    const int* cta_off;          // [n_cta + 1]
    const int* pages;
    const long long* mass_off;   // [n_segments]: first entry of each segment in `mass`
    const uint8_t* k_pool;
    const float* lse;            // [Hq][lse_stride] from segpa_attention_fwd
    float* mass;
    long long lse_stride;
    float scale;
    int n_cta;
    int G, D, P, tile_tokens, page_bytes;
    unsigned long long* trace;   // [32 warps][kTraceCap] records of CTA 0, as FwdParams::trace; debug builds only
};
cudaError_t launch_attention_mass(const MassParams& p, cudaStream_t st);
cudaError_t launch_mass_select(const float* mass, const long long* mass_off_dev, const int* kv_len_dev, int n_segments, float tau,
                               unsigned char* selected, int* n_selected, cudaStream_t st);

// Launch with programmatic dependent launch allowed: the kernel may begin (prologue up to its pdl_wait()) while the
// previous kernel of the stream drains, which hides launch latency between the back-to-back kernels of a layer.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

// kernel launchers (each returns the CUDA error of its launch)
cudaError_t launch_scatter_pages(uint8_t* k_pool, uint8_t* v_pool, const ScatterJob* jobs_dev, int n_jobs,
                                 const int* page_ids_dev, long long total_chunks, int D, int P, cudaStream_t st);
#ifdef SEGPA_BRINGUP
cudaError_t launch_attention_simt(const FwdParams& p, cudaStream_t st);   // test build only (libsegpa_bringup.so)
#endif
cudaError_t launch_attention_tc(const FwdParams& p, cudaStream_t st);
cudaError_t launch_attention_tc1(const FwdParams& p, cudaStream_t st);   // tiles_per_item == 1, not decode-shaped (segpa_attn_tc1.cu)
cudaError_t launch_combine(const FwdParams& p, cudaStream_t st);

}  // namespace segpa
