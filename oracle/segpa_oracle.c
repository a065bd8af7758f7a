/*
 * segpa_oracle.c -- plain, slow, fp64 CPU oracle for SegPagedAttention.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or helper with the CUDA
 * path under paper_2606_06256_b200/csrc and does not include include/segpa.h.
 *
 * What it computes (the definition, not an algorithm): the method reaches EXACT masked softmax
 * attention ("all paths are numerically equivalent", Sec. 5.3), so the oracle is
 * that definition written out, gathering K/V through the page tables literally
 * (Alg. 2 line 12 "Translate(T_page, U_h)").
 *
 * For every execution segment (request, KV head h) with stream length kv_len, every group head
 * g in [0,G) and every query t in [0,q_len):
 *   1. i = kv_len - q_len + t                      query position, bottom-right aligned
 *                                                  (reading A4; the paper's kernel is
 *                                                  flash_attn_varlen_func)
 *      q = Q[q_row_start + t][h*G + g][:]          contiguous GQA groups (reading A8)
 *   2. visible set V(i) = { j : 0 <= j <= i and (class == GLOBAL or j > i - W or j < n_sink) }
 *        GLOBAL: "full visible range"              PAPER.md:265 (Alg. 2 line 7)
 *        LOCAL : W(i) = S_sink U [max(0,i-w), i]   PAPER.md:219 (Sec. 4.2), with w = W - 1
 *                (W counts the keys INCLUDING the query's own position: reading A1; the paper's
 *                 example i=1000, w=256 -> 744..1000 is W = 257)
 *   3. for j in V(i), ascending: k_j = Kpool[pt[page(j)]][slot(j)][:], v_j likewise;
 *      s_j = scale * sum_d q_d k_{j,d}
 *      A head's stream is the concatenation of its head segments, each mapped to its OWN consecutive virtual
 *      pages ("T_seg maps each head segment (l, h, s) to the virtual pages"): with segment lengths
 *      n_0, n_1, ... token j lies in the segment s with  t_s <= j < t_s + n_s  (t_s = n_0 + ... + n_{s-1}), at offset
 *      o = j - t_s, so  page(j) = (ceil(n_0 / P) + ... + ceil(n_{s-1} / P)) + o / P  and  slot(j) = o % P.  A segment whose
 *      length is not a multiple of P leaves the rest of its last page unused in mid-stream (ragged chunk tails,
 *      SURVEY 8(f) NEXT #1).  Without a segment table the stream is one segment: page(j) = j / P, slot(j) = j % P.
 *   4. m = max_j s_j ; l = sum_j exp(s_j - m) ; p_j = exp(s_j - m) / l     (two passes)
 *   5. O[row][head][:] = sum_j p_j v_j ;  LSE[head][row] = m + ln l         (natural log of the
 *      SCALED scores: reading A6; pinned by the Q=0 closed form LSE = ln #V)
 *
 * bf16 inputs are widened exactly to fp64; scale is the caller's fp32 widened to fp64.  All sums
 * run in ascending index order, so results are bit-reproducible for any thread count (OpenMP
 * parallelism is over independent (segment, head, row) units only).  No tiling, no online
 * softmax, no fusion.
 *
 * Parity pins (tests/test_oracle_pins.py): brute-force dense masked softmax on tiny inputs
 * (oracle/bruteforce.py, independent gather + explicit mask), Q=0 closed forms for the visible-set
 * counts incl. the paper's i=1000 example, W=1 exactness, LOCAL(W>=kv_len) == GLOBAL, page
 * permutation / page size invariance, softmax row sums, constant-V, LSE merge identity
 * (PAPER.md:302), power-of-two scale, GQA == replicated MHA, poison, batch
 * independence / aliasing, torch fp64 causal SDPA at mid size; the row_subset path against the full
 * run (T13); the head-segment table against the brute force's own concatenation of segments, against the
 * dense stream when every segment is a page multiple, and against a dense re-layout of the same tokens (T14).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t num_q_heads;
    int32_t num_kv_heads;
    int32_t head_dim;
    int32_t page_size;
} oracle_shape_t;

typedef struct {
    int32_t stream;      /* index into pt_offsets / kv_lens */
    int32_t kv_head;
    int32_t head_class;  /* 0 GLOBAL, 1 LOCAL */
    int32_t window;      /* W: number of visible keys including self (LOCAL) */
    int32_t n_sink;
    int32_t q_len;
    int64_t q_row_start;
} oracle_segment_t;

static double bf16_to_f64(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* is key j visible to the query at position i?  (step 2 above) */
static int visible(int64_t j, int64_t i, int32_t head_class, int64_t W, int64_t n_sink)
{
    if (j < 0 || j > i) return 0;
    if (head_class == 0) return 1;
    if (j > i - W) return 1;
    if (j < n_sink) return 1;
    return 0;
}

/*
 * Token j of a stream -> index of its (page, slot) in the stream's page table (step 3).
 * seg_lens[0 .. n_seg) are the lengths of the stream's head segments (n_seg == 0: one segment, the whole stream).
 * Returns page_index * P + slot.
 */
static int64_t locate(const int64_t *seg_lens, int64_t n_seg, int64_t P, int64_t j)
{
    if (n_seg == 0) return j;
    int64_t t = 0, page0 = 0;
    for (int64_t s = 0; s < n_seg; ++s) {
        if (j < t + seg_lens[s]) return (page0 + (j - t) / P) * P + (j - t) % P;
        t += seg_lens[s];
        page0 += (seg_lens[s] + P - 1) / P;
    }
    return -1;   /* not reached: the segment lengths sum to kv_len (validated) */
}

/* position of row r inside the sorted subset, or -1 */
static int64_t subset_find(const int64_t *subset, int64_t n, int64_t r)
{
    int64_t lo = 0, hi = n - 1;
    while (lo <= hi) {
        int64_t mid = (lo + hi) / 2;
        if (subset[mid] == r) return mid;
        if (subset[mid] < r) lo = mid + 1; else hi = mid - 1;
    }
    return -1;
}

/*
 * Returns 0 on success, negative on invalid input (q_len < 1, q_len > kv_len, LOCAL with W < 1,
 * page id out of range, bad head index): same rejections as the ABI, so no visible set is empty.
 *
 * row_subset == NULL : out is [T][Hq][D], lse is [Hq][T]; only (row, head) pairs covered by a
 *                      segment are written.
 * row_subset != NULL : ascending global q rows; out is [n_subset][Hq][D], lse is [Hq][n_subset],
 *                      indexed by position in the subset; other rows are skipped.
 * p_out (optional)   : [rows][Hq][p_stride] softmax probabilities p_j at index j (0 elsewhere is
 *                      the caller's job), rows indexed like out.
 * pairs_out (opt.)   : number of (query, key) pairs evaluated, summed over q heads.
 * seg_offsets/seg_lens: head-segment table (optional; NULL = every stream is one segment): the segments of
 *                      stream s are seg_lens[seg_offsets[s] .. seg_offsets[s+1]); they must sum to kv_lens[s] and
 *                      the stream's page table must hold sum ceil(n / P) pages.
 */
int oracle_attention(const oracle_shape_t *shape,
                     const uint16_t *k_pool, const uint16_t *v_pool, int64_t num_pages,
                     const int32_t *page_table, const int64_t *pt_offsets, const int64_t *kv_lens,
                     int32_t n_streams,
                     const oracle_segment_t *segs, int32_t n_segs,
                     const uint16_t *q, int64_t q_row_stride, int64_t T, float scale_f32,
                     const int64_t *row_subset, int64_t n_subset,
                     double *out, double *lse, double *p_out, int64_t p_stride,
                     int64_t *pairs_out,
                     const int64_t *seg_offsets, const int64_t *seg_lens)
{
    const int64_t Hq = shape->num_q_heads, Hkv = shape->num_kv_heads;
    const int64_t D = shape->head_dim, P = shape->page_size;
    if (Hq < 1 || Hkv < 1 || Hq % Hkv != 0 || D < 1 || P < 1) return -1;
    const int64_t G = Hq / Hkv;
    const double scale = (double)scale_f32;
    const int64_t n_rows_out = row_subset ? n_subset : T;

    /* validation pass */
    for (int32_t s = 0; s < n_segs; ++s) {
        const oracle_segment_t *sg = &segs[s];
        if (sg->stream < 0 || sg->stream >= n_streams) return -2;
        if (sg->kv_head < 0 || sg->kv_head >= Hkv) return -3;
        const int64_t kv_len = kv_lens[sg->stream];
        if (sg->q_len < 1 || sg->q_len > kv_len) return -4;
        if (sg->head_class != 0 && sg->head_class != 1) return -5;
        if (sg->head_class == 1 && sg->window < 1) return -6;
        if (sg->n_sink < 0) return -7;
        if (sg->q_row_start < 0 || sg->q_row_start + sg->q_len > T) return -8;
        const int64_t npg = pt_offsets[sg->stream + 1] - pt_offsets[sg->stream];
        int64_t need_pages = (kv_len + P - 1) / P;
        if (seg_offsets && seg_offsets[sg->stream + 1] > seg_offsets[sg->stream]) {
            int64_t tot = 0;
            need_pages = 0;
            for (int64_t k = seg_offsets[sg->stream]; k < seg_offsets[sg->stream + 1]; ++k) {
                if (seg_lens[k] < 1) return -11;
                tot += seg_lens[k];
                need_pages += (seg_lens[k] + P - 1) / P;
            }
            if (tot != kv_len) return -12;
        }
        if (npg < need_pages) return -9;
        for (int64_t pg = 0; pg < need_pages; ++pg) {
            int32_t id = page_table[pt_offsets[sg->stream] + pg];
            if (id < 0 || id >= num_pages) return -10;
        }
    }

    int64_t pairs_total = 0;
    for (int32_t s = 0; s < n_segs; ++s) {
        const oracle_segment_t *sg = &segs[s];
        const int64_t kv_len = kv_lens[sg->stream];
        const int32_t *pt = page_table + pt_offsets[sg->stream];
        const int64_t *sl = seg_offsets ? seg_lens + seg_offsets[sg->stream] : NULL;
        const int64_t n_sl = seg_offsets ? seg_offsets[sg->stream + 1] - seg_offsets[sg->stream] : 0;
        const int64_t units = (int64_t)sg->q_len * G;
        int64_t pairs_seg = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : pairs_seg)
        for (int64_t u = 0; u < units; ++u) {
            const int64_t t = u / G, g = u % G;
            const int64_t row = sg->q_row_start + t;
            int64_t orow = row;
            if (row_subset) {
                orow = subset_find(row_subset, n_subset, row);
                if (orow < 0) continue;
            }
            const int64_t head = (int64_t)sg->kv_head * G + g;
            const int64_t i = kv_len - sg->q_len + t;
            const uint16_t *qp = q + row * q_row_stride + head * D;

            double *sc = (double *)malloc((size_t)(i + 1) * sizeof(double));
            double *qd = (double *)malloc((size_t)D * sizeof(double));
            for (int64_t d = 0; d < D; ++d) qd[d] = bf16_to_f64(qp[d]);

            /* pass 1: scores and max */
            double m = -INFINITY;
            int64_t nvis = 0;
            for (int64_t j = 0; j <= i; ++j) {
                if (!visible(j, i, sg->head_class, sg->window, sg->n_sink)) continue;
                const int64_t u = locate(sl, n_sl, P, j);
                const uint16_t *kp = k_pool + ((int64_t)pt[u / P] * P + (u % P)) * D;
                double acc = 0.0;
                for (int64_t d = 0; d < D; ++d) acc += qd[d] * bf16_to_f64(kp[d]);
                sc[j] = scale * acc;
                if (sc[j] > m) m = sc[j];
                ++nvis;
            }
            /* pass 2: sum of exponentials */
            double l = 0.0;
            for (int64_t j = 0; j <= i; ++j) {
                if (!visible(j, i, sg->head_class, sg->window, sg->n_sink)) continue;
                l += exp(sc[j] - m);
            }
            /* output */
            double *op = out + (orow * Hq + head) * D;
            for (int64_t d = 0; d < D; ++d) op[d] = 0.0;
            for (int64_t j = 0; j <= i; ++j) {
                if (!visible(j, i, sg->head_class, sg->window, sg->n_sink)) continue;
                const double p = exp(sc[j] - m) / l;
                const int64_t u = locate(sl, n_sl, P, j);
                const uint16_t *vp = v_pool + ((int64_t)pt[u / P] * P + (u % P)) * D;
                for (int64_t d = 0; d < D; ++d) op[d] += p * bf16_to_f64(vp[d]);
                if (p_out && j < p_stride) p_out[(orow * Hq + head) * p_stride + j] = p;
            }
            lse[head * n_rows_out + orow] = m + log(l);
            pairs_seg += nvis;
            free(sc);
            free(qd);
        }
        pairs_total += pairs_seg;
    }
    if (pairs_out) *pairs_out = pairs_total;
    return 0;
}
