"""Pins for the fp64 oracle (oracle/segpa_oracle.c) against things other than itself.

T1  brute-force dense masked softmax (independent gather + explicit mask)   BASELINE north_star
T2  Q=0 closed forms for the visible-set counts, incl. the paper's i=1000 example
T3  W=1 returns V at the query's own position, LSE = scale*q.k_i            BASELINE north_star
T4  LOCAL with W >= kv_len is bit-identical to GLOBAL                       BASELINE north_star
T5  page-permutation and page-size invariance                              BASELINE north_star
T6  softmax rows sum to 1; constant V => O = c                              BASELINE north_star
T7  LSE merge identity
T8  power-of-two rescaling of (Q, scale) is bit-identical
T9  GQA == replicated MHA (contiguous groups)
T10 poison: non-visible K/V never enter the softmax
T11 batch independence and page-table aliasing
T12 library special case: torch fp64 causal SDPA at mid size
T13 the row_subset path equals the full run bit for bit
T14 head-segment table (ragged chunk tails): brute force, page-multiple split == dense, dense re-layout
"""
import math
import os

import numpy as np
import pytest
import torch

import oracle
from oracle import bruteforce
from paper_2606_06256_b200 import workloads as wl
from paper_2606_06256_b200.workloads import GLOBAL, LOCAL
from tests.helpers import bits, covered_mask, from_bits, run_oracle, widen

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def tiny(kv_len, heads, *, Hq=4, Hkv=2, D=8, P=4, seed=1, requests=None, scale=None, identity=False):
    reqs = requests if requests is not None else [{"kv_len": kv_len, "heads": heads}]
    return wl.make_workload("tiny", Hq=Hq, Hkv=Hkv, D=D, P=P, requests=reqs, seed=seed, scale=scale,
                            identity_pages=identity)


def values(w, layer=0):
    k, v = wl.pool_values(w)
    return k, v, wl.q_values(w, layer)


# ------------------------------------------------------------------------------------------ T1
GRID = []
for P in (4, 16):
    for kv_len in (1, 5, 16, 33, 67):
        for q_len in sorted({1, max(1, kv_len // 2), kv_len}):
            for W in sorted({1, 2, P - 1, P, P + 1, kv_len, kv_len + 5}):
                for n_sink in (0, 3):
                    GRID.append((P, kv_len, q_len, W, n_sink))


@pytest.mark.parametrize("D", [8, 16])
def test_T1_bruteforce_grid(D):
    worst = 0.0
    for idx, (P, kv_len, q_len, W, n_sink) in enumerate(GRID):
        w = tiny(kv_len, {0: (GLOBAL, 0, 0, q_len), 1: (LOCAL, W, n_sink, q_len)}, D=D, P=P,
                 seed=100 + idx)
        k, v, q = values(w)
        res = run_oracle(w, 0, k, v, q, want_p=kv_len)
        sm = w.stream_map()
        for s in w.segments:
            st = sm[(0, s.kv_head, 0)]
            for g in range(w.G):
                h = s.kv_head * w.G + g
                qb = bits(q)[s.q_row_start:s.q_row_start + s.q_len, h]
                O, L, p = bruteforce.dense_masked_attention(qb, bits(k), bits(v), st.page_ids, kv_len, P,
                                                           s.head_class, s.window, s.n_sink, w.scale)
                rows = slice(s.q_row_start, s.q_row_start + s.q_len)
                worst = max(worst, np.abs(res.out[rows, h] - O).max(), np.abs(res.lse[h, rows] - L).max(),
                            np.abs(res.p[rows, h, :kv_len] - p).max())
    assert worst < 1e-12, worst


# ------------------------------------------------------------------------------------------ T2
def _count(i, cls, W, n_sink):
    """closed form for #V(i): GLOBAL i+1; LOCAL min(i+1, W) plus sinks not already in the window."""
    if cls == GLOBAL:
        return i + 1
    win = min(i + 1, W)
    first = i - win + 1
    return win + max(0, min(n_sink, first))


def test_T2_zero_q_counts():
    for (P, kv_len, q_len, W, n_sink) in GRID:
        w = tiny(kv_len, {0: (GLOBAL, 0, 0, q_len), 1: (LOCAL, W, n_sink, q_len)}, P=P, seed=7)
        k, v, q = values(w)
        q = torch.zeros_like(q)
        res = run_oracle(w, 0, k, v, q, want_p=kv_len)
        for s in w.segments:
            for t in range(s.q_len):
                i = kv_len - s.q_len + t
                n = _count(i, s.head_class, s.window, s.n_sink)
                for g in range(w.G):
                    h = s.kv_head * w.G + g
                    assert abs(res.lse[h, s.q_row_start + t] - math.log(n)) < 1e-13
                    # uniform softmax => O = mean of the visible V rows
                    pv = res.p[s.q_row_start + t, h]
                    assert np.count_nonzero(pv) == n
                    assert np.allclose(pv[pv > 0], 1.0 / n, rtol=0, atol=1e-15)


def test_T2_paper_window_example():
    """i=1000, w=256 -> positions 744..1000 (W = w + 1 = 257 keys)."""
    rows = [ln.split() for ln in open(os.path.join(GOLDEN, "paper_window_example.txt"))
            if ln.strip() and not ln.startswith("#")]
    for i, wpaper, first, last, n in [tuple(map(int, r)) for r in rows]:
        W = wpaper + 1
        kv_len = i + 1
        w = tiny(kv_len, {0: (LOCAL, W, 0, 1), 1: (LOCAL, W, 4, 1)}, P=16, seed=3)
        k, v, q = values(w)
        res = run_oracle(w, 0, k, v, torch.zeros_like(q), want_p=kv_len)
        p0 = res.p[0, 0]
        nz = np.nonzero(p0)[0]
        assert nz[0] == first and nz[-1] == last and len(nz) == n
        assert abs(res.lse[0, 0] - math.log(n)) < 1e-13
        # with 4 sink tokens (the paper's GQA setting): 4 more keys, at 0..3
        p1 = res.p[0, w.G]
        nz1 = np.nonzero(p1)[0]
        assert list(nz1[:4]) == [0, 1, 2, 3] and nz1[4] == first and len(nz1) == n + 4


# ------------------------------------------------------------------------------------------ T3
def test_T3_window_one_returns_own_v():
    w = tiny(37, {0: (LOCAL, 1, 0, 37), 1: (LOCAL, 1, 0, 5)}, P=4, seed=11)
    k, v, q = values(w)
    res = run_oracle(w, 0, k, v, q)
    sm = w.stream_map()
    for s in w.segments:
        st = sm[(0, s.kv_head, 0)]
        for t in range(s.q_len):
            i = st.kv_len - s.q_len + t
            vi = widen(v[int(st.page_ids[i // w.P]), i % w.P])
            ki = widen(k[int(st.page_ids[i // w.P]), i % w.P])
            for g in range(w.G):
                h = s.kv_head * w.G + g
                row = s.q_row_start + t
                assert np.array_equal(res.out[row, h], vi)          # exact
                sc = np.float64(np.float32(w.scale)) * float(np.dot(widen(q[row, h]), ki))
                assert abs(res.lse[h, row] - sc) < 1e-12


# ------------------------------------------------------------------------------------------ T4
@pytest.mark.parametrize("extra", [0, 1, 100])
def test_T4_local_full_window_equals_global(extra):
    kv_len = 50
    wg = tiny(kv_len, {0: (GLOBAL, 0, 0, 20), 1: (GLOBAL, 0, 0, 50)}, seed=5)
    wloc = tiny(kv_len, {0: (LOCAL, kv_len + extra, 0, 20), 1: (LOCAL, kv_len + extra, 2, 50)}, seed=5)
    k, v, q = values(wg)
    a = run_oracle(wg, 0, k, v, q)
    b = run_oracle(wloc, 0, k, v, q)
    assert np.array_equal(a.out, b.out, equal_nan=True) and np.array_equal(a.lse, b.lse, equal_nan=True)


# ------------------------------------------------------------------------------------------ T5
def test_T5_page_permutation_and_page_size_invariance():
    heads = {0: (GLOBAL, 0, 0, 30), 1: (LOCAL, 9, 2, 61)}
    ref = None
    for P, seed in ((4, 1), (4, 2), (16, 3), (1, 4), (64, 5)):
        w = tiny(61, heads, P=P, seed=seed)
        # same LOGICAL streams: draw logical rows once, then scatter into this placement
        rng = torch.Generator().manual_seed(99)
        Kl = torch.randn(2, 61, w.D, generator=rng).to(torch.bfloat16)
        Vl = torch.randn(2, 61, w.D, generator=rng).to(torch.bfloat16)
        q = wl.randn_bf16((w.T[0], w.Hq, w.D), 1234)
        k = torch.full((w.num_pages, P, w.D), float("nan"), dtype=torch.bfloat16)
        v = torch.full((w.num_pages, P, w.D), float("nan"), dtype=torch.bfloat16)
        for s in w.streams:
            for j in range(s.kv_len):
                k[int(s.page_ids[j // P]), j % P] = Kl[s.kv_head, j]
                v[int(s.page_ids[j // P]), j % P] = Vl[s.kv_head, j]
        res = run_oracle(w, 0, k, v, q)
        assert not np.isnan(res.out[covered_mask(w, 0)]).any()
        if ref is None:
            ref = res
        else:
            assert np.array_equal(ref.out, res.out, equal_nan=True)
            assert np.array_equal(ref.lse, res.lse, equal_nan=True)


# ------------------------------------------------------------------------------------------ T6
def test_T6_rows_sum_to_one_and_constant_v():
    w = tiny(45, {0: (GLOBAL, 0, 0, 45), 1: (LOCAL, 7, 3, 45)}, P=16, seed=21)
    k, v, q = values(w)
    res = run_oracle(w, 0, k, v, q, want_p=45)
    assert np.abs(res.p.sum(axis=2) - 1.0).max() < 1e-14
    c = 0.71875  # exactly representable in bf16
    vc = torch.full_like(v, c)
    res2 = run_oracle(w, 0, k, vc, q)
    assert np.abs(res2.out - c).max() < 1e-14


# ------------------------------------------------------------------------------------------ T7
@pytest.mark.parametrize("j0", [1, 13, 16, 40])
def test_T7_lse_merge_identity(j0):
    """partial results over a split key set, merged with LSE, equal the softmax over
    the union.  Part a = GLOBAL over the first j0 keys; part b = the remaining keys as their own
    stream, with a window wide enough that the causal bound alone applies."""
    kv_len, D, P = 41, 8, 4
    rng = torch.Generator().manual_seed(5)
    Kl = torch.randn(kv_len, D, generator=rng).to(torch.bfloat16)
    Vl = torch.randn(kv_len, D, generator=rng).to(torch.bfloat16)
    qrow = torch.randn(1, 1, D, generator=rng).to(torch.bfloat16)

    def run(K, V):
        n = K.shape[0]
        w = tiny(n, {0: (GLOBAL, 0, 0, 1)}, Hq=1, Hkv=1, D=D, P=P, seed=n)
        k = torch.zeros(w.num_pages, P, D, dtype=torch.bfloat16)
        v = torch.zeros(w.num_pages, P, D, dtype=torch.bfloat16)
        st = w.streams[0]
        for j in range(n):
            k[int(st.page_ids[j // P]), j % P] = K[j]
            v[int(st.page_ids[j // P]), j % P] = V[j]
        r = run_oracle(w, 0, k, v, qrow)
        return r.out[0, 0], r.lse[0, 0]

    O, L = run(Kl, Vl)
    Oa, La = run(Kl[:j0], Vl[:j0])
    Ob, Lb = run(Kl[j0:], Vl[j0:])
    Lm = np.logaddexp(La, Lb)
    Om = (np.exp(La - Lm) * Oa + np.exp(Lb - Lm) * Ob)
    assert abs(L - Lm) < 1e-13 and np.abs(O - Om).max() < 1e-13


# ------------------------------------------------------------------------------------------ T8
def test_T8_power_of_two_scale():
    w = tiny(33, {0: (GLOBAL, 0, 0, 33), 1: (LOCAL, 5, 0, 33)}, scale=0.25, seed=8)
    k, v, q = values(w)
    a = run_oracle(w, 0, k, v, q)
    w2 = tiny(33, {0: (GLOBAL, 0, 0, 33), 1: (LOCAL, 5, 0, 33)}, scale=0.125, seed=8)
    q2 = (q.float() * 2).to(torch.bfloat16)
    b = run_oracle(w2, 0, k, v, q2)
    assert np.array_equal(a.out, b.out) and np.array_equal(a.lse, b.lse)


# ------------------------------------------------------------------------------------------ T9
def test_T9_gqa_equals_replicated_mha():
    heads = {0: (GLOBAL, 0, 0, 19), 1: (LOCAL, 6, 1, 19)}
    w = tiny(19, heads, Hq=6, Hkv=2, P=4, seed=31)       # G = 3
    k, v, q = values(w)
    a = run_oracle(w, 0, k, v, q)
    # MHA: 6 kv heads; kv head hq uses the pages of GQA head hq // 3
    heads6 = {h: heads[h // 3] for h in range(6)}
    w6 = tiny(19, heads6, Hq=6, Hkv=6, P=4, seed=31)
    for s in w6.streams:
        s.page_ids = w.stream_map()[(0, s.kv_head // 3, 0)].page_ids.copy()
    w6.num_pages = w.num_pages
    b = run_oracle(w6, 0, k, v, q)
    assert np.array_equal(a.out, b.out) and np.array_equal(a.lse, b.lse)


# ------------------------------------------------------------------------------------------ T10
def test_T10_poison_invisible_tokens():
    """Evicted / non-visible tokens 'never enter the softmax'."""
    kv_len, P, W, n_sink, q_len = 70, 4, 9, 2, 3
    w = tiny(kv_len, {0: (LOCAL, W, n_sink, q_len), 1: (GLOBAL, 0, 0, q_len)}, P=P, seed=41)
    k, v, q = values(w)
    a = run_oracle(w, 0, k, v, q)
    k2, v2 = k.clone(), v.clone()
    used = set()
    for s in w.streams:
        used.update(int(x) for x in s.page_ids)
    for pg in range(w.num_pages):
        if pg not in used:
            k2[pg] = float("nan")
            v2[pg] = float("inf")
    st = w.stream_map()[(0, 0, 0)]
    lo_vis = kv_len - q_len - W + 1          # first key visible to the first query of the LOCAL head
    for j in range(n_sink, lo_vis):
        k2[int(st.page_ids[j // P]), j % P] = float("nan")
        v2[int(st.page_ids[j // P]), j % P] = 1e30
    for s in w.streams:                       # page tails beyond kv_len
        for j in range(s.kv_len, len(s.page_ids) * P):
            k2[int(s.page_ids[j // P]), j % P] = float("nan")
            v2[int(s.page_ids[j // P]), j % P] = float("nan")
    b = run_oracle(w, 0, k2, v2, q)
    assert np.array_equal(a.out, b.out) and np.array_equal(a.lse, b.lse)
    # zero-filling instead of evicting is NOT the same thing: it adds exp(0) mass
    k3, v3 = k.clone(), v.clone()
    wg = tiny(kv_len, {0: (GLOBAL, 0, 0, q_len), 1: (GLOBAL, 0, 0, q_len)}, P=P, seed=41)
    for j in range(n_sink, lo_vis):
        k3[int(st.page_ids[j // P]), j % P] = 0
        v3[int(st.page_ids[j // P]), j % P] = 0
    c = run_oracle(wg, 0, k3, v3, q)
    assert np.abs(c.out[:, :w.G] - a.out[:, :w.G]).max() > 1e-3


# ------------------------------------------------------------------------------------------ T11
def test_T11_batch_independence_and_aliasing():
    r0 = {"kv_len": 23, "heads": {0: (GLOBAL, 0, 0, 7), 1: (LOCAL, 5, 0, 23)}}
    r1 = {"kv_len": 40, "heads": {0: (LOCAL, 11, 2, 1), 1: (GLOBAL, 0, 0, 40)}}
    w = tiny(0, None, requests=[r0, r1], seed=51)
    k, v, q = values(w)
    both = run_oracle(w, 0, k, v, q)
    only0 = run_oracle(w, 0, k, v, q, segments=[s for s in w.segments if s.seq_id == 0])
    rows0 = slice(0, 23)
    assert np.array_equal(both.out[rows0], only0.out[rows0], equal_nan=True)
    # aliasing: request 2 = same page tables and same Q rows as request 0 => identical rows
    w2 = tiny(0, None, requests=[r0, r1, r0], seed=51)
    sm = w2.stream_map()
    for h in (0, 1):
        sm[(0, h, 2)].page_ids = sm[(0, h, 0)].page_ids.copy()
    q2 = wl.q_values(w2, 0)
    q2[63:86] = q2[0:23]
    k2, v2 = wl.pool_values(w2)
    r = run_oracle(w2, 0, k2, v2, q2)
    assert np.array_equal(r.out[0:23], r.out[63:86], equal_nan=True)
    assert np.array_equal(r.lse[:, 0:23], r.lse[:, 63:86], equal_nan=True)


# ------------------------------------------------------------------------------------------ T12
def test_T12_torch_sdpa_causal_midsize():
    """GLOBAL, q_len = kv_len, identity page table == textbook causal attention."""
    L, D, Hq, Hkv, P = 300, 64, 4, 2, 16
    w = wl.make_workload("mid", Hq=Hq, Hkv=Hkv, D=D, P=P, seed=61, identity_pages=True,
                         requests=[{"kv_len": L, "heads": {0: (GLOBAL, 0, 0, L), 1: (GLOBAL, 0, 0, L)}}])
    k, v, q = values(w)
    res = run_oracle(w, 0, k, v, q)
    Q = q.to(torch.float64).permute(1, 0, 2)[None]                       # [1][Hq][L][D]
    K = torch.stack([wl.stream_rows(k, s, P) for s in w.streams]).to(torch.float64)   # [Hkv][L][D]
    V = torch.stack([wl.stream_rows(v, s, P) for s in w.streams]).to(torch.float64)
    K = K.repeat_interleave(w.G, dim=0)[None]
    V = V.repeat_interleave(w.G, dim=0)[None]
    O = torch.nn.functional.scaled_dot_product_attention(Q, K, V, is_causal=True, scale=w.scale)
    O = O[0].permute(1, 0, 2).numpy()
    assert np.abs(res.out - O).max() < 1e-12
    S = (Q[0] @ K[0].transpose(1, 2)) * w.scale
    S = S.masked_fill(~torch.ones(L, L, dtype=torch.bool).tril(), float("-inf"))
    assert np.abs(res.lse - torch.logsumexp(S, dim=-1).numpy()).max() < 1e-12


# ---------------------------------------------------------------------- row_subset path (T13)
@pytest.mark.parametrize("P", [4, 16])
def test_T13_row_subset_equals_full_run_bit_for_bit(P):
    """Every full-size expected value goes through oracle_attention(row_subset=R) (subset_find + the
    subset-indexed outputs): pin it to the full run at rows R, bit for bit, for out, lse, p and pairs.
    R is handed over unsorted with duplicates and holds rows of every kind: covered by all heads, by one
    KV head only (the other head's q range is shorter), the first and the last row of a segment, and -- second
    request -- rows that other requests own.  `pairs` is checked against the T2 closed form, not the full run."""
    reqs = [{"kv_len": 67, "heads": {0: (GLOBAL, 0, 0, 67), 1: (LOCAL, 9, 3, 20)}},
            {"kv_len": 33, "heads": {0: (LOCAL, 5, 0, 33), 1: (GLOBAL, 0, 0, 1)}}]
    w = tiny(0, None, requests=reqs, P=P, seed=77)
    k, v, q = values(w)
    T = w.T[0]
    full = run_oracle(w, 0, k, v, q, want_p=67)
    R = np.array([99, 0, 66, 47, 46, 5, 67, 98, 5, 66, 13, 80], dtype=np.int64)     # unsorted, 5 and 66 twice
    assert R.max() < T
    sub = run_oracle(w, 0, k, v, q, row_subset=R, want_p=67)
    rows = sub.rows
    assert np.array_equal(rows, np.unique(R))
    cov = covered_mask(w, 0, rows)
    assert cov.any() and (~cov).any()                       # rows 0..46 are not covered by kv head 1 (q_len 20)
    # bit for bit (NaN where no segment covers the pair, on both sides)
    assert np.array_equal(sub.out, full.out[rows], equal_nan=True)
    assert np.array_equal(sub.lse, full.lse[:, rows], equal_nan=True)
    assert np.array_equal(sub.p, full.p[rows])
    assert np.isnan(sub.out[~cov]).all() and np.isnan(sub.lse.T[~cov]).all()
    assert not np.isnan(sub.out[cov]).any()
    # pairs of the subset: closed-form counts of exactly these rows
    sm = w.stream_map()
    want = 0
    for s in w.segments:
        kv_len = sm[(0, s.kv_head, s.seq_id)].kv_len
        for r in rows:
            t = int(r) - s.q_row_start
            if 0 <= t < s.q_len:
                want += w.G * _count(kv_len - s.q_len + t, s.head_class, s.window, s.n_sink)
    assert sub.pairs == want
    # a subset that no segment covers at all is legal and evaluates nothing
    w2 = tiny(20, {0: (GLOBAL, 0, 0, 4), 1: (LOCAL, 3, 0, 2)}, P=P, seed=5)
    k2, v2, q2 = values(w2)
    w2.T = [9]                                              # rows 4..8 exist in q / out but belong to nobody
    q2 = wl.randn_bf16((9, w2.Hq, w2.D), 11)
    none = run_oracle(w2, 0, k2, v2, q2, row_subset=np.array([8, 5]))
    assert none.pairs == 0 and np.isnan(none.out).all() and np.isnan(none.lse).all()
    # the whole row range as a subset is the full run
    allr = run_oracle(w, 0, k, v, q, row_subset=np.arange(T)[::-1].copy(), want_p=67)
    assert np.array_equal(allr.out, full.out, equal_nan=True) and np.array_equal(allr.lse, full.lse, equal_nan=True)
    assert allr.pairs == full.pairs


# ------------------------------------------------------------------- head-segment table (T14)
RAGGED_CHUNKS = [
    # (P, chunk lengths): tails of every size, single-token segments, a segment of exactly one page, many segments per block
    (4, [5, 3, 1, 8, 2, 7, 6]),
    (4, [4, 4, 9, 1, 1, 1]),
    (16, [17, 1, 30, 16, 3]),
    (16, [1, 66]),
]


@pytest.mark.parametrize("case", range(len(RAGGED_CHUNKS)))
def test_T14_segment_table_against_bruteforce_concatenation(case):
    """A stream made of head segments, each on its own consecutive pages: the oracle locates token j
    through the segment table; the brute force concatenates the segments' rows into a dense stream first.  All
    classes / windows / sinks of the T1 grid that matter at a tail: windows that end, start and straddle a ragged tail."""
    P, chunks = RAGGED_CHUNKS[case]
    kv_len = sum(chunks)
    worst = 0.0
    for q_len in sorted({1, kv_len // 2, kv_len}):
        for W in sorted({1, 2, P, P + 1, chunks[-1], chunks[-1] + 1, kv_len}):
            for n_sink in (0, 3, chunks[0] + 1):
                w = tiny(0, None, P=P, seed=300 + case, requests=[
                    {"kv_len": kv_len, "chunks": chunks, "heads": {0: (GLOBAL, 0, 0, q_len), 1: (LOCAL, W, n_sink, q_len)}}])
                k, v, q = values(w)
                res = run_oracle(w, 0, k, v, q, want_p=kv_len)
                sm = w.stream_map()
                for s in w.segments:
                    st = sm[(0, s.kv_head, 0)]
                    assert len(st.page_ids) == sum((n + P - 1) // P for n in chunks) > (kv_len + P - 1) // P - 1
                    for g in range(w.G):
                        h = s.kv_head * w.G + g
                        qb = bits(q)[s.q_row_start:s.q_row_start + s.q_len, h]
                        O, L, p = bruteforce.dense_masked_attention(qb, bits(k), bits(v), st.page_ids, kv_len, P, s.head_class,
                                                                   s.window, s.n_sink, w.scale, chunk_lens=chunks)
                        rows = slice(s.q_row_start, s.q_row_start + s.q_len)
                        worst = max(worst, np.abs(res.out[rows, h] - O).max(), np.abs(res.lse[h, rows] - L).max(),
                                    np.abs(res.p[rows, h, :kv_len] - p).max())
    assert worst < 1e-12, worst


def test_T14_page_multiple_segments_equal_the_dense_stream():
    """Splitting a stream into segments at page multiples changes nothing: same page table, same tokens -> the oracle
    must return the dense stream's result bit for bit (the segment table then only restates j -> page j / P)."""
    P = 4
    heads = {0: (GLOBAL, 0, 0, 40), 1: (LOCAL, 7, 2, 25)}
    wd = tiny(40, heads, P=P, seed=9)
    ws = tiny(0, None, P=P, seed=9, requests=[{"kv_len": 40, "chunks": [8, 4, 16, 12], "heads": heads}])
    assert all(np.array_equal(a.page_ids, b.page_ids) for a, b in zip(wd.streams, ws.streams))
    k, v, q = values(wd)
    a = run_oracle(wd, 0, k, v, q, want_p=40)
    b = run_oracle(ws, 0, k, v, q, want_p=40)
    assert np.array_equal(a.out, b.out, equal_nan=True) and np.array_equal(a.lse, b.lse, equal_nan=True) and np.array_equal(a.p, b.p)
    assert a.pairs == b.pairs


def test_T14_ragged_layout_equals_dense_relayout_and_ignores_the_tails():
    """The same tokens stored (a) as ragged segments and (b) densely in another pool give bit-identical results, and
    the unused slots after a segment's tail never enter the softmax (poisoned with NaN / 1e30)."""
    P, chunks = 16, [17, 1, 30, 16, 3]
    kv_len = sum(chunks)
    heads = {0: (GLOBAL, 0, 0, kv_len), 1: (LOCAL, 20, 2, 40)}
    wr = tiny(0, None, P=P, seed=21, requests=[{"kv_len": kv_len, "chunks": chunks, "heads": heads}])
    wdn = tiny(kv_len, heads, P=P, seed=22)
    kr, vr, q = values(wr)
    kd, vd = torch.zeros((wdn.num_pages, P, wr.D), dtype=torch.bfloat16), torch.zeros((wdn.num_pages, P, wr.D), dtype=torch.bfloat16)
    for sr, sd in zip(wr.streams, wdn.streams):
        rows_k, rows_v = wl.stream_rows(kr, sr, P), wl.stream_rows(vr, sr, P)
        assert rows_k.shape[0] == kv_len
        for j in range(kv_len):
            kd[int(sd.page_ids[j // P]), j % P] = rows_k[j]
            vd[int(sd.page_ids[j // P]), j % P] = rows_v[j]
    a = run_oracle(wr, 0, kr, vr, q, want_p=kv_len)
    b = run_oracle(wdn, 0, kd, vd, q, want_p=kv_len)
    assert np.array_equal(a.out, b.out, equal_nan=True) and np.array_equal(a.lse, b.lse, equal_nan=True) and np.array_equal(a.p, b.p)
    # poison the dead slots behind every segment's tail
    kp, vp = kr.clone(), vr.clone()
    for s in wr.streams:
        for c, n in enumerate(chunks):
            if n % P:
                last = int(wl.chunk_pages(s, P, c)[-1])
                kp[last, n % P:] = float("nan")
                vp[last, n % P:] = 1e30
    c2 = run_oracle(wr, 0, kp, vp, q, want_p=kv_len)
    assert np.array_equal(a.out, c2.out, equal_nan=True) and np.array_equal(a.lse, c2.lse, equal_nan=True)
    # a segment table that does not add up is rejected
    wr.streams[0].chunk_lens = [17, 1, 30, 16, 4]
    with pytest.raises(ValueError):
        run_oracle(wr, 0, kr, vr, q)


# ------------------------------------------------------------------------------------ rejections
def test_oracle_rejects_invalid():
    w = tiny(10, {0: (GLOBAL, 0, 0, 11), 1: (LOCAL, 3, 0, 5)})
    k, v, _ = values(w)
    q = wl.randn_bf16((11, w.Hq, w.D), 1)
    w.T = [11]
    with pytest.raises(ValueError):
        run_oracle(w, 0, k, v, q)                       # q_len > kv_len
    w = tiny(10, {0: (GLOBAL, 0, 0, 5), 1: (LOCAL, 0, 0, 5)})
    k, v, q = values(w)
    with pytest.raises(ValueError):
        run_oracle(w, 0, k, v, q)                       # LOCAL with W < 1


# -------------------------------------------------------------------- generators / config sanity
def test_visible_pairs_matches_oracle_count():
    w = tiny(67, {0: (GLOBAL, 0, 0, 30), 1: (LOCAL, 9, 3, 67)}, P=16, seed=2)
    k, v, q = values(w)
    res = run_oracle(w, 0, k, v, q)
    assert res.pairs * 4 * w.D == wl.useful_flops(w)


def test_config_shapes():
    c1 = wl.config1()
    assert (c1.Hq, c1.Hkv, c1.D, c1.P, c1.num_pages, c1.T[0]) == (8, 2, 64, 16, 192, 512)
    assert wl.useful_flops(c1) == (1573888 + 262144) * 4 * 64
    c2 = wl.config2()
    assert len(c2.segments) == 32 and all(2048 <= L <= 8192 for L in c2.notes["lengths"])
    c3 = wl.config3()
    assert sum(c3.notes["chunks"]) == 64512 and all(2048 <= x <= 8192 and x % 16 == 0 for x in c3.notes["chunks"])
    assert abs(wl.useful_flops(c3) / 1e12 - 8.856) < 0.001
    c4 = wl.config4()
    assert len(c4.segments) == 512 and c4.notes["n_global"] == 67
    assert sorted(set(c4.notes["qlen"]))[0] == 1 and c4.notes["qlen"].count(1) == 32
    c5 = wl.config5()
    assert len(c5.segments) == 112 and sum(s.head_class == GLOBAL for s in c5.segments) == 16
    assert abs(wl.useful_flops(c5) / 1e12 - 74.08) < 0.01


# ---------------------------------------------------------------------------------------------
# RoPEAlign oracle pinned to things other than itself
# ---------------------------------------------------------------------------------------------
def _rope_inputs(n=37, D=16, seed=3):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n, D)), rng.integers(0, 5000, size=n), rng.integers(0, 70000, size=n)


def test_rope_printed_constants_and_identity():
    # D = 2: theta_0 = 1, one pair: (1, 0) at delta 1 -> (cos 1, sin 1); (0, 1) -> (-sin 1, cos 1)
    out = oracle.rope_align(np.array([[1.0, 0.0], [0.0, 1.0]]), np.array([0, 0]), np.array([1, 1]))
    assert np.allclose(out, [[0.5403023058681398, 0.8414709848078965], [-0.8414709848078965, 0.5403023058681398]], atol=1e-15)
    k, p_off, _ = _rope_inputs()
    assert np.allclose(oracle.rope_align(k, p_off, p_off), k, atol=1e-12)            # delta = 0


def test_rope_composition_norm_and_pairing():
    k, p_off, p_on = _rope_inputs()
    D = k.shape[1]
    a = oracle.rope_align(k, p_off, p_on)
    # R(p_on) R(p_off)^-1 = R(p_on - p_off): one rotation by the difference gives the same rows
    assert np.allclose(a, oracle.rope_rotate(k, p_on - p_off), atol=1e-9)
    # each (d, d + D/2) pair keeps its norm; only those two elements mix
    assert np.allclose(a[:, :D // 2] ** 2 + a[:, D // 2:] ** 2, k[:, :D // 2] ** 2 + k[:, D // 2:] ** 2, atol=1e-9)
    k2 = k.copy()
    k2[:, 3] += 1.0
    diff = np.abs(oracle.rope_align(k2, p_off, p_on) - a) > 1e-12
    assert diff[:, [3, 3 + D // 2]].any() and not np.delete(diff, [3, 3 + D // 2], axis=1).any()


def test_rope_relative_position_property_and_complex_form():
    k, p_off, p_on = _rope_inputs()
    n, D = k.shape
    rng = np.random.default_rng(5)
    q = rng.standard_normal((n, D))
    m = rng.integers(0, 70000, size=n)
    # <R(m) q, K(p_on)> = <R(m - p_on + p_off) q, K(p_off)>: scores depend on relative position only
    lhs = np.sum(oracle.rope_rotate(q, m) * oracle.rope_align(k, p_off, p_on), axis=1)
    rhs = np.sum(oracle.rope_rotate(q, m - p_on + p_off) * k, axis=1)
    assert np.allclose(lhs, rhs, atol=1e-8)
    # library special case: the pair (a, b) as the complex number a + ib times e^{i delta theta_d}
    theta = 10000.0 ** (-2.0 * np.arange(D // 2) / D)
    z = (k[:, :D // 2] + 1j * k[:, D // 2:]) * np.exp(1j * np.outer(p_on - p_off, theta))
    assert np.allclose(oracle.rope_align(k, p_off, p_on), np.concatenate([z.real, z.imag], axis=1), atol=1e-9)
