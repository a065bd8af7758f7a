"""GPU parity of segpa_attention_mass / segpa_mass_select (SelectImportantTokens by-product).

Oracle: the attention oracle's own probabilities p(t, g, j) (want_p), summed over a segment's rows and group heads.
Tolerance: p is recomputed as ex2 of an fp32 score (bf16 products, fp32 accumulate) minus
the fp32 LSE the forward pass wrote (|dLSE| <= 1e-3 by the forward tolerance, measured ~1e-6), so each term is off by
at most ~1e-3 relative: |gpu - oracle| <= 4e-3 * oracle + 1e-3 per key; the total mass equals rows x G within 1e-3."""
import numpy as np
import pytest
import torch

from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
from paper_2606_06256_b200.workloads import GLOBAL, LOCAL
from tests.gpu_helpers import GpuRun
from tests.helpers import run_oracle

pytestmark = pytest.mark.gpu

CASES = [
    (8, 2, 128, 16, [{"kv_len": 700, "heads": {0: (GLOBAL, 0, 0, 300), 1: (LOCAL, 100, 0, 300)}}]),
    (8, 2, 64, 32, [{"kv_len": 515, "heads": {0: (LOCAL, 64, 4, 515), 1: (GLOBAL, 0, 0, 130)}},
                    {"kv_len": 1300, "heads": {0: (GLOBAL, 0, 0, 1), 1: (LOCAL, 300, 130, 3)}}]),
    (28, 4, 128, 32, [{"kv_len": 900, "heads": {0: (GLOBAL, 0, 0, 200), 1: (LOCAL, 257, 0, 200), 2: (LOCAL, 4096, 0, 77), 3: (GLOBAL, 0, 0, 19)}}]),
]


@pytest.mark.parametrize("case", range(len(CASES)))
def test_attention_mass_matches_oracle_column_sums(case):
    Hq, Hkv, D, P, reqs = CASES[case]
    w = wl.make_workload("mass%d" % case, Hq=Hq, Hkv=Hkv, D=D, P=P, requests=reqs, seed=500 + case)
    g = GpuRun(w, "tc", 2)
    try:
        q, out, lse = g.layer(0)
        segs = g.segs[0]
        offs = B.segpa_segments_mass_layout(segs)
        mass = torch.full((int(offs[-1]),), -1.0, dtype=torch.float32, device=g.dev)
        B.segpa_attention_mass(g.cache, segs, q, w.scale, lse, mass)
        m2 = torch.zeros_like(mass)
        B.segpa_attention_mass(g.cache, segs, q, w.scale, lse, m2)          # deterministic
        torch.cuda.synchronize()
        assert torch.equal(mass, m2)
        mass = mass.cpu().numpy().astype(np.float64)
        kv_max = max(s.kv_len for s in w.streams)
        res = run_oracle(w, 0, g.k_pool, g.v_pool, q, want_p=kv_max)
        sm = w.stream_map()
        for si, s in enumerate(w.layer_segments(0)):
            kv = sm[(0, s.kv_head, s.seq_id)].kv_len
            want = res.p[s.q_row_start:s.q_row_start + s.q_len, s.kv_head * w.G:(s.kv_head + 1) * w.G, :kv].sum(axis=(0, 1))
            got = mass[offs[si]:offs[si] + kv]
            assert np.all(np.abs(got - want) <= 4e-3 * want + 1e-3), (si, np.abs(got - want).max())
            assert abs(got.sum() - s.q_len * w.G) <= 1e-3 * s.q_len * w.G          # every row's p sums to 1
            assert np.all(mass[offs[si] + kv:offs[si + 1]] == 0)                   # padding
            assert np.all(got[want == 0] == 0)                                     # keys nobody sees
    finally:
        g.close()


def test_attention_mass_at_cfg2_size():
    """The mass kernel on the whole of cfg2 (32 segments, 16713 rows: the multi-CTA LPT, the Q ring wrapping around
    many times, wholly visible tiles on the fast path), compared with the oracle on the longest request's GLOBAL
    segment and one of its LOCAL segments (every key of both; the oracle's p summed over the segment's rows in
    chunks, on the two KV heads only: the oracle is handed q restricted to their 8 query heads)."""
    import oracle
    w = wl.config2()
    g = GpuRun(w, "tc", 2)
    try:
        q, out, lse = g.layer(0)
        segs = g.segs[0]
        offs = B.segpa_segments_mass_layout(segs)
        mass = torch.full((int(offs[-1]),), -1.0, dtype=torch.float32, device=g.dev)
        B.segpa_attention_mass(g.cache, segs, q, w.scale, lse, mass)
        torch.cuda.synchronize()
        mass = mass.cpu().numpy().astype(np.float64)
        all_segs = w.layer_segments(0)
        sm = w.stream_map()
        # every segment: total mass = rows x G, padding 0
        for si, s in enumerate(all_segs):
            kv = sm[(0, s.kv_head, s.seq_id)].kv_len
            assert abs(mass[offs[si]:offs[si] + kv].sum() - s.q_len * w.G) <= 1e-3 * s.q_len * w.G
            assert np.all(mass[offs[si] + kv:offs[si + 1]] == 0)
        seq = int(np.argmax(w.notes["lengths"]))
        heads = (0, 5)                                         # GLOBAL head 0, LOCAL head 5 (W = 1024)
        pick = [si for si, s in enumerate(all_segs) if s.seq_id == seq and s.kv_head in heads]
        assert [all_segs[si].head_class for si in pick] == [GLOBAL, LOCAL]
        table, pt_off, kv_lens, index = wl.csr_page_tables(w, 0)
        qh = torch.cat([torch.arange(h * w.G, (h + 1) * w.G) for h in heads]).to(q.device)
        q_sub = q[:, qh].contiguous()                          # [T][8][D]: the oracle sees a 2-KV-head problem
        tup = [(index[(all_segs[si].kv_head, seq)], k, all_segs[si].head_class, all_segs[si].window, all_segs[si].n_sink,
                all_segs[si].q_row_start, all_segs[si].q_len) for k, si in enumerate(pick)]
        L = w.notes["lengths"][seq]
        q0 = all_segs[pick[0]].q_row_start
        want = np.zeros((2, L))
        for lo in range(0, L, 512):
            rows = np.arange(q0 + lo, q0 + min(L, lo + 512))
            res = oracle.oracle_attention(Hq=2 * w.G, Hkv=2, D=w.D, P=w.P, k_pool=g.k_pool, v_pool=g.v_pool, page_table=table,
                                          pt_offsets=pt_off, kv_lens=kv_lens, segments=tup, q=q_sub, T=w.T[0], scale=w.scale,
                                          row_subset=rows, want_p=L)
            for k in range(2):
                want[k] += res.p[:, k * w.G:(k + 1) * w.G, :].sum(axis=(0, 1))
        for k, si in enumerate(pick):
            got = mass[offs[si]:offs[si] + L]
            err = np.abs(got - want[k])
            assert np.all(err <= 4e-3 * want[k] + 1e-3), (si, err.max(), int(np.argmax(err)))
            assert np.all(got[want[k] == 0] == 0)
    finally:
        g.close()


@pytest.mark.parametrize("tau", [0.05, 0.5, 0.9, 1.0])
def test_mass_select_is_the_smallest_covering_set(tau):
    Hq, Hkv, D, P, reqs = CASES[0]
    w = wl.make_workload("sel", Hq=Hq, Hkv=Hkv, D=D, P=P, requests=reqs, seed=600)
    g = GpuRun(w, "tc", 2)
    try:
        q, out, lse = g.layer(0)
        segs = g.segs[0]
        offs = B.segpa_segments_mass_layout(segs)
        mass = torch.zeros((int(offs[-1]),), dtype=torch.float32, device=g.dev)
        B.segpa_attention_mass(g.cache, segs, q, w.scale, lse, mass)
        sel = torch.full((int(offs[-1]),), 7, dtype=torch.uint8, device=g.dev)
        cnt = torch.zeros((len(offs) - 1,), dtype=torch.int32, device=g.dev)
        B.segpa_mass_select(g.cache, segs, mass, tau, sel, cnt)
        torch.cuda.synchronize()
        m, sl, cn = mass.cpu().numpy().astype(np.float64), sel.cpu().numpy(), cnt.cpu().numpy()
        sm = w.stream_map()
        for si, s in enumerate(w.layer_segments(0)):
            kv = sm[(0, s.kv_head, s.seq_id)].kv_len
            mm, ss = m[offs[si]:offs[si] + kv], sl[offs[si]:offs[si] + kv].astype(bool)
            tot = mm.sum()
            assert ss.sum() == cn[si] and np.all(sl[offs[si] + kv:offs[si + 1]] == 0)
            # valid: covers tau of the mass; every selected key is at least as heavy as every unselected one
            assert mm[ss].sum() >= tau * tot * (1 - 1e-5)
            if (~ss).any() and ss.any():
                assert mm[ss].min() >= mm[~ss].max()
            # smallest: without its lightest member the set no longer covers tau (up to fp32 summation noise)
            if ss.any():
                assert mm[ss].sum() - mm[ss].min() < tau * tot * (1 + 1e-5)
            # what is unique: the size of the smallest covering set (compare with a sort-based restatement)
            order = np.sort(mm)[::-1]
            k_star = int(np.searchsorted(np.cumsum(order), tau * tot * (1 - 1e-6)) + 1)
            assert abs(int(cn[si]) - min(k_star, kv)) <= 1
    finally:
        g.close()


def test_mass_select_takes_ties_lowest_position_first():
    """Keys of equal mass at the threshold: the lowest positions are taken, exactly as many as are needed (the tie
    rule of segpa.h; the pass that applies it is spread over the block, each thread with a range of positions and the
    number of threshold keys before it).  Synthetic masses on the segments of a real plan."""
    Hq, Hkv, D, P, reqs = CASES[0]
    w = wl.make_workload("selties", Hq=Hq, Hkv=Hkv, D=D, P=P, requests=reqs, seed=601)
    g = GpuRun(w, "tc", 2)
    try:
        g.layer(0)
        segs = g.segs[0]
        offs = B.segpa_segments_mass_layout(segs)
        sm = w.stream_map()
        kvs = [sm[(0, s.kv_head, s.seq_id)].kv_len for s in w.layer_segments(0)]
        rng = np.random.default_rng(11)
        for variant in range(4):
            mass = np.zeros((int(offs[-1]),), dtype=np.float32)
            want = np.zeros_like(mass, dtype=np.uint8)
            tau = [0.5, 0.3, 0.77, 1.0][variant]
            for si, kv in enumerate(kvs):
                if variant == 0:
                    mm = np.ones(kv, dtype=np.float32)                       # all equal
                elif variant == 1:
                    mm = rng.choice(np.array([0.25, 0.5, 1.0, 2.0], dtype=np.float32), size=kv)   # four levels, many ties
                elif variant == 2:
                    mm = np.where(np.arange(kv) % 7 == 3, 4.0, 0.5).astype(np.float32)
                else:
                    mm = rng.choice(np.array([0.0, 1.0], dtype=np.float32), size=kv)              # tau = 1: every key with mass
                mass[offs[si]:offs[si] + kv] = mm
                # reference: heaviest first, ties by position, until tau of the total is covered (exact in fp64 for these values)
                need = np.float32(tau) * np.float32(mm.sum(dtype=np.float64))
                order = np.lexsort((np.arange(kv), -mm))
                csum = np.cumsum(mm[order].astype(np.float64))
                k = int(np.searchsorted(csum, float(need) - 1e-9) + 1)
                k = min(k, kv)
                if variant == 3:
                    k = int((mm > 0).sum())
                want[offs[si] + order[:k]] = 1
            md = torch.from_numpy(mass).to(g.dev)
            sel = torch.full((int(offs[-1]),), 7, dtype=torch.uint8, device=g.dev)
            cnt = torch.zeros((len(offs) - 1,), dtype=torch.int32, device=g.dev)
            B.segpa_mass_select(g.cache, segs, md, tau, sel, cnt)
            torch.cuda.synchronize()
            got = sel.cpu().numpy()
            for si, kv in enumerate(kvs):
                a, b = got[offs[si]:offs[si] + kv], want[offs[si]:offs[si] + kv]
                assert np.array_equal(a, b), (variant, si, int(a.sum()), int(b.sum()), np.flatnonzero(a != b)[:8])
                assert int(cnt[si]) == int(b.sum())
    finally:
        g.close()
