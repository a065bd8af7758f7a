"""CPU tests of libsegpa.so's host logic on a planning-only cache (device = -1): exports, pool
bookkeeping, visible-page selection (Alg. 2 lines 6-12), tile schedule, error behaviour."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
from paper_2606_06256_b200.workloads import GLOBAL, LOCAL

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def plan_cache(Hq=8, Hkv=2, D=128, P=16, num_pages=4096, layers=1, tiles=0):
    return B.segpa_create_cache(num_layers=layers, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P,
                                num_pages=num_pages, device=-1, tiles_per_item=tiles)


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "segpa.h")).read()
    declared = sorted(set(re.findall(r"\b(segpa_[a-z_]+)\s*\(", hdr)))
    assert set(declared) == set(B.EXPORTS), (declared, B.EXPORTS)
    L = ctypes.CDLL(B.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    assert B.segpa_version() == 1


def test_product_library_has_no_second_backend():
    """BASELINE north_star "no multi-backend dispatch": the SIMT cross-check kernel and its switch exist only in
    the test build (libsegpa_bringup.so, -DSEGPA_BRINGUP); the product library holds neither, and reads no
    SEGPA_* environment variable."""
    import subprocess
    L = ctypes.CDLL(B.LIB_PATH)
    assert not hasattr(L, "segpa_bringup_use_simt")
    syms = subprocess.run(["nm", "-C", B.LIB_PATH], capture_output=True, text=True).stdout
    assert "attention_simt" not in syms and "attention_tc_kernel" in syms
    blob = open(B.LIB_PATH, "rb").read()
    assert b"SEGPA_KERNEL" not in blob and b"SEGPA_TC_TILES" not in blob and b"SEGPA_TRACE" not in blob
    T = ctypes.CDLL(B.BRINGUP_LIB_PATH)
    assert hasattr(T, "segpa_bringup_use_simt")
    with pytest.raises(B.SegpaError, match="tiles_per_item"):
        plan_cache(tiles=3)


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(B.SegpaError) as e:
        B.segpa_create_cache(num_layers=1, num_q_heads=8, num_kv_heads=2, head_dim=128, page_size=16, num_pages=8, device=0)
    assert e.value.status == B.ERR_CUDA
    c = plan_cache()
    B.segpa_append_pages(c, 0, 0, 0, None, None, 16, page_ids=[0])
    segs = B.segpa_build_segments(c, 0, [(0, 0, GLOBAL, 0, 0, 0, 1)])
    rc = B.lib().segpa_attention_fwd(c, segs, ctypes.c_void_p(16), 1024, ctypes.c_float(1.0), ctypes.c_void_p(16), 1024,
                                     None, 0, 1, None)
    assert rc == B.ERR_STATE
    # the host-buffer entry points too: no device, no result (and nothing to wait for)
    for fn in (B.lib().segpa_attention_fwd_host, B.lib().segpa_attention_fwd_host_async):
        assert fn(c, segs, ctypes.c_void_p(16), ctypes.c_float(1.0), ctypes.c_void_p(16), None, 1, None) == B.ERR_STATE
    B.segpa_host_wait(c)
    assert B.lib().segpa_host_wait(None) == B.ERR_INVALID
    B.segpa_destroy(c)


def test_create_cache_rejections():
    def mk(**kw):
        d = dict(num_layers=1, num_q_heads=8, num_kv_heads=2, head_dim=128, page_size=16, num_pages=8, device=-1)
        d.update(kw)
        return B.segpa_create_cache(**d)
    for kw, st in [(dict(num_q_heads=7), B.ERR_INVALID), (dict(head_dim=96), B.ERR_UNSUPPORTED),
                   (dict(page_size=8), B.ERR_UNSUPPORTED), (dict(num_pages=0), B.ERR_INVALID),
                   (dict(num_q_heads=34, num_kv_heads=2), B.ERR_UNSUPPORTED), (dict(num_layers=0), B.ERR_INVALID)]:
        with pytest.raises(B.SegpaError) as e:
            mk(**kw)
        assert e.value.status == st, kw


def test_pool_bookkeeping_attach_and_refcounts():
    c = plan_cache(num_pages=64)
    B.segpa_append_pages(c, 0, 0, 1, None, None, 40, page_ids=[5, 9, 2])          # 40 tokens -> 3 pages
    kv, ids = B.segpa_stream_info(c, 0, 0, 1)
    assert kv == 40 and list(ids) == [5, 9, 2]
    assert B.segpa_pool_stats(c) == (3, 61)
    # alias the first two pages from another request, then extend
    B.segpa_append_pages(c, 0, 0, 2, None, None, 32, page_ids=[5, 9])
    B.segpa_append_pages(c, 0, 0, 2, None, None, 16, page_ids=[7])
    assert B.segpa_pool_stats(c) == (4, 60)
    # attach to a stream whose last page is partial (stream 1 has 40 tokens): the attached chunk is a new head segment
    # on its own pages; the 8 unused slots of page 2 stay unused in mid-stream
    B.segpa_append_pages(c, 0, 0, 1, None, None, 16, page_ids=[11])
    kv, ids = B.segpa_stream_info(c, 0, 0, 1)
    assert kv == 56 and list(ids) == [5, 9, 2, 11]
    assert B.segpa_pool_stats(c) == (5, 59)
    with pytest.raises(B.SegpaError):
        B.segpa_append_pages(c, 0, 0, 3, None, None, 16, page_ids=[64])               # out of range
    with pytest.raises(B.SegpaError):
        B.segpa_append_pages(c, 0, 0, 3, None, None, 17, page_ids=[1])                # wrong page count
    with pytest.raises(B.SegpaError):
        B.segpa_append_pages(c, 0, 2, 3, None, None, 16, page_ids=[1])                # kv_head out of range
    with pytest.raises(B.SegpaError):
        B.segpa_append_pages(c, 1, 0, 3, None, None, 16, page_ids=[1])                # layer out of range
    B.segpa_free_stream(c, 0, 0, 1)
    assert B.segpa_pool_stats(c) == (3, 61)          # pages 5, 9 still referenced by stream 2; page 2 freed
    B.segpa_free_stream(c, 0, 0, 2)
    assert B.segpa_pool_stats(c) == (0, 64)
    with pytest.raises(B.SegpaError):
        B.segpa_free_stream(c, 0, 0, 2)
    B.segpa_destroy(c)


def test_batched_append_is_ordered_and_all_or_nothing():
    c = plan_cache(num_pages=64)
    # a later request of the batch aliases pages an earlier one introduces, and a stream is extended twice
    B.segpa_append_pages_batch(c, [(0, 0, 1, None, None, 32, [5, 9]),
                                   (0, 0, 2, None, None, 32, [5, 9]),
                                   (0, 0, 2, None, None, 16, [7]),
                                   (0, 1, 1, None, None, 48, [1, 2, 3])])
    assert B.segpa_stream_info(c, 0, 0, 2)[0] == 48 and list(B.segpa_stream_info(c, 0, 0, 2)[1]) == [5, 9, 7]
    assert B.segpa_pool_stats(c) == (6, 58)
    # the third request is invalid (page id out of range): nothing of the batch may stick
    with pytest.raises(B.SegpaError) as e:
        B.segpa_append_pages_batch(c, [(0, 0, 3, None, None, 16, [20]),
                                       (0, 0, 1, None, None, 16, [21]),
                                       (0, 0, 4, None, None, 16, [64])])
    assert e.value.status == B.ERR_INVALID and "[2]" in str(e.value)
    assert B.segpa_pool_stats(c) == (6, 58)
    assert B.segpa_stream_info(c, 0, 0, 1)[0] == 32
    with pytest.raises(B.SegpaError):
        B.segpa_stream_info(c, 0, 0, 3)
    B.segpa_clear_streams(c)
    assert B.segpa_pool_stats(c) == (0, 64)
    with pytest.raises(B.SegpaError):
        B.segpa_stream_info(c, 0, 0, 1)
    B.segpa_destroy(c)


def _expected_pages(kv_len, q_len, cls, W, P, page_ids, zero):
    """Independent restatement of Alg. 2 lines 6-12 for one segment."""
    vis_lo = 0 if cls == GLOBAL else max(0, kv_len - q_len - W + 1)
    kb_lo, kb_hi = vis_lo // 128, (kv_len - 1) // 128 + 1
    ppb = 128 // P
    out = []
    for pg in range(kb_lo * ppb, kb_hi * ppb):
        visible = any(vis_lo <= j < kv_len for j in range(pg * P, pg * P + P))
        out.append(int(page_ids[pg]) if visible else zero)
    return kb_lo * ppb, out


@pytest.mark.parametrize("P", [16, 32])
def test_visible_page_selection_and_tiles(P):
    rng = np.random.default_rng(P)
    for trial in range(40):
        kv_len = int(rng.integers(1, 3000))
        q_len = int(rng.integers(1, kv_len + 1))
        cls = int(rng.integers(0, 2))
        W = int(rng.choice([1, 2, P - 1, P, P + 1, 127, 128, 129, 700, 5000]))
        G = int(rng.choice([1, 4, 7, 8]))
        npg = (kv_len + P - 1) // P
        ids = rng.permutation(1024)[:npg].astype(np.int32)
        for tiles in (1, 2):
            c = plan_cache(Hq=2 * G, Hkv=2, P=P, num_pages=1024, tiles=tiles)
            B.segpa_append_pages(c, 0, 1, 42, None, None, kv_len, page_ids=ids)
            segs = B.segpa_build_segments(c, 0, [(42, 1, cls, W, 0, 10, q_len)])
            first, got = B.segpa_segments_pages(segs, 0)
            efirst, exp = _expected_pages(kv_len, q_len, cls, W, P, ids, 1024)
            assert first == efirst and list(got) == exp, (kv_len, q_len, cls, W, P)
            st = B.segpa_segments_stats(segs)
            items = B.segpa_segments_items(segs)
            TT = 128 // G
            assert st["tile_tokens"] == TT and st["q_rows"] == 10 + q_len
            # brute force: per item, the blocks holding at least one visible (row, key) pair
            pairs = 0
            seen_tok = np.zeros(q_len, dtype=int)
            by_tile = {}
            for it in items:
                by_tile.setdefault(it["tile"], []).append(it)
            for tile, parts in by_tile.items():
                parts.sort(key=lambda x: x["kb_lo"])
                t0, n_tok = parts[0]["t0"], parts[0]["n_tok"]
                assert n_tok <= TT * tiles
                seen_tok[t0:t0 + n_tok] += 1
                need = set()
                for t in range(t0, t0 + n_tok):
                    i = kv_len - q_len + t
                    lo = 0 if cls == GLOBAL else max(0, i - W + 1)
                    need.update(range(lo // 128, i // 128 + 1))
                    pairs += (i - lo + 1) * G
                got_blocks = []
                for pt in parts:
                    assert pt["kb_hi"] > pt["kb_lo"]                # no empty item
                    got_blocks += list(range(pt["kb_lo"], pt["kb_hi"]))
                assert sorted(need) == got_blocks                    # exactly the attended blocks, once each
                assert all(pt["n_splits"] == len(parts) for pt in parts)
            assert np.all(seen_tok == 1)
            assert st["attended_pairs"] == pairs
            costs = [it["kb_hi"] - it["kb_lo"] for it in items]
            assert st["kv_blocks"] == sum(costs)
            # LPT schedule: items listed CTA by CTA, longest first inside a CTA, loads balanced to within one item
            ctas = [it["cta"] for it in items]
            assert ctas == sorted(ctas) and ctas[0] == 0 and ctas[-1] == min(len(items), 148) - 1
            loads = {}
            for it, cst in zip(items, costs):
                loads.setdefault(it["cta"], []).append(cst)
            for q, cs in loads.items():
                assert cs == sorted(cs, reverse=True)
            tot = [sum(3 * x + 2 for x in cs) for cs in loads.values()]
            assert max(tot) - min(tot) <= 3 * max(costs) + 2
            B.segpa_free_segments(c, segs)
            B.segpa_destroy(c)


@pytest.mark.parametrize("P", [16, 32])
def test_ragged_streams_are_planned_in_slot_space(P):
    """Streams spliced from chunks of arbitrary length (each on its own pages): the page lists and the
    tiles' KV block ranges follow the SLOT of a token (token index + the unused slots behind earlier chunks' tails).
    Checked against a restatement that lays the stream out slot by slot."""
    rng = np.random.default_rng(100 + P)
    for trial in range(30):
        n_chunks = int(rng.integers(2, 9))
        chunks = [int(rng.choice([1, P - 1, P, P + 1, 100, 333, 700])) for _ in range(n_chunks)]
        kv_len = sum(chunks)
        q_len = int(rng.integers(1, kv_len + 1))
        cls = int(rng.integers(0, 2))
        W = int(rng.choice([1, 7, 128, 300, 5000]))
        n_sink = int(rng.choice([0, 0, 4, 50])) if cls == LOCAL else 0
        G = int(rng.choice([1, 4, 8]))
        c = plan_cache(Hq=2 * G, Hkv=2, P=P, num_pages=2048)
        # slot-by-slot layout: tok_of_slot[u] = token or -1
        tok_of_slot, ids_all, next_id = [], [], 0
        for n in chunks:
            npg = (n + P - 1) // P
            ids = list(range(next_id, next_id + npg))
            next_id += npg
            ids_all += ids
            B.segpa_append_pages(c, 0, 1, 42, None, None, n, page_ids=ids)
            base = len([t for t in tok_of_slot if t >= 0])
            tok_of_slot += [base + o if o < n else -1 for o in range(npg * P)]
        kv, got_ids = B.segpa_stream_info(c, 0, 1, 42)
        assert kv == kv_len and list(got_ids) == ids_all
        slot_of = {t: u for u, t in enumerate(tok_of_slot) if t >= 0}
        segs = B.segpa_build_segments(c, 0, [(42, 1, cls, W, n_sink, 3, q_len)])
        st = B.segpa_segments_stats(segs)
        items = B.segpa_segments_items(segs)
        first, pages = B.segpa_segments_pages(segs, 0)
        ppb = 128 // P
        # visible tokens of the whole segment and of each tile
        def visible(i):
            lo = 0 if cls == GLOBAL else max(0, i - W + 1)
            sinks = range(0, min(n_sink, lo)) if (cls == LOCAL and kv_len > W) else range(0)
            return list(sinks) + list(range(lo, i + 1))
        need_pages = set()
        pairs = 0
        by_tile = {}
        for it in items:
            by_tile.setdefault(it["tile"], []).append(it)
        for tile, parts in by_tile.items():
            t0, n_tok = parts[0]["t0"], parts[0]["n_tok"]
            need_blocks = set()
            for t in range(t0, t0 + n_tok):
                vis = visible(kv_len - q_len + t)
                pairs += len(vis) * G
                need_blocks.update(slot_of[j] // 128 for j in vis)
                need_pages.update(slot_of[j] // P for j in vis)
            got_blocks = set()
            for pt in parts:
                got_blocks.update(range(pt["kb_lo"], pt["kb_hi"]))
            assert need_blocks <= got_blocks                      # every attended block is visited ...
            assert got_blocks <= set(range(min(need_blocks), max(need_blocks) + 1))   # ... and nothing outside their hull
        assert st["attended_pairs"] == pairs
        # every page that holds a visible token is listed with its physical id; pages outside the hull are the zero page
        for pg in need_pages:
            assert pages[pg - first] == ids_all[pg], (trial, pg)
        for k, pid in enumerate(pages):
            assert pid == 2048 or pid == ids_all[first + k]
        B.segpa_destroy(c)


def test_split_kv_plan_for_decode():
    c = plan_cache(num_pages=4096, tiles=1)
    B.segpa_append_pages(c, 0, 0, 0, None, None, 30000, page_ids=np.arange(1875))
    segs = B.segpa_build_segments(c, 0, [(0, 0, GLOBAL, 0, 0, 0, 1)])
    st = B.segpa_segments_stats(segs)
    assert st["n_tiles"] == 1 and st["n_split_tiles"] == 1 and st["n_items"] > 8
    assert st["workspace_bytes"] == st["n_items"] * 128 * (128 + 2) * 4
    B.segpa_destroy(c)


def test_build_segments_rejections():
    c = plan_cache(num_pages=256)
    B.segpa_append_pages(c, 0, 0, 0, None, None, 100, page_ids=np.arange(7))
    B.segpa_append_pages(c, 0, 1, 0, None, None, 100, page_ids=np.arange(7, 14))
    bad = [
        ([(0, 0, GLOBAL, 0, 0, 0, 101)], B.ERR_INVALID),                 # q_len > kv_len
        ([(0, 0, GLOBAL, 0, 0, 0, 0)], B.ERR_INVALID),                   # q_len < 1
        ([(0, 0, LOCAL, 0, 0, 0, 5)], B.ERR_INVALID),                    # LOCAL window < 1
        ([(0, 0, 2, 4, 0, 0, 5)], B.ERR_INVALID),                        # bad class
        ([(9, 0, GLOBAL, 0, 0, 0, 5)], B.ERR_INVALID),                   # unknown stream
        ([(0, 2, GLOBAL, 0, 0, 0, 5)], B.ERR_INVALID),                   # kv_head out of range
        ([(0, 0, GLOBAL, 0, 0, -1, 5)], B.ERR_INVALID),                  # negative row
        ([(0, 0, GLOBAL, 0, 0, 0, 50), (0, 0, LOCAL, 8, 0, 49, 10)], B.ERR_INVALID),   # (row, head) overlap
        ([(0, 0, LOCAL, 8, -1, 0, 5)], B.ERR_INVALID),                   # negative n_sink
        ([], B.ERR_INVALID),
    ]
    for reqs, st in bad:
        with pytest.raises(B.SegpaError) as e:
            B.segpa_build_segments(c, 0, reqs)
        assert e.value.status == st, reqs
    # different kv heads may share rows; same head may use disjoint rows
    segs = B.segpa_build_segments(c, 0, [(0, 0, GLOBAL, 0, 0, 0, 50), (0, 1, LOCAL, 8, 0, 0, 50), (0, 0, GLOBAL, 0, 0, 50, 10)])
    assert B.segpa_segments_stats(segs)["n_segments"] == 3
    with pytest.raises(B.SegpaError):
        B.segpa_build_segments(c, 1, [(0, 0, GLOBAL, 0, 0, 0, 5)])       # layer out of range
    B.segpa_destroy(c)


def test_sinks_select_two_page_ranges_and_eviction_is_checked():
    """LOCAL with sinks (Alg. 2 lines 9-10): sink pages + recent-window pages are translated, the
    middle maps to the zero page and may be evicted; an evicted VISIBLE page is an error."""
    P, n_pages_pool = 16, 512
    c = plan_cache(P=P, num_pages=n_pages_pool)
    kv_len, q_len, W, n_sink = 5000, 3, 700, 40
    ids = np.arange(100, 100 + (kv_len + P - 1) // P)
    B.segpa_append_pages(c, 0, 0, 0, None, None, kv_len, page_ids=ids)
    segs = B.segpa_build_segments(c, 0, [(0, 0, LOCAL, W, n_sink, 0, q_len)])
    first, pages = B.segpa_segments_pages(segs, 0)
    assert first == 0
    vis_lo = kv_len - q_len - W + 1
    for pg, got in enumerate(pages):
        in_sink = pg * P < n_sink
        in_win = (pg + 1) * P > vis_lo and pg < len(ids)
        assert got == (ids[pg] if (in_sink or in_win) else n_pages_pool), pg
    st = B.segpa_segments_stats(segs)
    want = sum(min(i + 1, W) + max(0, min(n_sink, i - W + 1)) for i in range(kv_len - q_len, kv_len)) * 4
    assert st["attended_pairs"] == want
    it = B.segpa_segments_items(segs)
    assert len(it) == 1 and it[0]["kb_lo"] == 0 and st["kv_blocks"] == 1 + (kv_len - 1) // 128 + 1 - vis_lo // 128
    # evict the middle: fine; evict into the window or the sinks: build fails
    mid_lo, mid_hi = (n_sink + P - 1) // P, vis_lo // P
    B.segpa_evict_pages(c, 0, 0, 0, mid_lo, mid_hi - mid_lo)
    assert B.segpa_pool_stats(c)[0] == len(ids) - (mid_hi - mid_lo)
    assert list(B.segpa_stream_info(c, 0, 0, 0)[1][mid_lo:mid_lo + 2]) == [-1, -1]
    segs2 = B.segpa_build_segments(c, 0, [(0, 0, LOCAL, W, n_sink, 0, q_len)])
    assert list(B.segpa_segments_pages(segs2, 0)[1]) == list(pages)
    with pytest.raises(B.SegpaError):
        B.segpa_evict_pages(c, 0, 0, 0, mid_lo, 1)                        # already evicted
    with pytest.raises(B.SegpaError):
        B.segpa_evict_pages(c, 0, 0, 0, len(ids) - 1, 1)                  # partial last page
    B.segpa_evict_pages(c, 0, 0, 0, mid_hi, 1)                            # first window page
    with pytest.raises(B.SegpaError) as e:
        B.segpa_build_segments(c, 0, [(0, 0, LOCAL, W, n_sink, 0, q_len)])
    assert e.value.status == B.ERR_INVALID
    with pytest.raises(B.SegpaError):
        B.segpa_build_segments(c, 0, [(0, 0, GLOBAL, 0, 0, 0, q_len)])    # a global head needs every page
    B.segpa_free_stream(c, 0, 0, 0)
    assert B.segpa_pool_stats(c) == (0, n_pages_pool)
    B.segpa_destroy(c)


def test_config_plans_match_closed_forms():
    """Useful work of the five BASELINE configs as planned by the library == generator closed forms."""
    for cfg in (1, 2, 3, 4):
        w = wl.CONFIGS[cfg]()
        c = B.segpa_create_cache(num_layers=1, num_q_heads=w.Hq, num_kv_heads=w.Hkv, head_dim=w.D, page_size=w.P,
                                 num_pages=w.num_pages, device=-1)
        H.append_workload(c, w)
        segs = H.build_layer(c, w, 0)
        st = B.segpa_segments_stats(segs)
        assert st["attended_pairs"] * 4 * w.D == wl.useful_flops(w, 0)
        used, free = B.segpa_pool_stats(c)
        assert used == len({int(p) for s in w.streams for p in s.page_ids})
        B.segpa_destroy(c)


def test_lpt_assignment_matches_plain_heap_restatement():
    """The scheduler's CTA assignment (counting sort + sorted-run insertion in the library) equals the textbook
    statement of LPT written with heapq: items by descending cost (ties: creation order), each to the CTA with
    the smallest (load, cta); load grows by 3 * blocks + 2 thirds of a block-time.
    Workloads without strided or sink items, where the cost is kb_hi - kb_lo."""
    import heapq
    rng = np.random.default_rng(3)
    for trial in range(4):
        n_req = int(rng.integers(2, 7))
        reqs = []
        for r in range(n_req):
            L = int(rng.integers(200, 9000))
            reqs.append({"kv_len": L, "heads": {0: (GLOBAL, 0, 0, L), 1: (LOCAL, int(rng.choice([256, 1024, 3000])), 0, L)}})
        w = wl.make_workload("lpt%d" % trial, Hq=8, Hkv=2, D=128, P=16, requests=reqs, seed=trial)
        c = B.segpa_create_cache(num_layers=1, num_q_heads=w.Hq, num_kv_heads=w.Hkv, head_dim=w.D, page_size=w.P,
                                 num_pages=w.num_pages, device=-1)
        H.append_workload(c, w)
        segs = H.build_layer(c, w, 0)
        items = B.segpa_segments_items(segs)
        n_cta = min(len(items), 148)
        created = sorted(range(len(items)), key=lambda i: (items[i]["tile"], max(items[i]["split"], 0)))
        order = sorted(created, key=lambda i: -(items[i]["kb_hi"] - items[i]["kb_lo"]))   # stable: ties keep creation order
        heap = [(0, q) for q in range(n_cta)]
        heapq.heapify(heap)
        expect = {}
        per_cta = {q: [] for q in range(n_cta)}
        for i in order:
            load, q = heapq.heappop(heap)
            expect[i] = q
            per_cta[q].append(i)
            heapq.heappush(heap, (load + 3 * (items[i]["kb_hi"] - items[i]["kb_lo"]) + 2, q))
        assert [items[i]["cta"] for i in range(len(items))] == [expect[i] for i in range(len(items))]
        # and the list is laid out CTA by CTA in assignment order
        flat = [i for q in range(n_cta) for i in per_cta[q]]
        assert flat == list(range(len(items)))
        B.segpa_free_segments(c, segs)
        B.segpa_destroy(c)
