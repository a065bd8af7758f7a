"""segpa_gather_rows_noalloc: the gather entry point that allocates nothing (its scratch, the device copy of the page
ids, is a fixed 64 KB array inside the library) against the existing segpa_gather_rows.

Byte work: the bar is bit-exact.  Two calls in a row on one stream (the second reuses the scratch the first has
filled), a ragged stream (several pieces per call), the size limit, and no change in free device memory across the
calls.  Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
from paper_2606_06256_b200.workloads import GLOBAL, LOCAL

pytestmark = pytest.mark.gpu


def _both(cache, layer, kv_head, seq, t0, n, D, dev, stream=None):
    """(K, V) through the existing path and through the no-alloc entry point."""
    ka, va = torch.full((n, D), 7.0, dtype=torch.bfloat16, device=dev), torch.full((n, D), 7.0, dtype=torch.bfloat16, device=dev)
    kb, vb = torch.full((n, D), 9.0, dtype=torch.bfloat16, device=dev), torch.full((n, D), 9.0, dtype=torch.bfloat16, device=dev)
    B.segpa_gather_rows(cache, layer, kv_head, seq, t0, n, ka, va, stream=stream)
    B.segpa_gather_rows_noalloc(cache, layer, kv_head, seq, t0, n, kb, vb, stream=stream)
    return ka, va, kb, vb


def test_gather_rows_noalloc_matches_gather_rows_on_two_calls_in_a_row():
    dev = torch.device("cuda:0")
    chunks = [100, 37, 260, 50]          # a ragged stream: every chunk on its own pages
    reqs = [{"kv_len": 3000, "heads": {0: (GLOBAL, 0, 0, 8), 1: (LOCAL, 64, 0, 8)}},
            {"kv_len": sum(chunks), "chunks": chunks, "heads": {0: (GLOBAL, 0, 0, 8), 1: (LOCAL, 64, 0, 8)}}]
    w = wl.make_workload("noalloc", Hq=8, Hkv=2, D=128, P=16, requests=reqs, seed=4242)
    k, v = wl.pool_values(w, dev)
    cache = H.create_cache(w, 0)
    try:
        H.append_workload(cache, w, k, v)
        sm = w.stream_map()
        # warm both paths once (the existing one may grow its staging buffer on its first call), then measure
        _both(cache, 0, 0, 0, 0, 3000, w.D, dev)
        torch.cuda.synchronize()
        # two calls in a row on one stream, different streams of the cache and different ranges: the second call
        # overwrites the scratch the first has filled, in stream order
        kb1 = torch.full((2500, w.D), 9.0, dtype=torch.bfloat16, device=dev)
        vb1 = torch.full((2500, w.D), 9.0, dtype=torch.bfloat16, device=dev)
        kb2 = torch.full((401, w.D), 9.0, dtype=torch.bfloat16, device=dev)
        vb2 = torch.full((401, w.D), 9.0, dtype=torch.bfloat16, device=dev)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        B.segpa_gather_rows_noalloc(cache, 0, 1, 0, 333, 2500, kb1, vb1)
        B.segpa_gather_rows_noalloc(cache, 0, 0, 1, 23, 401, kb2, vb2)          # ragged: crosses three chunk tails
        torch.cuda.synchronize()
        free2, _ = torch.cuda.mem_get_info()
        assert free2 == free1, "the no-alloc entry point changed the free device memory"
        ka1, va1 = torch.zeros_like(kb1), torch.zeros_like(vb1)
        ka2, va2 = torch.zeros_like(kb2), torch.zeros_like(vb2)
        B.segpa_gather_rows(cache, 0, 1, 0, 333, 2500, ka1, va1)
        B.segpa_gather_rows(cache, 0, 0, 1, 23, 401, ka2, va2)
        torch.cuda.synchronize()
        assert torch.equal(ka1, kb1) and torch.equal(va1, vb1)
        assert torch.equal(ka2, kb2) and torch.equal(va2, vb2)
        # ... and both equal the rows that were stored
        want_k, want_v = wl.stream_rows(k, sm[(0, 1, 0)], w.P), wl.stream_rows(v, sm[(0, 1, 0)], w.P)
        assert torch.equal(kb1, want_k[333:2833]) and torch.equal(vb1, want_v[333:2833])
        want_k, want_v = wl.stream_rows(k, sm[(0, 0, 1)], w.P), wl.stream_rows(v, sm[(0, 0, 1)], w.P)
        assert torch.equal(kb2, want_k[23:424]) and torch.equal(vb2, want_v[23:424])
        # a third and fourth call, interleaved with the existing path, K only / V only
        for (h, seq, t0, n) in [(0, 0, 0, 3000), (1, 1, 446, 1), (0, 1, 0, sum(chunks)), (1, 0, 2999, 1)]:
            ka, va, kb, vb = _both(cache, 0, h, seq, t0, n, w.D, dev)
            torch.cuda.synchronize()
            assert torch.equal(ka, kb) and torch.equal(va, vb), (h, seq, t0, n)
        only_k = torch.zeros((50, w.D), dtype=torch.bfloat16, device=dev)
        B.segpa_gather_rows_noalloc(cache, 0, 0, 0, 10, 50, only_k, None)
        torch.cuda.synchronize()
        assert torch.equal(only_k, wl.stream_rows(k, sm[(0, 0, 0)], w.P)[10:60])
    finally:
        B.segpa_destroy(cache)


def test_gather_rows_noalloc_rejects_ranges_beyond_its_scratch():
    """More than SEGPA_NOALLOC_MAX_PAGES pages in one call: INVALID with a message that names the limit; nothing is
    written.  The same stream in two calls works."""
    dev = torch.device("cuda:0")
    P, D = 16, 64
    n_tok = (B.NOALLOC_MAX_PAGES + 1) * P
    cache = B.segpa_create_cache(num_layers=1, num_q_heads=2, num_kv_heads=1, head_dim=D, page_size=P,
                                 num_pages=B.NOALLOC_MAX_PAGES + 8, device=0)
    try:
        rows = wl.randn_bf16((n_tok, D), 99, dev)
        B.segpa_append_pages(cache, 0, 0, 5, rows, rows, n_tok)
        out = torch.full((n_tok, D), 3.0, dtype=torch.bfloat16, device=dev)
        with pytest.raises(B.SegpaError, match="fixed scratch of this entry point holds %d" % B.NOALLOC_MAX_PAGES) as e:
            B.segpa_gather_rows_noalloc(cache, 0, 0, 5, 0, n_tok, out, None)
        assert e.value.status == B.ERR_INVALID
        torch.cuda.synchronize()
        assert bool((out == 3.0).all())
        half = B.NOALLOC_MAX_PAGES * P
        B.segpa_gather_rows_noalloc(cache, 0, 0, 5, 0, half, out[:half], None)           # exactly the limit
        B.segpa_gather_rows_noalloc(cache, 0, 0, 5, half, n_tok - half, out[half:], None)
        torch.cuda.synchronize()
        assert torch.equal(out, rows)
        with pytest.raises(B.SegpaError):
            B.segpa_gather_rows_noalloc(cache, 0, 0, 5, n_tok - 3, 4, out[:4], None)      # range outside the stream
        with pytest.raises(B.SegpaError):
            B.segpa_gather_rows_noalloc(cache, 0, 0, 6, 0, 4, out[:4], None)              # no such stream
    finally:
        B.segpa_destroy(cache)
