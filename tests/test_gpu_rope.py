"""GPU parity of segpa_rope_align (RoPEAlign) and segpa_gather_rows against the fp64 oracle.

Tolerance: the device forms a*cos - b*sin in fp32 from fp32 cos / sin (relative error
of a few 2^-24) and rounds once to bf16 (relative 2^-9 of the result, whose magnitude is at most |a| + |b|):
|gpu - oracle| <= 2^-8 * (|a| + |b|) + 1e-6 per element, a and b being the pair's inputs."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
from paper_2606_06256_b200.workloads import GLOBAL, LOCAL
from tests.gpu_helpers import GpuRun, compare

pytestmark = pytest.mark.gpu


def _pair_bound(k):
    half = k.shape[1] // 2
    s = np.abs(k[:, :half]) + np.abs(k[:, half:])
    return 2.0 ** -8 * np.concatenate([s, s], axis=1) + 1e-6


@pytest.mark.parametrize("D,P", [(128, 16), (64, 32), (128, 32)])
def test_gather_rows_roundtrip_and_rope_align(D, P):
    w = wl.make_workload("rope", Hq=8, Hkv=2, D=D, P=P, seed=77,
                         requests=[{"kv_len": 1000, "heads": {0: (GLOBAL, 0, 0, 10), 1: (LOCAL, 64, 0, 10)}}])
    dev = torch.device("cuda:0")
    k, v = wl.pool_values(w, dev)
    g = GpuRun(w, "tc", 2, k, v)
    try:
        st = w.stream_map()[(0, 0, 0)]
        k_rows = wl.stream_rows(k, st, w.P)
        v_rows = wl.stream_rows(v, st, w.P)
        # gather is the exact inverse of the scatter, also from an unaligned token range
        kd = torch.zeros((700, D), dtype=torch.bfloat16, device=dev)
        vd = torch.zeros_like(kd)
        B.segpa_gather_rows(g.cache, 0, 0, 0, 133, 700, kd, vd)
        torch.cuda.synchronize()
        assert torch.equal(kd, k_rows[133:833]) and torch.equal(vd, v_rows[133:833])
        # RoPEAlign a reused chunk: tokens [133, 833) cached at positions 133.. move to 40133..
        delta = 40000
        B.segpa_rope_align(g.cache, 0, 0, 0, 133, 700, delta, 10000.0)
        kall = torch.zeros((1000, D), dtype=torch.bfloat16, device=dev)
        vall = torch.zeros_like(kall)
        B.segpa_gather_rows(g.cache, 0, 0, 0, 0, 1000, kall, vall)
        torch.cuda.synchronize()
        assert torch.equal(vall, v_rows)                                                  # V untouched
        assert torch.equal(kall[:133], k_rows[:133]) and torch.equal(kall[833:], k_rows[833:])   # outside the range
        k64 = k_rows[133:833].to(torch.float64).cpu().numpy()
        p_off = np.arange(133, 833)
        want = oracle.rope_align(k64, p_off, p_off + delta)
        got = kall[133:833].to(torch.float64).cpu().numpy()
        assert np.all(np.abs(got - want) <= _pair_bound(k64)), np.abs(got - want).max()
        # rotating back (delta negative) returns the original rows up to two bf16 roundings
        B.segpa_rope_align(g.cache, 0, 0, 0, 133, 700, -delta, 10000.0)
        B.segpa_gather_rows(g.cache, 0, 0, 0, 133, 700, kd, None)
        torch.cuda.synchronize()
        assert np.all(np.abs(kd.to(torch.float64).cpu().numpy() - k64) <= 2.5 * _pair_bound(k64))
        # error behaviour
        with pytest.raises(B.SegpaError):
            B.segpa_rope_align(g.cache, 0, 0, 0, 900, 200, 5, 10000.0)       # range outside the stream
        with pytest.raises(B.SegpaError):
            B.segpa_rope_align(g.cache, 0, 0, 0, 0, 10, 5, 1.0)             # base must be > 1
    finally:
        g.close()


def test_attention_after_rope_align_matches_oracle_on_rotated_keys():
    """The step before the hot path feeds it: keys rotated in the pool by segpa_rope_align, then attention;
    the oracle side rotates the same keys with the RoPE oracle (rounded to bf16 as the pool holds them)."""
    reqs = [{"kv_len": 2000, "heads": {0: (GLOBAL, 0, 0, 300), 1: (LOCAL, 500, 4, 300)}}]
    w = wl.make_workload("rope_attn", Hq=8, Hkv=2, D=128, P=16, requests=reqs, seed=78)
    dev = torch.device("cuda:0")
    k, v = wl.pool_values(w, dev)
    g = GpuRun(w, "tc", 2, k, v)
    try:
        delta = 12345
        k2 = k.clone()
        for h in (0, 1):
            B.segpa_rope_align(g.cache, 0, h, 0, 256, 1024, delta, 10000.0)
            st = w.stream_map()[(0, h, 0)]
            out_rows = torch.zeros((1024, 128), dtype=torch.bfloat16, device=dev)
            B.segpa_gather_rows(g.cache, 0, h, 0, 256, 1024, out_rows, None)
            # the oracle's pool: what the device now holds (already checked against the RoPE oracle above)
            idx = torch.from_numpy(st.page_ids.astype(np.int64)).to(dev)
            rows = k2[idx].reshape(-1, 128)
            rows[256:1280] = out_rows
            k2[idx] = rows.reshape(-1, 16, 128)
            k64 = wl.stream_rows(k, st, 16)[256:1280].to(torch.float64).cpu().numpy()
            want = oracle.rope_align(k64, np.arange(256, 1280), np.arange(256, 1280) + delta)
            assert np.all(np.abs(out_rows.to(torch.float64).cpu().numpy() - want) <= _pair_bound(k64))
        q, out, lse = g.layer(0)
        print(compare(w, 0, k2, v, q, out, lse, label="attention after rope_align"))
    finally:
        g.close()


def test_rope_align_batch_matches_single_calls():
    reqs_w = [{"kv_len": 900 + 50 * r, "heads": {0: (GLOBAL, 0, 0, 5), 1: (LOCAL, 64, 0, 5)}} for r in range(3)]
    w = wl.make_workload("rope_b", Hq=8, Hkv=2, D=128, P=16, requests=reqs_w, seed=79)
    dev = torch.device("cuda:0")
    k, v = wl.pool_values(w, dev)
    chunks = [(s.layer, s.kv_head, s.seq_id, lo, n, d) for s in w.streams for (lo, n, d) in ((3, 200, 777), (300, 333, -5000), (700, 150, 65000))]
    outs = []
    for mode in ("batch", "single"):
        g = GpuRun(w, "tc", 2, k, v)
        if mode == "batch":
            B.segpa_rope_align_batch(g.cache, chunks, 10000.0)
        else:
            for c in chunks:
                B.segpa_rope_align(g.cache, *c, 10000.0)
        got = []
        for s in w.streams:
            kd = torch.zeros((s.kv_len, 128), dtype=torch.bfloat16, device=dev)
            B.segpa_gather_rows(g.cache, s.layer, s.kv_head, s.seq_id, 0, s.kv_len, kd, None)
            got.append(kd)
        torch.cuda.synchronize()
        outs.append(got)
        if mode == "batch":
            with pytest.raises(B.SegpaError):     # overlapping ranges in one batch
                B.segpa_rope_align_batch(g.cache, [(0, 0, 0, 0, 100, 1), (0, 0, 0, 50, 100, 2)], 10000.0)
        g.close()
    for a, b in zip(*outs):
        assert torch.equal(a, b)
    s0 = w.streams[0]
    k64 = wl.stream_rows(k, s0, 16)[300:633].to(torch.float64).cpu().numpy()
    want = oracle.rope_align(k64, np.arange(300, 633), np.arange(300, 633) - 5000)
    assert np.all(np.abs(outs[0][0][300:633].to(torch.float64).cpu().numpy() - want) <= _pair_bound(k64))


def test_rope_align_refuses_shared_pages():
    c = B.segpa_create_cache(num_layers=1, num_q_heads=8, num_kv_heads=2, head_dim=128, page_size=16, num_pages=64, device=0)
    dev = torch.device("cuda:0")
    rows = torch.randn((64, 128), device=dev).to(torch.bfloat16)
    B.segpa_append_pages(c, 0, 0, 1, rows, rows, 64, page_ids=[3, 4, 5, 6])
    B.segpa_append_pages(c, 0, 0, 2, None, None, 32, page_ids=[3, 4])         # alias the first two pages
    with pytest.raises(B.SegpaError) as e:
        B.segpa_rope_align(c, 0, 0, 1, 0, 64, 7, 10000.0)
    assert e.value.status == B.ERR_INVALID
    B.segpa_rope_align(c, 0, 0, 1, 32, 32, 7, 10000.0)                        # the unshared tail is fine
    B.segpa_destroy(c)
