"""GPU-side test plumbing: run a Workload through libsegpa.so and compare with the oracle."""
from __future__ import annotations

import numpy as np
import torch

from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
from tests.helpers import covered_mask, run_oracle

OUT_SENTINEL = 123.0
LSE_SENTINEL = -777.0
TOL_OUT_MAX, TOL_OUT_MEAN, TOL_LSE = 2e-2, 2e-3, 1e-3     # BASELINE.json:north_star


class GpuRun:
    """kernel "tc": the product library.  kernel "simt": the test build (libsegpa_bringup.so) with its SIMT
    cross-check kernel -- the binding is switched to that library for the lifetime of the run."""

    def __init__(self, w: wl.Workload, kernel: str = "tc", tiles: int = 1, k_pool=None, v_pool=None):
        assert kernel in ("tc", "simt")
        self.w = w
        self.dev = torch.device("cuda:0")
        if k_pool is None:
            k_pool, v_pool = wl.pool_values(w, self.dev)
        self.k_pool, self.v_pool = k_pool, v_pool
        self.bringup = kernel == "simt"
        if self.bringup:
            B.use_library("bringup")
        self.cache = H.create_cache(w, 0, tiles_per_item=tiles)
        if self.bringup:
            B.segpa_bringup_use_simt(self.cache)
        H.append_workload(self.cache, w, k_pool, v_pool)
        self.segs = {}

    def layer(self, layer: int, q=None):
        w = self.w
        if layer not in self.segs:
            self.segs[layer] = H.build_layer(self.cache, w, layer)
        if q is None:
            q = wl.q_values(w, layer, self.dev)
        out = torch.full((w.T[layer], w.Hq, w.D), OUT_SENTINEL, dtype=torch.bfloat16, device=self.dev)
        lse = torch.full((w.Hq, w.T[layer]), LSE_SENTINEL, dtype=torch.float32, device=self.dev)
        B.segpa_attention_fwd(self.cache, self.segs[layer], q, w.scale, out, lse)
        torch.cuda.synchronize()
        return q, out, lse

    def close(self):
        B.segpa_destroy(self.cache)
        self.cache = None
        if self.bringup:
            B.use_library("product")


def compare(w, layer, k_pool, v_pool, q, out, lse, rows=None, label=""):
    """Element-by-element comparison with the fp64 oracle on the covered (row, head) pairs."""
    res = run_oracle(w, layer, k_pool, v_pool, q, row_subset=rows)
    sel = res.rows if rows is not None else np.arange(w.T[layer])
    cov = covered_mask(w, layer, sel)
    o = out[torch.from_numpy(sel).to(out.device)].to(torch.float64).cpu().numpy()
    ls = lse[:, torch.from_numpy(sel).to(lse.device)].to(torch.float64).cpu().numpy()
    assert cov.any()
    diff = np.abs(o - res.out)[cov]
    assert not np.isnan(o[cov]).any(), label + ": NaN in GPU output"
    dl = np.abs(ls.T - res.lse.T)[cov]
    worst = np.unravel_index(np.argmax(np.where(cov[..., None], np.abs(o - res.out), 0)), o.shape)
    msg = "%s: out max %.4g mean %.4g, lse max %.4g; worst at row %d head %d d %d (gpu %.5f oracle %.5f)" % (
        label, diff.max(), diff.mean(), dl.max(), sel[worst[0]], worst[1], worst[2], o[worst], res.out[worst])
    assert diff.max() <= TOL_OUT_MAX and diff.mean() <= TOL_OUT_MEAN and dl.max() <= TOL_LSE, msg
    # uncovered pairs must still hold the sentinels
    if (~cov).any():
        assert np.all(o[~cov] == OUT_SENTINEL), label + ": uncovered out rows were written"
        assert np.all(ls.T[~cov] == LSE_SENTINEL), label + ": uncovered lse entries were written"
    a, b = o[cov].ravel(), res.out[cov].ravel()
    cos = float(np.dot(a, b) / (np.linalg.norm(a) * np.linalg.norm(b) + 1e-300))
    assert cos > 0.99998, label + ": cosine %.7f (PAPER.md:350)" % cos
    return msg


def sample_rows(w, layer, n_random=256, seed=0, tile_edges=8, block_edges=6, ends=40, dense_tail=0):
    """Stratified row sample: the first and last `ends` rows of each segment (`dense_tail`: at
    least that many last rows), rows around `tile_edges` tile edges and `block_edges` 128-key block edges spread
    over the segment, plus seeded uniform rows (n_random over the layer).  Every row it picks is compared."""
    rng = np.random.default_rng(seed)
    rows = set()
    sm = w.stream_map()
    TT = 128 // w.G
    for s in w.layer_segments(layer):
        q0, ql = s.q_row_start, s.q_len
        kv = sm[(s.layer, s.kv_head, s.seq_id)].kv_len
        for t in list(range(min(ql, ends))) + list(range(max(0, ql - max(ends, dense_tail)), ql)):
            rows.add(q0 + t)
        for edge in range(TT, ql, TT * max(1, ql // (TT * tile_edges))):
            for d in (-1, 0, 1):
                if 0 <= edge + d < ql:
                    rows.add(q0 + edge + d)
        # rows whose position sits at a 128-key block edge
        p0 = kv - ql
        for blk in range((p0 // 128 + 1) * 128, kv, 128 * max(1, (kv - p0) // (128 * block_edges))):
            for d in (-1, 0, 1):
                t = blk + d - p0
                if 0 <= t < ql:
                    rows.add(q0 + t)
        if ql > 2 * ends:
            for t in rng.integers(0, ql, size=max(4, n_random // max(1, len(w.layer_segments(layer))))):
                rows.add(q0 + int(t))
    return np.array(sorted(rows), dtype=np.int64)
