"""GPU-side test plumbing: run a Workload through libsegpa.so and compare with the oracle."""
from __future__ import annotations

import os

import numpy as np
import torch

from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
from tests.helpers import covered_mask, run_oracle

OUT_SENTINEL = 123.0
LSE_SENTINEL = -777.0
TOL_OUT_MAX, TOL_OUT_MEAN, TOL_LSE = 2e-2, 2e-3, 1e-3     # BASELINE.json:north_star


class GpuRun:
    def __init__(self, w: wl.Workload, kernel: str = "tc", tiles: int = 1, k_pool=None, v_pool=None):
        os.environ["SEGPA_KERNEL"] = kernel
        os.environ["SEGPA_TC_TILES"] = str(tiles)
        self.w = w
        self.dev = torch.device("cuda:0")
        if k_pool is None:
            k_pool, v_pool = wl.pool_values(w, self.dev)
        self.k_pool, self.v_pool = k_pool, v_pool
        self.cache = H.create_cache(w, 0)
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


def sample_rows(w, layer, n_random=256, seed=0):
    """Stratified row sample: heads and tails of each segment, rows around tile and
    128-key block edges, plus seeded uniform rows."""
    rng = np.random.default_rng(seed)
    rows = set()
    sm = w.stream_map()
    TT = 128 // w.G
    for s in w.layer_segments(layer):
        q0, ql = s.q_row_start, s.q_len
        kv = sm[(s.layer, s.kv_head, s.seq_id)].kv_len
        for t in list(range(min(ql, 40))) + list(range(max(0, ql - 40), ql)):
            rows.add(q0 + t)
        for edge in range(TT, ql, TT * max(1, ql // (TT * 8))):
            for d in (-1, 0, 1):
                if 0 <= edge + d < ql:
                    rows.add(q0 + edge + d)
        # rows whose position sits at a 128-key block edge
        p0 = kv - ql
        for blk in range((p0 // 128 + 1) * 128, kv, 128 * max(1, (kv - p0) // (128 * 6))):
            for d in (-1, 0, 1):
                t = blk + d - p0
                if 0 <= t < ql:
                    rows.add(q0 + t)
        if ql > 80:
            for t in rng.integers(0, ql, size=max(4, n_random // max(1, len(w.layer_segments(layer))))):
                rows.add(q0 + int(t))
    return np.array(sorted(rows), dtype=np.int64)
