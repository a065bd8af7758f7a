"""Shared test plumbing: runs the oracle on a Workload.  No method arithmetic here."""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_2606_06256_b200 import workloads as wl


def bits(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def from_bits(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).view(torch.bfloat16)


def widen(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().to(torch.float64).numpy()


def run_oracle(w: wl.Workload, layer, k_pool, v_pool, q, row_subset=None, want_p=0, segments=None):
    table, offs, kv_lens, index = wl.csr_page_tables(w, layer)
    segs = segments if segments is not None else w.layer_segments(layer)
    tup = [(index[(s.kv_head, s.seq_id)], s.kv_head, s.head_class, s.window, s.n_sink,
            s.q_row_start, s.q_len) for s in segs]
    seg_offsets, seg_lens = wl.csr_segment_tables(w, layer)
    return oracle.oracle_attention(Hq=w.Hq, Hkv=w.Hkv, D=w.D, P=w.P, k_pool=k_pool, v_pool=v_pool,
                                   page_table=table, pt_offsets=offs, kv_lens=kv_lens, segments=tup,
                                   q=q, T=w.T[layer], scale=w.scale, row_subset=row_subset,
                                   want_p=want_p, seg_offsets=seg_offsets, seg_lens=seg_lens)


def covered_mask(w: wl.Workload, layer, rows=None) -> np.ndarray:
    """bool [rows][Hq]: (row, head) pairs covered by some segment."""
    T = w.T[layer]
    m = np.zeros((T, w.Hq), dtype=bool)
    for s in w.layer_segments(layer):
        m[s.q_row_start:s.q_row_start + s.q_len, s.kv_head * w.G:(s.kv_head + 1) * w.G] = True
    return m if rows is None else m[rows]
