"""Feeds a workloads.Workload through the C ABI (segpa_create_cache / segpa_append_pages /
segpa_build_segments).  Plumbing only; used by tests/, bench.py and __graft_entry__.smoke()."""
from __future__ import annotations

from typing import Dict, List, Optional, Tuple

import numpy as np

from . import binding as B
from . import workloads as wl


def create_cache(w: wl.Workload, device: int = 0, tiles_per_item: int = 0) -> int:
    return B.segpa_create_cache(num_layers=w.num_layers, num_q_heads=w.Hq, num_kv_heads=w.Hkv, head_dim=w.D,
                                page_size=w.P, num_pages=w.num_pages, device=device, tiles_per_item=tiles_per_item)


def append_requests(w: wl.Workload, k_pool=None, v_pool=None) -> List[tuple]:
    """The workload's appends as segpa_append_pages_batch request tuples: owners first (copy mode with
    the workload's page placement), then aliasing streams (attach the shared prefix pages, copy the rest).
    k_pool / v_pool: torch bf16 [num_pages][P][D] on the cache's device, or None for a planning-only
    cache (attach everything)."""
    owners = [s for s in w.streams if s.shared_from is None]
    aliased = [s for s in w.streams if s.shared_from is not None]
    reqs = []
    for s in owners + aliased:
        if s.chunk_lens is not None:
            # A stream spliced from reused chunks (PIC): every chunk but the last is first stored under an
            # id of its own (what an offline cache holds) and then ATTACHED, each chunk on its own pages whatever its
            # length; the last chunk is the request's new suffix, copied in (it starts a fresh page after the attach).
            for c, n in enumerate(s.chunk_lens):
                ids = wl.chunk_pages(s, w.P, c)
                last = c == len(s.chunk_lens) - 1
                if k_pool is None:
                    reqs.append((s.layer, s.kv_head, s.seq_id, None, None, n, ids))
                elif last:
                    reqs.append((s.layer, s.kv_head, s.seq_id, wl.chunk_rows(k_pool, s, w.P, c), wl.chunk_rows(v_pool, s, w.P, c), n, ids))
                else:
                    src = chunk_source_id(s.seq_id, c)
                    reqs.append((s.layer, s.kv_head, src, wl.chunk_rows(k_pool, s, w.P, c), wl.chunk_rows(v_pool, s, w.P, c), n, ids))
                    reqs.append((s.layer, s.kv_head, s.seq_id, None, None, n, ids))
            continue
        if k_pool is None:
            reqs.append((s.layer, s.kv_head, s.seq_id, None, None, s.kv_len, s.page_ids))
            continue
        pp = s.n_shared_prefix_pages
        if pp > 0:
            reqs.append((s.layer, s.kv_head, s.seq_id, None, None, pp * w.P, s.page_ids[:pp]))
        n_rest = s.kv_len - pp * w.P
        if n_rest > 0:
            kr = wl.stream_rows(k_pool, s, w.P, lo_page=pp)
            vr = wl.stream_rows(v_pool, s, w.P, lo_page=pp)
            reqs.append((s.layer, s.kv_head, s.seq_id, kr, vr, n_rest, s.page_ids[pp:]))
    return reqs


def chunk_source_id(seq_id: int, c: int) -> int:
    """seq_id under which reused chunk c of a spliced stream is stored before it is attached."""
    return (c + 1) * (1 << 32) + seq_id


def append_workload(cache: int, w: wl.Workload, k_pool=None, v_pool=None, stream=None, batched: bool = True) -> None:
    """Stores the whole workload: one segpa_append_pages_batch call, or (batched=False) one
    segpa_append_pages call per request."""
    reqs = append_requests(w, k_pool, v_pool)
    if batched:
        B.segpa_append_pages_batch(cache, reqs, stream=stream)
        return
    for (layer, kvh, seq, kr, vr, n, ids) in reqs:
        B.segpa_append_pages(cache, layer, kvh, seq, kr, vr, n, page_ids=ids, stream=stream)


def segment_reqs(w: wl.Workload, layer: int) -> List[tuple]:
    return [(s.seq_id, s.kv_head, s.head_class, s.window, s.n_sink, s.q_row_start, s.q_len)
            for s in w.layer_segments(layer)]


def build_layer(cache: int, w: wl.Workload, layer: int, stream=None) -> int:
    return B.segpa_build_segments(cache, layer, segment_reqs(w, layer), stream=stream)
