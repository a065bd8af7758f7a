"""Seeded synthetic inputs for SegPagedAttention (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic: it only draws lengths, head classes, page
placements and random Q/K/V values, with the shapes and structure of the paper's workloads
(BASELINE.json:configs).  The paper measured on QA datasets with real models
(§5.1); none of that is available, so these inputs stand in for it.

Generation is pool-first: every pool page gets values, then page tables are drawn over it, so
page-table aliasing (config 4's shared prefixes) is meaningful.

Logical layouts handed to both sides (plain, row-major):
    k_pool, v_pool : [num_pages][P][D] bf16      one generic page = P tokens of one KV head
    q              : [T][Hq][D]        bf16      (per layer)
    stream         : (layer, kv_head, seq_id) -> kv_len, page_ids[ceil(kv_len/P)]
                     token j lives in page page_ids[j // P], slot j % P
                     (a stream with chunk_lens is the concatenation of head segments, each starting on a
                     fresh page: page_ids then holds sum ceil(n_s / P) pages and a segment's last page may be partial)
    segment        : (seq_id, kv_head, class, window W, n_sink, q_row_start, q_len)
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np
import torch

GLOBAL = 0
LOCAL = 1

BASE_SEED = 20260606


@dataclass
class Stream:
    layer: int
    kv_head: int
    seq_id: int
    kv_len: int
    page_ids: np.ndarray            # int32 [ceil(kv_len / P)]
    n_shared_prefix_pages: int = 0  # leading pages that alias another stream's pages
    shared_from: Optional[Tuple[int, int, int]] = None  # (layer, kv_head, seq_id) of the owner
    chunk_lens: Optional[List[int]] = None  # head segments (reused chunks), each on its own pages; None = one segment

    def chunks(self) -> List[int]:
        return [self.kv_len] if self.chunk_lens is None else list(self.chunk_lens)


@dataclass
class Segment:
    layer: int
    seq_id: int
    kv_head: int
    head_class: int   # GLOBAL | LOCAL
    window: int       # W = number of visible keys including self (LOCAL only; ignored for GLOBAL)
    n_sink: int
    q_row_start: int
    q_len: int


@dataclass
class Workload:
    name: str
    num_layers: int
    Hq: int
    Hkv: int
    D: int
    P: int
    num_pages: int
    scale: float
    streams: List[Stream]
    segments: List[Segment]
    T: List[int]                       # total query rows per layer
    seed: int
    k_channel_scale: Optional[np.ndarray] = None   # [Hkv][D] float32, config 2 outlier channels
    notes: Dict[str, object] = field(default_factory=dict)

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    def stream_map(self) -> Dict[Tuple[int, int, int], Stream]:
        return {(s.layer, s.kv_head, s.seq_id): s for s in self.streams}

    def layer_segments(self, layer: int) -> List[Segment]:
        return [s for s in self.segments if s.layer == layer]

    def layer_streams(self, layer: int) -> List[Stream]:
        return [s for s in self.streams if s.layer == layer]


# ----------------------------------------------------------------------------------------------
# values
# ----------------------------------------------------------------------------------------------

def _torch_gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def randn_bf16(shape, seed: int, device="cpu", chunk_elems: int = 1 << 27) -> torch.Tensor:
    """bf16 tensor of N(0,1) draws (rounded to nearest even from fp32). Chunked to bound memory."""
    out = torch.empty(shape, dtype=torch.bfloat16, device=device)
    flat = out.view(-1)
    g = _torch_gen(seed, device)
    n = flat.numel()
    for lo in range(0, n, chunk_elems):
        hi = min(n, lo + chunk_elems)
        flat[lo:hi] = torch.randn(hi - lo, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
    return out


def pool_values(w: Workload, device="cpu") -> Tuple[torch.Tensor, torch.Tensor]:
    """K and V pools [num_pages][P][D] bf16, every page filled (pool-first)."""
    k = randn_bf16((w.num_pages, w.P, w.D), w.seed * 16 + 1, device)
    v = randn_bf16((w.num_pages, w.P, w.D), w.seed * 16 + 2, device)
    if w.k_channel_scale is not None:
        # K = bf16(N(0,1) * c[h][d]); pages belong to one kv head each
        cs = torch.from_numpy(w.k_channel_scale).to(device)
        for s in w.streams:
            if s.shared_from is not None and s.n_shared_prefix_pages == len(s.page_ids):
                continue
            own = s.page_ids[s.n_shared_prefix_pages:]
            if len(own) == 0:
                continue
            idx = torch.from_numpy(own.astype(np.int64)).to(device)
            k[idx] = (k[idx].float() * cs[s.kv_head]).to(torch.bfloat16)
    return k, v


def q_values(w: Workload, layer: int, device="cpu") -> torch.Tensor:
    """Q [T][Hq][D] bf16 for one layer."""
    return randn_bf16((w.T[layer], w.Hq, w.D), w.seed * 16 + 3 + 7 * layer, device)


def stream_rows(pool: torch.Tensor, s: Stream, P: int, lo_page: int = 0) -> torch.Tensor:
    """Rows [n][D] of a stream's tokens starting at page index lo_page (plain gather, no arithmetic)."""
    if s.chunk_lens is not None:
        assert lo_page == 0
        return torch.cat([chunk_rows(pool, s, P, c) for c in range(len(s.chunk_lens))])
    idx = torch.from_numpy(s.page_ids[lo_page:].astype(np.int64)).to(pool.device)
    rows = pool[idx].reshape(-1, pool.shape[-1])
    n = s.kv_len - lo_page * P
    return rows[:n].contiguous()


def chunk_pages(s: Stream, P: int, c: int) -> np.ndarray:
    """page ids of head segment c of a stream (each segment starts on a fresh page)."""
    lens = s.chunks()
    first = sum(_pages_for(n, P) for n in lens[:c])
    return s.page_ids[first:first + _pages_for(lens[c], P)]


def chunk_rows(pool: torch.Tensor, s: Stream, P: int, c: int) -> torch.Tensor:
    """Rows [n_c][D] of head segment c of a stream."""
    idx = torch.from_numpy(chunk_pages(s, P, c).astype(np.int64)).to(pool.device)
    return pool[idx].reshape(-1, pool.shape[-1])[:s.chunks()[c]].contiguous()


# ----------------------------------------------------------------------------------------------
# oracle-side packing (CSR page tables); plain index plumbing
# ----------------------------------------------------------------------------------------------

def csr_page_tables(w: Workload, layer: int):
    """(page_table int32, pt_offsets int64 [n+1], kv_lens int64 [n], index {(kv_head, seq_id): i})"""
    ss = w.layer_streams(layer)
    offs = np.zeros(len(ss) + 1, dtype=np.int64)
    for i, s in enumerate(ss):
        offs[i + 1] = offs[i] + len(s.page_ids)
    table = np.concatenate([s.page_ids for s in ss]).astype(np.int32) if ss else np.zeros(0, np.int32)
    kv_lens = np.array([s.kv_len for s in ss], dtype=np.int64)
    index = {(s.kv_head, s.seq_id): i for i, s in enumerate(ss)}
    return table, offs, kv_lens, index


def csr_segment_tables(w: Workload, layer: int):
    """Head-segment table of the layer's streams (same stream order as csr_page_tables): (seg_offsets int64 [n+1],
    seg_lens int64), or (None, None) when every stream is a single segment."""
    ss = w.layer_streams(layer)
    if all(s.chunk_lens is None for s in ss):
        return None, None
    offs = np.zeros(len(ss) + 1, dtype=np.int64)
    lens: List[int] = []
    for i, s in enumerate(ss):
        lens += s.chunks()
        offs[i + 1] = len(lens)
    return offs, np.array(lens, dtype=np.int64)


# ----------------------------------------------------------------------------------------------
# structure helpers
# ----------------------------------------------------------------------------------------------

def _pages_for(kv_len: int, P: int) -> int:
    return (kv_len + P - 1) // P


def _place(rng: np.random.Generator, n_live: int, num_pages: int) -> np.ndarray:
    """first n_live entries of a seeded permutation of [0, num_pages)."""
    return rng.permutation(num_pages)[:n_live].astype(np.int32)


def visible_pairs(kv_len: int, q_len: int, head_class: int, W: int, n_sink: int = 0) -> int:
    """Number of attended (query, key) pairs of one q head of a segment. Pure counting, used for
    the useful-FLOP figure (4*D per pair per q head)."""
    p0 = kv_len - q_len
    i = np.arange(p0, kv_len, dtype=np.int64)
    if head_class == GLOBAL:
        return int((i + 1).sum())
    win = np.minimum(i + 1, W)
    first = i - win + 1                      # first key inside the window
    sinks = np.minimum(n_sink, first)        # sink keys not already inside the window
    return int((win + np.maximum(sinks, 0)).sum())


def useful_flops(w: Workload, layer: Optional[int] = None) -> int:
    sm = w.stream_map()
    tot = 0
    for s in w.segments:
        if layer is not None and s.layer != layer:
            continue
        kv_len = sm[(s.layer, s.kv_head, s.seq_id)].kv_len
        tot += w.G * visible_pairs(kv_len, s.q_len, s.head_class, s.window, s.n_sink)
    return 4 * w.D * tot


def make_workload(name: str, *, Hq: int, Hkv: int, D: int, P: int, requests, seed: int,
                  num_layers: int = 1, pool_factor: float = 1.5, scale: Optional[float] = None,
                  identity_pages: bool = False) -> Workload:
    """Generic builder used by the tests.

    requests: list of dicts {kv_len, heads: {kv_head: (class, W, n_sink, q_len)}[, chunks: [n_0, n_1, ...]]}; each
    request's q rows are packed consecutively, q_row_start shared by its heads; a head with a shorter q_len
    takes the LAST q_len rows of the request's row range (bottom-right).  "chunks" (summing to
    kv_len) makes every stream of the request a concatenation of head segments of those lengths, each on its own
    pages (reused chunks of arbitrary length: ragged chunk tails).
    """
    rng = np.random.default_rng(seed)

    def npages(r):
        return sum(_pages_for(n, P) for n in r["chunks"]) if "chunks" in r else _pages_for(r["kv_len"], P)
    n_live = 0
    for _ in range(num_layers):
        for r in requests:
            assert "chunks" not in r or sum(r["chunks"]) == r["kv_len"]
            n_live += len(r["heads"]) * npages(r)
    num_pages = max(1, int(math.ceil(pool_factor * n_live)))
    place = np.arange(n_live, dtype=np.int32) if identity_pages else _place(rng, n_live, num_pages)
    streams, segments, T = [], [], []
    cur = 0
    for layer in range(num_layers):
        row = 0
        for sid, r in enumerate(requests):
            qmax = max(h[3] for h in r["heads"].values())
            for kvh, (cls, W, n_sink, q_len) in sorted(r["heads"].items()):
                npg = npages(r)
                streams.append(Stream(layer, kvh, sid, r["kv_len"], place[cur:cur + npg].copy(),
                                      chunk_lens=list(r["chunks"]) if "chunks" in r else None))
                cur += npg
                segments.append(Segment(layer, sid, kvh, cls, W, n_sink, row + qmax - q_len, q_len))
            row += qmax
        T.append(row)
    return Workload(name, num_layers, Hq, Hkv, D, P, num_pages,
                    float(np.float32(scale if scale is not None else 1.0 / math.sqrt(D))),
                    streams, segments, T, seed)


# ----------------------------------------------------------------------------------------------
# the five BASELINE.json configs; seeds: BASE_SEED + c
# ----------------------------------------------------------------------------------------------

def config1() -> Workload:
    """Tiny: 1 layer, Hq 8, Hkv 2, D 64, P 16; kv 1024, last 512 are queries; head 0 GLOBAL,
    head 1 LOCAL W=128 (BASELINE.json:configs[0])."""
    w = make_workload("cfg1_tiny", Hq=8, Hkv=2, D=64, P=16, seed=BASE_SEED + 1,
                      requests=[{"kv_len": 1024, "heads": {0: (GLOBAL, 0, 0, 512), 1: (LOCAL, 128, 0, 512)}}],
                      scale=0.125)
    return w


def config2() -> Workload:
    """Llama-3-8B-shaped layer: Hq 32, Hkv 8, D 128, P 16; 4 requests L~U{2048..8192} fully
    prefilled; head 0 GLOBAL, heads 1-7 LOCAL W=1024; K outlier channels (BASELINE.json:configs[1])."""
    seed = BASE_SEED + 2
    rng = np.random.default_rng(seed * 16)
    Ls = [int(x) for x in rng.integers(2048, 8193, size=4)]
    reqs = []
    for L in Ls:
        heads = {0: (GLOBAL, 0, 0, L)}
        for h in range(1, 8):
            heads[h] = (LOCAL, 1024, 0, L)
        reqs.append({"kv_len": L, "heads": heads})
    w = make_workload("cfg2_llama8b_layer", Hq=32, Hkv=8, D=128, P=16, seed=seed, requests=reqs)
    crng = np.random.default_rng(seed * 16 + 5)
    w.k_channel_scale = np.exp(crng.normal(0.0, 0.5, size=(8, 128))).astype(np.float32)
    w.notes["lengths"] = Ls
    return w


def _cfg3_chunks(rng: np.random.Generator, P: int, total: int = 64512, n: int = 12) -> List[int]:
    """12 chunk lengths U{2048..8192}, multiples of P, rescaled to sum to `total`."""
    raw = rng.integers(2048, 8193, size=n).astype(np.float64)
    lens = np.clip(np.round(raw * (total / raw.sum()) / P) * P, 2048, 8192).astype(np.int64)
    # fix the residue in page-sized steps without leaving [2048, 8192]
    diff = int(total - lens.sum())
    i = n - 1
    guard = 0
    while diff != 0 and guard < 100000:
        step = P if diff > 0 else -P
        if 2048 <= lens[i] + step <= 8192:
            lens[i] += step
            diff -= step
        else:
            i = (i - 1) % n
        guard += 1
    assert lens.sum() == total, (lens, total)
    return [int(x) for x in lens]


def config3() -> Workload:
    """Llama-3.3-70B-shaped 64K prompt: Hq 64, Hkv 8, D 128, P 16; head 0 GLOBAL queries all 65536
    rows; heads 1-7 LOCAL W=2048 query only the 1024-token suffix (BASELINE.json:configs[2])."""
    seed = BASE_SEED + 3
    rng = np.random.default_rng(seed * 16)
    chunks = _cfg3_chunks(rng, 16)
    L = 65536
    heads = {0: (GLOBAL, 0, 0, L)}
    for h in range(1, 8):
        heads[h] = (LOCAL, 2048, 0, 1024)
    w = make_workload("cfg3_llama70b_64k", Hq=64, Hkv=8, D=128, P=16, seed=seed,
                      requests=[{"kv_len": L, "heads": heads}])
    w.notes["chunks"] = chunks
    return w


def config4(decode_only: bool = False) -> Workload:
    """Mixed serving batch: 64 requests, Hq 32, Hkv 8, D 128, P 16; ctx log-uniform 4096..32768;
    q mix 32 decode / 19 in 16..256 / 13 in 1024..4096; 67/512 segments GLOBAL; LOCAL W=2048;
    8 groups x 8 requests share a prefix by page-table aliasing (BASELINE.json:configs[3];
    SURVEY A11-A13).  decode_only=True keeps only the q=1 requests (reported as "4d")."""
    seed = BASE_SEED + 4
    Hq, Hkv, D, P = 32, 8, 128, 16
    rng = np.random.default_rng(seed * 16)
    n_req = 64
    ctx = np.round(np.exp(rng.uniform(math.log(4096), math.log(32768), size=n_req))).astype(np.int64)
    ctx = np.clip(ctx, 4096, 32768)
    kinds = np.array([0] * 32 + [1] * 19 + [2] * 13)
    rng.shuffle(kinds)
    qlen = np.where(kinds == 0, 1, np.where(kinds == 1, rng.integers(16, 257, size=n_req),
                                            rng.integers(1024, 4097, size=n_req))).astype(np.int64)
    g0 = int(rng.integers(0, Hkv))
    cls = np.full((n_req, Hkv), LOCAL, dtype=np.int64)
    cls[:, g0] = GLOBAL
    cand = [(r, h) for r in range(n_req) for h in range(Hkv) if h != g0]
    for k in rng.choice(len(cand), size=3, replace=False):
        cls[cand[k][0], cand[k][1]] = GLOBAL
    # shared prefixes: 8 groups of 8 consecutive requests
    prefix_pages = np.zeros(n_req, dtype=np.int64)
    for g in range(8):
        members = range(8 * g, 8 * g + 8)
        pp = int((0.5 * min(int(ctx[r]) for r in members)) // P)
        for r in members:
            prefix_pages[r] = pp
    # count live pages (owner's prefix counted once)
    n_live = 0
    for r in range(n_req):
        npg = _pages_for(int(ctx[r]), P)
        own = npg if r % 8 == 0 else npg - int(prefix_pages[r])
        n_live += Hkv * own
    num_pages = int(math.ceil(1.5 * n_live))
    place = _place(np.random.default_rng(seed * 16 + 4), n_live, num_pages)
    cur = 0
    streams: List[Stream] = []
    segments: List[Segment] = []
    owner_pages: Dict[Tuple[int, int], np.ndarray] = {}
    row = 0
    for r in range(n_req):
        npg = _pages_for(int(ctx[r]), P)
        keep = (not decode_only) or qlen[r] == 1
        for h in range(Hkv):
            if r % 8 == 0:
                ids = place[cur:cur + npg].copy()
                cur += npg
                owner_pages[(r // 8, h)] = ids
                st = Stream(0, h, r, int(ctx[r]), ids)
            else:
                pp = int(prefix_pages[r])
                own = place[cur:cur + npg - pp].copy()
                cur += npg - pp
                ids = np.concatenate([owner_pages[(r // 8, h)][:pp], own]).astype(np.int32)
                st = Stream(0, h, r, int(ctx[r]), ids, n_shared_prefix_pages=pp,
                            shared_from=(0, h, 8 * (r // 8)))
            streams.append(st)       # streams are always all present (aliasing needs the owners)
            if keep:
                segments.append(Segment(0, r, h, int(cls[r, h]), 2048, 0, row, int(qlen[r])))
        if keep:
            row += int(qlen[r])
    w = Workload("cfg4_mixed_batch" + ("_decode_only" if decode_only else ""), 1, Hq, Hkv, D, P,
                 num_pages, float(np.float32(1.0 / math.sqrt(D))), streams, segments, [row], seed)
    w.notes.update(ctx=ctx.tolist(), qlen=qlen.tolist(), g0=g0,
                   n_global=int((cls == GLOBAL).sum()), prefix_pages=prefix_pages.tolist())
    return w


def config5(num_layers: int = 28) -> Workload:
    """Qwen2-7B-shaped sweep: 28 layers x 4 KV heads (Hq 28, G=7), D 128, P 32; 16 of 112
    (layer, head) pairs GLOBAL, rest LOCAL W=4096; one 32768-token prompt fully prefilled
    (BASELINE.json:configs[4]).  num_layers<28 keeps the first layers of the SAME class map."""
    seed = BASE_SEED + 5
    Hq, Hkv, D, P, L = 28, 4, 128, 32, 32768
    rng = np.random.default_rng(seed * 16)
    gl = set(int(x) for x in rng.choice(28 * Hkv, size=16, replace=False))
    npg = _pages_for(L, P)
    n_live = num_layers * Hkv * npg
    num_pages = int(math.ceil(1.5 * n_live))
    place = _place(np.random.default_rng(seed * 16 + 4), n_live, num_pages)
    streams, segments = [], []
    cur = 0
    for layer in range(num_layers):
        for h in range(Hkv):
            ids = place[cur:cur + npg].copy()
            cur += npg
            streams.append(Stream(layer, h, 0, L, ids))
            c = GLOBAL if (layer * Hkv + h) in gl else LOCAL
            segments.append(Segment(layer, 0, h, c, 4096, 0, 0, L))
    w = Workload("cfg5_qwen2_7b_sweep", num_layers, Hq, Hkv, D, P, num_pages,
                 float(np.float32(1.0 / math.sqrt(D))), streams, segments, [L] * num_layers, seed)
    w.notes["global_pairs"] = sorted(gl)
    return w


def fig9(L: int, mode: str, num_layers: int = 8) -> Workload:
    """The paper's own kernel-isolated micro-benchmark shape (Fig. 9(e)-(h)): Qwen3-32B-shaped
    layers, Hq 32 / Hkv 8 (GQA-4), D 128, bf16; half of the KV heads GLOBAL (full context), half LOCAL with a
    320-token visible set (sink + recent: n_sink 4 + W 316); contexts 8K / 32K / 128K; one request.
    mode "decode": q_len 1; mode "prefill": q_len = L (the paper does not state its prefill query length).
    The paper runs 64 layers sequentially; here `num_layers` distinct layers are generated (enough that the
    KV of consecutive launches never sits in L2 together) and the 64-layer figure is per-layer time x 64."""
    assert mode in ("decode", "prefill")
    seed = BASE_SEED + 9 + (0 if mode == "decode" else 1) + L
    Hq, Hkv, D, P = 32, 8, 128, 16
    q_len = 1 if mode == "decode" else L
    heads = {h: ((GLOBAL, 0, 0, q_len) if h < 4 else (LOCAL, 316, 4, q_len)) for h in range(Hkv)}
    w = make_workload("fig9_%s_%dk" % (mode, L // 1024), Hq=Hq, Hkv=Hkv, D=D, P=P, seed=seed, num_layers=num_layers,
                      requests=[{"kv_len": L, "heads": heads}])
    return w


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
