"""Thin ctypes binding of libsegpa.so (include/segpa.h).  Argument marshalling only: every step
of the path runs inside the library's host code and CUDA kernels.  Fails loudly when the shared
library is missing; there is no fallback of any kind.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsegpa.so")
# test build: the same sources compiled with -DSEGPA_BRINGUP (adds the SIMT cross-check kernel and one extra
# symbol, segpa_bringup_use_simt); never loaded unless a test asks for it with use_library("bringup")
BRINGUP_LIB_PATH = os.path.join(_HERE, "libsegpa_bringup.so")

OK, ERR_INVALID, ERR_OOM, ERR_CUDA, ERR_UNSUPPORTED, ERR_STATE = range(6)
GLOBAL, LOCAL = 0, 1
_STATUS = {0: "OK", 1: "INVALID", 2: "OOM", 3: "CUDA", 4: "UNSUPPORTED", 5: "STATE"}

EXPORTS = [
    "segpa_pool_bytes", "segpa_create_cache", "segpa_append_pages", "segpa_append_pages_batch",
    "segpa_clear_streams", "segpa_evict_pages", "segpa_rope_align", "segpa_rope_align_batch", "segpa_gather_rows", "segpa_gather_rows_noalloc", "segpa_free_stream",
    "segpa_stream_info", "segpa_pool_stats", "segpa_build_segments", "segpa_free_segments",
    "segpa_segments_stats", "segpa_segments_items", "segpa_segments_pages", "segpa_attention_fwd",
    "segpa_attention_fwd_host", "segpa_attention_fwd_host_async", "segpa_host_wait", "segpa_merge", "segpa_segments_mass_layout", "segpa_attention_mass",
    "segpa_mass_select", "segpa_last_launch_count", "segpa_destroy", "segpa_last_error",
    "segpa_version",
]


class SegpaError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__("segpa: %s: %s" % (_STATUS.get(status, status), msg))
        self.status = status


class CacheDesc(C.Structure):
    _fields_ = [("num_layers", C.c_int32), ("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("page_size", C.c_int32), ("device", C.c_int32),
                ("num_pages", C.c_int64), ("k_pool", C.c_void_p), ("v_pool", C.c_void_p),
                ("tiles_per_item", C.c_int32), ("reserved", C.c_int32)]


class SegmentReq(C.Structure):
    _fields_ = [("seq_id", C.c_int64), ("kv_head", C.c_int32), ("head_class", C.c_int32),
                ("window", C.c_int32), ("n_sink", C.c_int32), ("q_row_start", C.c_int64),
                ("q_len", C.c_int32), ("reserved", C.c_int32)]


class AppendReq(C.Structure):
    _fields_ = [("layer", C.c_int32), ("kv_head", C.c_int32), ("seq_id", C.c_int64), ("k_src", C.c_void_p),
                ("v_src", C.c_void_p), ("src_row_stride_elems", C.c_int64), ("n_tokens", C.c_int64),
                ("page_ids", C.c_void_p), ("n_page_ids", C.c_int32), ("src_is_host", C.c_int32)]


class RopeReq(C.Structure):
    _fields_ = [("layer", C.c_int32), ("kv_head", C.c_int32), ("seq_id", C.c_int64), ("first_token", C.c_int64),
                ("n_tokens", C.c_int64), ("delta_pos", C.c_int64)]


class PlanStats(C.Structure):
    _fields_ = [("n_segments", C.c_int32), ("n_tiles", C.c_int32), ("n_items", C.c_int32),
                ("n_split_tiles", C.c_int32), ("tile_tokens", C.c_int32), ("block_keys", C.c_int32),
                ("kv_blocks", C.c_int64), ("attended_pairs", C.c_int64), ("q_rows", C.c_int64),
                ("visible_kv_tokens", C.c_int64), ("workspace_bytes", C.c_int64)]


class Item(C.Structure):
    _fields_ = [("segment", C.c_int32), ("t0", C.c_int32), ("n_tok", C.c_int32), ("kb_lo", C.c_int32),
                ("kb_hi", C.c_int32), ("split", C.c_int32), ("n_splits", C.c_int32), ("tile", C.c_int32),
                ("cta", C.c_int32), ("reserved", C.c_int32)]


_lib = None
_libs = {}
_which = "product"


def use_library(which: str) -> None:
    """"product" (libsegpa.so, the default) or "bringup" (the test build): the library the functions below call."""
    global _lib, _which
    assert which in ("product", "bringup")
    _which = which
    _lib = _libs.get(which)


def segpa_bringup_use_simt(cache: int, on: bool = True) -> None:
    """Test build only: run this cache's plans on the SIMT cross-check kernel."""
    assert _which == "bringup", "segpa_bringup_use_simt exists only in libsegpa_bringup.so"
    L = lib()
    L.segpa_bringup_use_simt.argtypes = [C.c_void_p, C.c_int32]
    _check(L.segpa_bringup_use_simt(cache, 1 if on else 0))


def lib():
    global _lib
    if _lib is None:
        path = LIB_PATH if _which == "product" else BRINGUP_LIB_PATH
        if not os.path.exists(path):
            raise ImportError("%s is not built (%s); run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "or `python paper_2606_06256_b200/build.py`. There is no fallback path." % (os.path.basename(path), path))
        L = C.CDLL(path)
        L.segpa_pool_bytes.restype = C.c_int64
        L.segpa_last_error.restype = C.c_char_p
        L.segpa_version.restype = C.c_int32
        L.segpa_last_launch_count.restype = C.c_int32
        L.segpa_last_launch_count.argtypes = [C.c_void_p]
        L.segpa_create_cache.argtypes = [C.POINTER(CacheDesc), C.POINTER(C.c_void_p)]
        L.segpa_append_pages.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p,
                                         C.c_int64, C.c_int64, C.c_void_p, C.c_int32, C.c_void_p]
        L.segpa_append_pages_batch.argtypes = [C.c_void_p, C.POINTER(AppendReq), C.c_int32, C.c_void_p]
        L.segpa_clear_streams.argtypes = [C.c_void_p]
        L.segpa_rope_align.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int64, C.c_int64, C.c_int64,
                                       C.c_double, C.c_void_p]
        L.segpa_rope_align_batch.argtypes = [C.c_void_p, C.POINTER(RopeReq), C.c_int32, C.c_double, C.c_void_p]
        L.segpa_gather_rows.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int64, C.c_int64, C.c_void_p,
                                        C.c_void_p, C.c_int64, C.c_void_p]
        L.segpa_gather_rows_noalloc.argtypes = L.segpa_gather_rows.argtypes
        L.segpa_evict_pages.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int32, C.c_int32]
        L.segpa_free_stream.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64]
        L.segpa_stream_info.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.POINTER(C.c_int64),
                                        C.POINTER(C.c_int32), C.c_void_p, C.c_int32]
        L.segpa_pool_stats.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.segpa_build_segments.argtypes = [C.c_void_p, C.c_int32, C.POINTER(SegmentReq), C.c_int32,
                                           C.POINTER(C.c_void_p), C.c_void_p]
        L.segpa_free_segments.argtypes = [C.c_void_p, C.c_void_p]
        L.segpa_segments_stats.argtypes = [C.c_void_p, C.POINTER(PlanStats)]
        L.segpa_segments_items.argtypes = [C.c_void_p, C.POINTER(Item), C.c_int32, C.POINTER(C.c_int32)]
        L.segpa_segments_pages.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.c_void_p, C.c_int32,
                                           C.POINTER(C.c_int32)]
        L.segpa_attention_fwd.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_void_p,
                                          C.c_int64, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
        L.segpa_attention_fwd_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p,
                                               C.c_void_p, C.c_int64, C.c_void_p]
        L.segpa_attention_fwd_host_async.argtypes = L.segpa_attention_fwd_host.argtypes
        L.segpa_host_wait.argtypes = [C.c_void_p]
        L.segpa_merge.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64,
                                  C.c_int64, C.c_int64, C.c_void_p]
        L.segpa_segments_mass_layout.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        L.segpa_attention_mass.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_void_p, C.c_int64,
                                           C.c_int64, C.c_void_p, C.c_int64, C.c_void_p]
        L.segpa_mass_select.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
        L.segpa_destroy.argtypes = [C.c_void_p]
        _lib = L
        _libs[_which] = L
    return _lib


def _check(rc: int):
    if rc != OK:
        raise SegpaError(rc, lib().segpa_last_error().decode())


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        return None
    return int(getattr(stream, "cuda_stream", stream))


# ---------------------------------------------------------------------------------------------
# same names as the C ABI
# ---------------------------------------------------------------------------------------------

def segpa_create_cache(*, num_layers: int, num_q_heads: int, num_kv_heads: int, head_dim: int,
                       page_size: int, num_pages: int, device: int = 0, k_pool: int = 0, v_pool: int = 0,
                       tiles_per_item: int = 0) -> int:
    d = CacheDesc(num_layers, num_q_heads, num_kv_heads, head_dim, page_size, device, num_pages,
                  k_pool or None, v_pool or None, tiles_per_item, 0)
    out = C.c_void_p()
    _check(lib().segpa_create_cache(C.byref(d), C.byref(out)))
    return out.value


def segpa_append_pages(cache: int, layer: int, kv_head: int, seq_id: int, k_src, v_src, n_tokens: int,
                       page_ids: Optional[Sequence[int]] = None, src_row_stride_elems: Optional[int] = None,
                       stream=None) -> None:
    """k_src / v_src: torch bf16 device tensors [n_tokens][D] (rows may be strided), or None to attach."""
    kp = vp = None
    stride = 0
    if k_src is not None:
        assert k_src.is_cuda and v_src.is_cuda and k_src.stride(-1) == 1 and v_src.stride(-1) == 1
        assert k_src.stride(0) == v_src.stride(0)
        kp, vp = k_src.data_ptr(), v_src.data_ptr()
        stride = src_row_stride_elems if src_row_stride_elems is not None else k_src.stride(0)
    ids = None
    n_ids = 0
    if page_ids is not None:
        ids = np.ascontiguousarray(page_ids, dtype=np.int32)
        n_ids = len(ids)
    _check(lib().segpa_append_pages(cache, layer, kv_head, seq_id, kp, vp, stride, n_tokens,
                                    ids.ctypes.data_as(C.c_void_p) if ids is not None else None, n_ids,
                                    _stream_ptr(stream)))


class AppendBatch:
    """Marshalled argument array of segpa_append_pages_batch; can be prepared once and passed again
    (the tensors and page-id arrays it refers to are kept alive here)."""

    def __init__(self, reqs: Sequence[tuple]):
        """reqs: tuples (layer, kv_head, seq_id, k_src, v_src, n_tokens, page_ids) with k_src / v_src torch
        bf16 tensors [n_tokens][D] -- on the device, or on the host (src_is_host) -- or None (attach), page_ids an
        int sequence or None."""
        self.n = len(reqs)
        self.arr = (AppendReq * max(1, self.n))()
        self._keep = []
        for i, (layer, kvh, seq, k_src, v_src, n_tokens, page_ids) in enumerate(reqs):
            kp = vp = None
            stride = 0
            on_host = 0
            if k_src is not None:
                assert k_src.is_cuda == v_src.is_cuda and k_src.stride(-1) == 1 and v_src.stride(-1) == 1
                assert k_src.stride(0) == v_src.stride(0)
                kp, vp, stride = k_src.data_ptr(), v_src.data_ptr(), k_src.stride(0)
                on_host = 0 if k_src.is_cuda else 1       # CPU tensors (pinned for speed) go through src_is_host
                self._keep.append((k_src, v_src))
            ip, n_ids = None, 0
            if page_ids is not None:
                ids = np.ascontiguousarray(page_ids, dtype=np.int32)
                self._keep.append(ids)
                ip, n_ids = ids.ctypes.data, len(ids)
            self.arr[i] = AppendReq(int(layer), int(kvh), int(seq), kp, vp, int(stride), int(n_tokens), ip, n_ids, on_host)


def segpa_append_pages_batch(cache: int, batch, stream=None) -> None:
    """batch: an AppendBatch, or the list of tuples AppendBatch takes."""
    if not isinstance(batch, AppendBatch):
        batch = AppendBatch(batch)
    _check(lib().segpa_append_pages_batch(cache, batch.arr, batch.n, _stream_ptr(stream)))


def segpa_evict_pages(cache: int, layer: int, kv_head: int, seq_id: int, first_page_index: int, n_pages: int) -> None:
    _check(lib().segpa_evict_pages(cache, layer, kv_head, seq_id, first_page_index, n_pages))


def segpa_rope_align(cache: int, layer: int, kv_head: int, seq_id: int, first_token: int, n_tokens: int,
                     delta_pos: int, rope_base: float = 10000.0, stream=None) -> None:
    _check(lib().segpa_rope_align(cache, layer, kv_head, seq_id, first_token, n_tokens, delta_pos, rope_base,
                                  _stream_ptr(stream)))


class RopeBatch:
    """Marshalled segpa_rope_req_t array; can be prepared once and passed again."""

    def __init__(self, reqs: Sequence[tuple]):
        """reqs: tuples (layer, kv_head, seq_id, first_token, n_tokens, delta_pos)."""
        self.n = len(reqs)
        self.arr = (RopeReq * max(1, self.n))()
        for i, r in enumerate(reqs):
            self.arr[i] = RopeReq(*[int(x) for x in r])


def segpa_rope_align_batch(cache: int, reqs, rope_base: float = 10000.0, stream=None) -> None:
    """reqs: a RopeBatch, or the list of tuples RopeBatch takes."""
    if not isinstance(reqs, RopeBatch):
        reqs = RopeBatch(reqs)
    _check(lib().segpa_rope_align_batch(cache, reqs.arr, reqs.n, rope_base, _stream_ptr(stream)))


def segpa_gather_rows(cache: int, layer: int, kv_head: int, seq_id: int, first_token: int, n_tokens: int,
                      k_dst=None, v_dst=None, stream=None) -> None:
    """k_dst / v_dst: torch bf16 device tensors [n_tokens][D] (rows may be strided) or None."""
    ref = k_dst if k_dst is not None else v_dst
    assert ref is not None and ref.is_cuda and ref.stride(-1) == 1
    if k_dst is not None and v_dst is not None:
        assert k_dst.stride(0) == v_dst.stride(0)
    _check(lib().segpa_gather_rows(cache, layer, kv_head, seq_id, first_token, n_tokens,
                                   k_dst.data_ptr() if k_dst is not None else None,
                                   v_dst.data_ptr() if v_dst is not None else None, ref.stride(0), _stream_ptr(stream)))


NOALLOC_MAX_PAGES = 16384


def segpa_gather_rows_noalloc(cache: int, layer: int, kv_head: int, seq_id: int, first_token: int, n_tokens: int,
                              k_dst=None, v_dst=None, stream=None) -> None:
    """segpa_gather_rows without any device allocation (fixed 64 KB scratch in the library; at most NOALLOC_MAX_PAGES
    pages per call; calls that overlap on the GPU race on the scratch)."""
    ref = k_dst if k_dst is not None else v_dst
    assert ref is not None and ref.is_cuda and ref.stride(-1) == 1
    if k_dst is not None and v_dst is not None:
        assert k_dst.stride(0) == v_dst.stride(0)
    _check(lib().segpa_gather_rows_noalloc(cache, layer, kv_head, seq_id, first_token, n_tokens,
                                           k_dst.data_ptr() if k_dst is not None else None,
                                           v_dst.data_ptr() if v_dst is not None else None, ref.stride(0), _stream_ptr(stream)))


def segpa_clear_streams(cache: int) -> None:
    _check(lib().segpa_clear_streams(cache))


def segpa_free_stream(cache: int, layer: int, kv_head: int, seq_id: int) -> None:
    _check(lib().segpa_free_stream(cache, layer, kv_head, seq_id))


def segpa_stream_info(cache: int, layer: int, kv_head: int, seq_id: int):
    kv_len, n_pages = C.c_int64(), C.c_int32()
    _check(lib().segpa_stream_info(cache, layer, kv_head, seq_id, C.byref(kv_len), C.byref(n_pages), None, 0))
    ids = np.zeros(n_pages.value, dtype=np.int32)
    _check(lib().segpa_stream_info(cache, layer, kv_head, seq_id, None, None, ids.ctypes.data_as(C.c_void_p),
                                   n_pages.value))
    return kv_len.value, ids


def segpa_pool_stats(cache: int):
    a, b = C.c_int64(), C.c_int64()
    _check(lib().segpa_pool_stats(cache, C.byref(a), C.byref(b)))
    return a.value, b.value


class SegmentBatch:
    """Marshalled segpa_segment_req_t array; can be prepared once and passed again."""

    def __init__(self, reqs: Sequence[tuple]):
        """reqs: tuples (seq_id, kv_head, head_class, window, n_sink, q_row_start, q_len)."""
        self.n = len(reqs)
        self.arr = (SegmentReq * max(1, self.n))()
        for i, (seq, kvh, cls, W, ns, qs, ql) in enumerate(reqs):
            self.arr[i] = SegmentReq(int(seq), int(kvh), int(cls), int(W), int(ns), int(qs), int(ql), 0)


def segpa_build_segments(cache: int, layer: int, reqs, stream=None) -> int:
    """reqs: a SegmentBatch, or the list of tuples SegmentBatch takes."""
    if not isinstance(reqs, SegmentBatch):
        reqs = SegmentBatch(reqs)
    out = C.c_void_p()
    _check(lib().segpa_build_segments(cache, layer, reqs.arr, reqs.n, C.byref(out), _stream_ptr(stream)))
    return out.value


def segpa_free_segments(cache: int, segs: int) -> None:
    _check(lib().segpa_free_segments(cache, segs))


def segpa_segments_stats(segs: int) -> dict:
    st = PlanStats()
    _check(lib().segpa_segments_stats(segs, C.byref(st)))
    return {k: getattr(st, k) for k, _ in PlanStats._fields_}


def segpa_segments_items(segs: int) -> List[dict]:
    n = C.c_int32()
    _check(lib().segpa_segments_items(segs, None, 0, C.byref(n)))
    arr = (Item * max(1, n.value))()
    _check(lib().segpa_segments_items(segs, arr, n.value, C.byref(n)))
    return [{k: getattr(arr[i], k) for k, _ in Item._fields_} for i in range(n.value)]


def segpa_segments_pages(segs: int, segment: int):
    first, n = C.c_int32(), C.c_int32()
    _check(lib().segpa_segments_pages(segs, segment, C.byref(first), None, 0, C.byref(n)))
    ids = np.zeros(n.value, dtype=np.int32)
    _check(lib().segpa_segments_pages(segs, segment, C.byref(first), ids.ctypes.data_as(C.c_void_p), n.value,
                                      C.byref(n)))
    return first.value, ids


def segpa_attention_fwd(cache: int, segs: int, q, softmax_scale: float, out, lse=None, stream=None) -> None:
    """q, out: torch bf16 device tensors [T][Hq][D] (row-strided allowed); lse: fp32 [Hq][T] or None."""
    assert q.is_cuda and out.is_cuda and q.dim() == 3 and out.shape == q.shape
    assert q.stride(2) == 1 and q.stride(1) == q.shape[2] and out.stride(2) == 1 and out.stride(1) == out.shape[2]
    T = q.shape[0]
    lp, ls = None, 0
    if lse is not None:
        assert lse.is_cuda and lse.dim() == 2 and lse.stride(1) == 1
        lp, ls = lse.data_ptr(), lse.stride(0)
    _check(lib().segpa_attention_fwd(cache, segs, q.data_ptr(), q.stride(0), softmax_scale, out.data_ptr(),
                                     out.stride(0), lp, ls, T, _stream_ptr(stream)))


def segpa_attention_fwd_host(cache: int, segs: int, q_host, softmax_scale: float, out_host, lse_host=None,
                             stream=None, wait: bool = True) -> None:
    """q_host, out_host: CPU torch bf16 tensors [T][Hq][D] contiguous (pinned for speed); lse_host fp32 [Hq][T].
    wait=False: segpa_attention_fwd_host_async (results complete after segpa_host_wait)."""
    assert (not q_host.is_cuda) and (not out_host.is_cuda) and q_host.is_contiguous() and out_host.is_contiguous()
    T = q_host.shape[0]
    lp = None
    if lse_host is not None:
        assert (not lse_host.is_cuda) and lse_host.is_contiguous()
        lp = lse_host.data_ptr()
    fn = lib().segpa_attention_fwd_host if wait else lib().segpa_attention_fwd_host_async
    _check(fn(cache, segs, q_host.data_ptr(), softmax_scale, out_host.data_ptr(), lp, T, _stream_ptr(stream)))


def segpa_attention_fwd_host_async(cache: int, segs: int, q_host, softmax_scale: float, out_host, lse_host=None, stream=None) -> None:
    segpa_attention_fwd_host(cache, segs, q_host, softmax_scale, out_host, lse_host, stream=stream, wait=False)


def segpa_host_wait(cache: int) -> None:
    _check(lib().segpa_host_wait(cache))


def segpa_merge(cache: int, out_a, lse_a, out_b, lse_b, out, lse, stream=None) -> None:
    """out_*: torch bf16 device tensors [T][Hq][D] with the same row stride; lse_*: fp32 [Hq][T] with the same stride."""
    for t in (out_a, out_b, out):
        assert t.is_cuda and t.dim() == 3 and t.stride(2) == 1 and t.stride(1) == t.shape[2] and t.stride(0) == out.stride(0)
    for t in (lse_a, lse_b, lse):
        assert t.is_cuda and t.dim() == 2 and t.stride(1) == 1 and t.stride(0) == lse.stride(0)
    _check(lib().segpa_merge(cache, out_a.data_ptr(), lse_a.data_ptr(), out_b.data_ptr(), lse_b.data_ptr(), out.data_ptr(),
                             lse.data_ptr(), out.stride(0), lse.stride(0), out.shape[0], _stream_ptr(stream)))


def segpa_segments_mass_layout(segs: int) -> np.ndarray:
    """int64 offsets [n_segments + 1] of the attention-mass / selection arrays."""
    n = C.c_int32()
    _check(lib().segpa_segments_mass_layout(segs, None, 0, C.byref(n)))
    offs = np.zeros(n.value + 1, dtype=np.int64)
    _check(lib().segpa_segments_mass_layout(segs, offs.ctypes.data_as(C.c_void_p), n.value + 1, C.byref(n)))
    return offs


def segpa_attention_mass(cache: int, segs: int, q, softmax_scale: float, lse, mass, stream=None) -> None:
    """q: torch bf16 [T][Hq][D]; lse: fp32 [Hq][T] from segpa_attention_fwd; mass: fp32 device, layout above."""
    assert q.is_cuda and lse.is_cuda and mass.is_cuda and mass.dtype.is_floating_point and mass.is_contiguous()
    assert q.stride(2) == 1 and q.stride(1) == q.shape[2] and lse.stride(1) == 1
    _check(lib().segpa_attention_mass(cache, segs, q.data_ptr(), q.stride(0), softmax_scale, lse.data_ptr(), lse.stride(0),
                                      q.shape[0], mass.data_ptr(), mass.numel(), _stream_ptr(stream)))


def segpa_mass_select(cache: int, segs: int, mass, tau: float, selected, n_selected, stream=None) -> None:
    """selected: torch uint8 device (layout of mass); n_selected: torch int32 device [n_segments]."""
    assert mass.is_cuda and selected.is_cuda and n_selected.is_cuda and selected.numel() >= mass.numel()
    _check(lib().segpa_mass_select(cache, segs, mass.data_ptr(), tau, selected.data_ptr(), n_selected.data_ptr(),
                                   _stream_ptr(stream)))


def segpa_last_launch_count(cache: int) -> int:
    return int(lib().segpa_last_launch_count(cache))


def segpa_destroy(cache: int) -> None:
    _check(lib().segpa_destroy(cache))


def segpa_version() -> int:
    return int(lib().segpa_version())
