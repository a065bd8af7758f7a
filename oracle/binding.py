"""ctypes binding + build step for oracle/segpa_oracle.c (test infrastructure only).

Argument marshalling only; all arithmetic is in the C file, which cites PAPER.md per step.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "segpa_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp; no -ffast-math (summation order is part of the oracle's definition)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Shape(C.Structure):
    _fields_ = [("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("page_size", C.c_int32)]


class _Seg(C.Structure):
    _fields_ = [("stream", C.c_int32), ("kv_head", C.c_int32), ("head_class", C.c_int32),
                ("window", C.c_int32), ("n_sink", C.c_int32), ("q_len", C.c_int32),
                ("q_row_start", C.c_int64)]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.oracle_attention.restype = C.c_int
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(C.c_int(n))


@dataclass
class OracleResult:
    out: np.ndarray            # float64 [rows][Hq][D]  (NaN where no segment covers (row, head))
    lse: np.ndarray            # float64 [Hq][rows]
    pairs: int                 # attended (query, key) pairs summed over q heads
    p: Optional[np.ndarray]    # float64 [rows][Hq][p_stride] or None
    rows: Optional[np.ndarray]  # the row subset, or None for all rows


def _u16(a) -> np.ndarray:
    """bf16 bits as a C-contiguous uint16 array (accepts torch bf16 tensors or uint16 arrays)."""
    if hasattr(a, "dtype") and str(a.dtype) == "torch.bfloat16":
        import torch
        a = a.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def oracle_attention(*, Hq: int, Hkv: int, D: int, P: int, k_pool, v_pool,
                     page_table: np.ndarray, pt_offsets: np.ndarray, kv_lens: np.ndarray,
                     segments: Sequence[tuple], q, T: int, scale: float,
                     row_subset: Optional[np.ndarray] = None, want_p: int = 0,
                     seg_offsets: Optional[np.ndarray] = None, seg_lens: Optional[np.ndarray] = None) -> OracleResult:
    """segments: tuples (stream_idx, kv_head, head_class, window, n_sink, q_row_start, q_len).
    seg_offsets / seg_lens: optional head-segment table (CSR over streams): each segment of a stream
    starts on a fresh page of the stream's page table.

    k_pool/v_pool: [num_pages][P][D] bf16 (torch) or uint16 bits; q: [T][Hq][D] likewise.
    """
    lib = _load()
    kp, vp, qq = _u16(k_pool), _u16(v_pool), _u16(q)
    num_pages = kp.shape[0]
    assert kp.shape == (num_pages, P, D) and vp.shape == kp.shape, (kp.shape, vp.shape)
    assert qq.shape == (T, Hq, D), (qq.shape, (T, Hq, D))
    page_table = np.ascontiguousarray(page_table, dtype=np.int32)
    pt_offsets = np.ascontiguousarray(pt_offsets, dtype=np.int64)
    kv_lens = np.ascontiguousarray(kv_lens, dtype=np.int64)
    segs = (_Seg * max(1, len(segments)))()
    for i, (st, kvh, cls, W, ns, qs, ql) in enumerate(segments):
        segs[i] = _Seg(int(st), int(kvh), int(cls), int(W), int(ns), int(ql), int(qs))
    if row_subset is not None:
        row_subset = np.ascontiguousarray(np.unique(np.asarray(row_subset, dtype=np.int64)))
        rows = len(row_subset)
        sub_ptr = row_subset.ctypes.data_as(C.c_void_p)
    else:
        rows = T
        sub_ptr = None
    out = np.full((rows, Hq, D), np.nan, dtype=np.float64)
    lse = np.full((Hq, rows), np.nan, dtype=np.float64)
    p = np.zeros((rows, Hq, want_p), dtype=np.float64) if want_p else None
    pairs = C.c_int64(0)
    shape = _Shape(Hq, Hkv, D, P)
    so_ptr = sl_ptr = None
    if seg_offsets is not None:
        seg_offsets = np.ascontiguousarray(seg_offsets, dtype=np.int64)
        seg_lens = np.ascontiguousarray(seg_lens, dtype=np.int64)
        assert len(seg_offsets) == len(kv_lens) + 1 and seg_offsets[-1] == len(seg_lens)
        so_ptr, sl_ptr = seg_offsets.ctypes.data_as(C.c_void_p), seg_lens.ctypes.data_as(C.c_void_p)
    rc = lib.oracle_attention(
        C.byref(shape), kp.ctypes.data_as(C.c_void_p), vp.ctypes.data_as(C.c_void_p),
        C.c_int64(num_pages), page_table.ctypes.data_as(C.c_void_p),
        pt_offsets.ctypes.data_as(C.c_void_p), kv_lens.ctypes.data_as(C.c_void_p),
        C.c_int32(len(kv_lens)), segs, C.c_int32(len(segments)),
        qq.ctypes.data_as(C.c_void_p), C.c_int64(Hq * D), C.c_int64(T), C.c_float(scale),
        sub_ptr, C.c_int64(rows if row_subset is not None else 0),
        out.ctypes.data_as(C.c_void_p), lse.ctypes.data_as(C.c_void_p),
        p.ctypes.data_as(C.c_void_p) if p is not None else None, C.c_int64(want_p),
        C.byref(pairs), so_ptr, sl_ptr)
    if rc != 0:
        raise ValueError("oracle_attention rejected the input (code %d)" % rc)
    return OracleResult(out, lse, int(pairs.value), p, row_subset)
