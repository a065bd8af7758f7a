"""Brute-force dense masked softmax attention (tiny inputs only) -- TEST INFRASTRUCTURE ONLY.

An independent second opinion used to pin oracle/segpa_oracle.c: it first gathers each stream
into a dense [kv_len][D] array, builds an explicit boolean [q_len][kv_len] mask (the "dense +
mask" formulation the paper replaces), and applies softmax(mask ? s : -inf).
The visibility rule is written a different way from the oracle's:
    j <= i  and  (global  or  i - j < W  or  j < n_sink)         PAPER.md:219 (W = w + 1)
Shares no code with the oracle's C file or with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def widen(bits: np.ndarray) -> np.ndarray:
    """bf16 bit patterns (uint16) -> float64, exactly."""
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def dense_masked_attention(q_bits, k_pool_bits, v_pool_bits, page_ids, kv_len, P,
                           head_class, W, n_sink, scale, chunk_lens=None):
    """q_bits [q_len][D] of ONE q head; returns (O [q_len][D], LSE [q_len], p [q_len][kv_len]).
    chunk_lens: the stream's head segments, each on its own consecutive pages of page_ids; the dense
    stream is the concatenation of the segments' rows (None: one segment)."""
    q = widen(np.asarray(q_bits))
    q_len = q.shape[0]
    Kp, Vp = [], []
    first = 0
    for n in ([kv_len] if chunk_lens is None else list(chunk_lens)):
        npg = (n + P - 1) // P
        pages = np.asarray(page_ids)[first:first + npg]
        Kp.append(widen(np.asarray(k_pool_bits)[pages]).reshape(-1, q.shape[1])[:n])
        Vp.append(widen(np.asarray(v_pool_bits)[pages]).reshape(-1, q.shape[1])[:n])
        first += npg
    K, V = np.concatenate(Kp), np.concatenate(Vp)
    assert K.shape[0] == kv_len
    S = np.float64(np.float32(scale)) * (q @ K.T)
    i = (kv_len - q_len + np.arange(q_len))[:, None]
    j = np.arange(kv_len)[None, :]
    mask = j <= i
    if head_class != 0:
        mask &= ((i - j) < W) | (j < n_sink)
    S = np.where(mask, S, -np.inf)
    m = S.max(axis=1, keepdims=True)
    e = np.exp(S - m)
    l = e.sum(axis=1, keepdims=True)
    p = e / l
    return p @ V, (m + np.log(l))[:, 0], p
