"""rope_oracle.py -- plain fp64 statement of RoPE-based positional alignment.

TEST INFRASTRUCTURE ONLY (same rules as segpa_oracle.c): only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline leg may call it; it shares nothing with the CUDA path.

What it computes (the definition, written out): for a key cached at offline position p_off and reused at
online position p_on,
    K(p_on) = R(p_on) R(p_off)^-1 K(p_off)
where R(p) is the RoPE rotation matrix: block-diagonal 2x2 rotations, pair d in [0, D/2) rotated by the
angle p * theta_d, theta_d = base^(-2d/D).  R(p_on) and R(p_off)^-1 are applied one after the other exactly as
the formula states (no use of R(a)R(b) = R(a+b): that identity is one of the pins).
Pairing (paper silent; reading A20): elements (d, d + D/2) form pair d -- the "rotate-half" layout of
the Llama / Qwen / Mistral families the paper evaluates.

Pins (tests/test_oracle_pins.py): delta = 0 is the identity; R(a) R(b) = R(a + b); pair norms are preserved;
<R(m) q, K(p_on)> = <R(m - p_on + p_off) q, K(p_off)> (relative-position property of RoPE);
agreement with complex multiplication by e^{i p theta} (a numpy primitive); D = 2 printed constants
(cos 1, sin 1).
"""
from __future__ import annotations

import numpy as np


def rope_rotate(x: np.ndarray, pos: np.ndarray, base: float = 10000.0, inverse: bool = False) -> np.ndarray:
    """R(pos) x (or R(pos)^-1 x) for rows x [n][D] (fp64), pos [n] integer positions."""
    x = np.asarray(x, dtype=np.float64)
    n, D = x.shape
    half = D // 2
    out = np.empty_like(x)
    for d in range(half):
        theta = float(base) ** (-2.0 * d / D)
        ang = np.asarray(pos, dtype=np.float64) * theta
        c, s = np.cos(ang), np.sin(ang)
        if inverse:
            s = -s
        a, b = x[:, d], x[:, d + half]
        out[:, d] = a * c - b * s
        out[:, d + half] = a * s + b * c
    return out


def rope_align(k_off: np.ndarray, p_off: np.ndarray, p_on: np.ndarray, base: float = 10000.0) -> np.ndarray:
    """K(p_on) = R(p_on) R(p_off)^-1 K(p_off), applied literally in that order."""
    return rope_rotate(rope_rotate(k_off, p_off, base, inverse=True), p_on, base)
