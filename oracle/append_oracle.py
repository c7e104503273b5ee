"""Fused KV-append (+RoPE) before decode -- numpy oracle on top of pkv_oracle.attention.
TEST INFRASTRUCTURE, NOT THE PRODUCT (shares no code with the CUDA path).

PAPER.md:271 lists "fused RoPE/KV-cache writes" as future work and defines nothing; SURVEY.md
sec. 8(f) f4 asks for "fused KV-append (+RoPE) before decode".  Reading A29:

  * seq_lens[i] = N_i already counts the new token; its position is N_i - 1; rows with N_i = 0 append
    nothing.
  * RoPE in the rotate-half ("NeoX" / Llama) pairing: channel c < d/2 pairs with c + d/2,
        y[c]       = x[c] * cos[pos, c] - x[c + d/2] * sin[pos, c]
        y[c + d/2] = x[c + d/2] * cos[pos, c] + x[c] * sin[pos, c]
    with caller-supplied FP32 tables cos, sin [positions, d/2] (the usual cos_sin cache of a serving
    engine: inputs, so neither side evaluates a transcendental).  The rotation is evaluated in FP32,
    each product and the sum rounded separately (no fused multiply-add), and the result is rounded
    to FP16 -- the precision the kernel takes that decision in, so the bytes written to the cache
    are compared exactly.  No tables = no rotation.
  * the step:  q'_i = RoPE(q_i, N_i - 1);  k' = RoPE(k_new_i, N_i - 1), v' = v_new_i are written to
    the cache slot of token N_i - 1 (page block_table[i][(N_i-1) / P], slot (N_i-1) % P, every KV
    head);  out = Eq. (1) of PAPER.md:39 for q' over tokens 0 .. N_i - 1 of the updated cache.

Pins (tests/test_oracle_pins.py): the rotation against complex multiplication in FP64, pair norms,
position 0 / no tables = identity, the relative-position property of RoPE scores, and the step
against dense brute force on a gathered copy that never touches the cache-update code.
"""
from __future__ import annotations

from typing import Optional, Tuple

import numpy as np

from . import pkv_oracle


def rope_rotate_f16(x: np.ndarray, cos_row: np.ndarray, sin_row: np.ndarray) -> np.ndarray:
    """x [..., d] float16, cos_row / sin_row [d/2] float32 -> float16, FP32 arithmetic, op by op."""
    h = x.shape[-1] // 2
    x32 = x.astype(np.float32)
    x1, x2 = x32[..., :h], x32[..., h:]
    c, s = cos_row.astype(np.float32), sin_row.astype(np.float32)
    y1 = (x1 * c).astype(np.float32) - (x2 * s).astype(np.float32)
    y2 = (x2 * c).astype(np.float32) + (x1 * s).astype(np.float32)
    return np.concatenate([y1, y2], axis=-1).astype(np.float16)


def append_and_attend(q: np.ndarray, k_cache: np.ndarray, v_cache: np.ndarray, k_new: np.ndarray, v_new: np.ndarray,
                      block_table: np.ndarray, seq_lens: np.ndarray, cos: Optional[np.ndarray], sin: Optional[np.ndarray],
                      *, Hkv: int, page_size: int, scale: float) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]:
    """One fused step (reading A29).  Caches in the default layout [pages, P, Hkv, d] float16.
    Returns (out [B,Hq,d] f64, lse [B,Hq] f64, k_cache', v_cache')."""
    B, Hq, d = q.shape
    k2, v2, q2 = k_cache.copy(), v_cache.copy(), q.copy()
    for i in range(B):
        N = int(seq_lens[i])
        if N <= 0:
            continue
        pos = N - 1
        kn, qn = k_new[i], q[i]
        if cos is not None:
            kn = rope_rotate_f16(kn, cos[pos], sin[pos])
            qn = rope_rotate_f16(qn, cos[pos], sin[pos])
        page, slot = int(block_table[i, pos // page_size]), pos % page_size
        k2[page, slot] = kn
        v2[page, slot] = v_new[i]
        q2[i] = qn
    out, lse = pkv_oracle.attention(q2, k2, v2, block_table, seq_lens, Hkv=Hkv, page_size=page_size, scale=scale)
    return out, lse, k2, v2
