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

One-byte caches (reading A30; the caches of reading A28): the new token is rotated as
above (FP16 result), then each element is divided by its KV head's scale in FP32 and rounded ONCE to
the cache's code -- E4M3: the nearest finite E4M3 value, ties to the even code, magnitudes beyond 448
saturate to +-448 (the OCP "satfinite" conversion); INT8: round half to even, clamped to [-127, 127].
The code byte is what the cache receives and what the step attends over (k = k_scale * dec(code)).
The division is the decision's precision: both sides take it in FP32, so cache bytes compare exactly.
Pins: every finite E4M3 code survives decode -> encode; ties, saturation and subnormals in closed
form; torch.float8_e4m3fn on the whole FP16 grid inside +-448; the INT8 ties and clamp.
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


# ---------------------------------------------------------------- one-byte caches (reading A30)

def _e4m3_table() -> np.ndarray:
    """The 127 non-negative finite E4M3 values by code 0x00..0x7E (OCP FP8: bias 7, no infinity,
    0x7F = NaN), from the oracle's own decoder (pinned on all 256 codes)."""
    return np.array([pkv_oracle.e4m3_to_double(c) for c in range(0x7F)], dtype=np.float64)


def quantize_e4m3(x: np.ndarray) -> np.ndarray:
    """float32 -> E4M3 code bytes: nearest finite value, ties to the even code, |x| > 448 -> +-448,
    NaN -> 0x7F.  Written as the definition: the two neighbouring table values are compared in FP64
    (exact for FP32 inputs), no bit tricks."""
    x = np.asarray(x, dtype=np.float32)
    tab = _e4m3_table()                      # increasing with the code
    mag = np.abs(x.astype(np.float64))
    hi = np.searchsorted(tab, mag, side="left")            # first code with value >= |x|
    hi = np.minimum(hi, len(tab) - 1)
    lo = np.maximum(hi - 1, 0)
    d_lo, d_hi = mag - tab[lo], tab[hi] - mag
    pick_hi = (d_hi < d_lo) | ((d_hi == d_lo) & (hi % 2 == 0))
    code = np.where(pick_hi, hi, lo)
    code = np.where(mag >= tab[-1], len(tab) - 1, code)     # saturate (also the values that would round past 448)
    code = code.astype(np.uint8) | np.where(np.signbit(x), 0x80, 0).astype(np.uint8)
    return np.where(np.isnan(x), np.uint8(0x7F), code).astype(np.uint8)


def quantize_int8(x: np.ndarray) -> np.ndarray:
    """float32 -> two's-complement INT8 bytes (as uint8): round half to even, clamp to [-127, 127]."""
    x = np.asarray(x, dtype=np.float32)
    r = np.clip(np.rint(x.astype(np.float64)), -127.0, 127.0)
    return r.astype(np.int8).view(np.uint8)


def quantize_token(x16: np.ndarray, head_scale: np.ndarray, kv_kind: int) -> np.ndarray:
    """x16 [Hkv, d] float16, head_scale [Hkv] float32 -> code bytes [Hkv, d]: FP32 division, one rounding."""
    y = (x16.astype(np.float32) / head_scale.astype(np.float32)[:, None]).astype(np.float32)
    return quantize_int8(y) if kv_kind == 2 else quantize_e4m3(y)


def append_and_attend_q8(q: np.ndarray, k8: np.ndarray, v8: np.ndarray, k_scale: np.ndarray, v_scale: np.ndarray,
                         k_new: np.ndarray, v_new: np.ndarray, block_table: np.ndarray, seq_lens: np.ndarray,
                         cos: Optional[np.ndarray], sin: Optional[np.ndarray], *, Hkv: int, page_size: int, scale: float,
                         kv_kind: int = 1) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]:
    """One fused step on one-byte caches [pages, P, Hkv, d] uint8 (reading A30; kv_kind 1 = E4M3,
    2 = INT8); k_scale, v_scale [Hkv] float32 (None = 1).  Returns (out, lse, k8', v8')."""
    B, Hq, d = q.shape
    ks = np.ones(Hkv, dtype=np.float32) if k_scale is None else np.asarray(k_scale, dtype=np.float32)
    vs = np.ones(Hkv, dtype=np.float32) if v_scale is None else np.asarray(v_scale, dtype=np.float32)
    k2, v2, q2 = k8.copy(), v8.copy(), q.copy()
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
        k2[page, slot] = quantize_token(kn, ks, kv_kind)
        v2[page, slot] = quantize_token(v_new[i], vs, kv_kind)
        q2[i] = qn
    out, lse = pkv_oracle.attention_fp8(q2, k2, v2, ks, vs, block_table, seq_lens, Hkv=Hkv, page_size=page_size,
                                        scale=scale, kv_kind=kv_kind)
    return out, lse, k2, v2
