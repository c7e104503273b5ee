"""ctypes front end of ``pkv_oracle.c`` -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Compiles the C file with gcc on first use (``build()``), then exposes numpy-in / numpy-out
functions.  See the C file's header for what each entry point computes and the passages of
PAPER.md it follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pkv_oracle.c")
_SO = os.path.join(_HERE, "libpkv_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared.  -ffast-math is deliberately absent (FP64, IEEE semantics)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        i32, i64, f64 = ctypes.c_int, ctypes.c_int64, ctypes.c_double
        vp = ctypes.c_void_p
        lib.pkv_oracle_attention.argtypes = [i32] * 6 + [i64] * 3 + [vp] * 5 + [f64, vp, vp, i32]
        lib.pkv_oracle_attention.restype = i32
        lib.pkv_oracle_split_states.argtypes = ([i32] * 6 + [i64] * 3 + [vp] * 5 + [f64, vp, i32, i32]
                                                + [vp] * 3 + [i32])
        lib.pkv_oracle_split_states.restype = i32
        lib.pkv_oracle_merge.argtypes = [i32, i32, vp, vp, vp, vp, vp]
        lib.pkv_oracle_merge.restype = i32
        lib.pkv_oracle_max_threads.restype = i32
        lib.pkv_oracle_half_to_double.argtypes = [ctypes.c_uint16]
        lib.pkv_oracle_half_to_double.restype = f64
        lib.pkv_oracle_e4m3_to_double.argtypes = [ctypes.c_uint8]
        lib.pkv_oracle_e4m3_to_double.restype = f64
        lib.pkv_oracle_attention_q8.argtypes = [i32] * 6 + [i64] * 3 + [vp] * 5 + [i32, vp, vp, f64, vp, vp, i32]
        lib.pkv_oracle_attention_q8.restype = i32
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().pkv_oracle_max_threads())


def half_to_double(bits: int) -> float:
    return float(_load().pkv_oracle_half_to_double(int(bits) & 0xFFFF))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _default_strides(page_size: int, Hkv: int, d: int) -> Tuple[int, int, int]:
    """[num_pages, page_size, Hkv, d] (BASELINE.json north_star layout; reading A1)."""
    return page_size * Hkv * d, Hkv * d, d


def _check_inputs(q, k_cache, v_cache, block_table, seq_lens):
    assert q.dtype == np.float16 and k_cache.dtype == np.float16 and v_cache.dtype == np.float16
    assert block_table.dtype == np.int32 and seq_lens.dtype == np.int32
    for a in (q, k_cache, v_cache, block_table, seq_lens):
        assert a.flags["C_CONTIGUOUS"]


def attention(q: np.ndarray, k_cache: np.ndarray, v_cache: np.ndarray, block_table: np.ndarray,
              seq_lens: np.ndarray, *, Hkv: int, page_size: int, scale: float,
              strides: Optional[Tuple[int, int, int]] = None, num_threads: int = 0):
    """Eq. (1) of PAPER.md:39.  q [B,Hq,d] f16; caches: f16 buffers addressed through
    ``strides`` = (page, token, head) in elements (default: [num_pages, page_size, Hkv, d]);
    block_table [B,max_pages] i32; seq_lens [B] i32.  Returns (out [B,Hq,d] f64, lse [B,Hq] f64)."""
    _check_inputs(q, k_cache, v_cache, block_table, seq_lens)
    B, Hq, d = q.shape
    sp, st, sh = strides or _default_strides(page_size, Hkv, d)
    out = np.empty((B, Hq, d), dtype=np.float64)
    lse = np.empty((B, Hq), dtype=np.float64)
    rc = _load().pkv_oracle_attention(B, Hq, Hkv, d, page_size, block_table.shape[1], sp, st, sh,
                                      _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table),
                                      _ptr(seq_lens), float(scale), _ptr(out), _ptr(lse), num_threads)
    if rc != 0:
        raise RuntimeError("pkv_oracle_attention failed: %d" % rc)
    return out, lse


def e4m3_to_double(bits: int) -> float:
    return float(_load().pkv_oracle_e4m3_to_double(int(bits) & 0xFF))


def attention_int8(q, k8, v8, k_scale, v_scale, block_table, seq_lens, **kw):
    """Eq. (1) on INT8 caches (reading A28): k8, v8 uint8 views of two's-complement bytes."""
    return attention_fp8(q, k8, v8, k_scale, v_scale, block_table, seq_lens, kv_kind=2, **kw)


def attention_fp8(q: np.ndarray, k8: np.ndarray, v8: np.ndarray, k_scale: np.ndarray, v_scale: np.ndarray,
                  block_table: np.ndarray, seq_lens: np.ndarray, *, Hkv: int, page_size: int, scale: float,
                  strides: Optional[Tuple[int, int, int]] = None, num_threads: int = 0, kv_kind: int = 1):
    """Eq. (1) on one-byte caches (reading A28): k8, v8 uint8 bytes (E4M3, or INT8 with kv_kind=2),
    k_scale, v_scale [Hkv] (any float dtype; used as FP64).  Returns (out [B,Hq,d] f64, lse [B,Hq] f64)."""
    assert q.dtype == np.float16 and k8.dtype == np.uint8 and v8.dtype == np.uint8
    assert block_table.dtype == np.int32 and seq_lens.dtype == np.int32
    ks = np.ascontiguousarray(k_scale, dtype=np.float64)
    vs = np.ascontiguousarray(v_scale, dtype=np.float64)
    assert ks.shape == (Hkv,) and vs.shape == (Hkv,)
    for a in (q, k8, v8, block_table, seq_lens):
        assert a.flags["C_CONTIGUOUS"]
    B, Hq, d = q.shape
    sp, st, sh = strides or _default_strides(page_size, Hkv, d)
    out = np.empty((B, Hq, d), dtype=np.float64)
    lse = np.empty((B, Hq), dtype=np.float64)
    rc = _load().pkv_oracle_attention_q8(B, Hq, Hkv, d, page_size, block_table.shape[1], sp, st, sh,
                                         _ptr(q), _ptr(k8), _ptr(v8), _ptr(ks), _ptr(vs), int(kv_kind), _ptr(block_table),
                                         _ptr(seq_lens), float(scale), _ptr(out), _ptr(lse), num_threads)
    if rc != 0:
        raise RuntimeError("pkv_oracle_attention_q8 failed: %d" % rc)
    return out, lse


def split_states(q, k_cache, v_cache, block_table, seq_lens, tasks: np.ndarray, *, Hkv: int,
                 page_size: int, tile_tokens: int, scale: float,
                 strides: Optional[Tuple[int, int, int]] = None, num_threads: int = 0):
    """PAPER.md:56 per task.  tasks [num_tasks,5] i32 = (row, kvh, split, t_begin, t_end).
    Returns (m [T,G], l [T,G], a [T,G,d]) in f64."""
    _check_inputs(q, k_cache, v_cache, block_table, seq_lens)
    tasks = np.ascontiguousarray(tasks, dtype=np.int32).reshape(-1, 5)
    B, Hq, d = q.shape
    G = Hq // Hkv
    T = tasks.shape[0]
    sp, st, sh = strides or _default_strides(page_size, Hkv, d)
    m = np.empty((T, G), dtype=np.float64)
    l = np.empty((T, G), dtype=np.float64)
    a = np.empty((T, G, d), dtype=np.float64)
    rc = _load().pkv_oracle_split_states(B, Hq, Hkv, d, page_size, block_table.shape[1], sp, st, sh,
                                         _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table),
                                         _ptr(seq_lens), float(scale), _ptr(tasks), T, tile_tokens,
                                         _ptr(m), _ptr(l), _ptr(a), num_threads)
    if rc != 0:
        raise RuntimeError("pkv_oracle_split_states failed: %d" % rc)
    return m, l, a


def merge(m_s: np.ndarray, l_s: np.ndarray, a_s: np.ndarray):
    """PAPER.md:60-61 for one (row, query head): m_s [n], l_s [n], a_s [n,d] -> (O [d], LSE)."""
    m_s = np.ascontiguousarray(m_s, dtype=np.float64)
    l_s = np.ascontiguousarray(l_s, dtype=np.float64)
    a_s = np.ascontiguousarray(a_s, dtype=np.float64)
    n = m_s.shape[0]
    d = a_s.shape[-1] if a_s.ndim == 2 else 0
    out = np.empty((d,), dtype=np.float64)
    lse = np.empty((1,), dtype=np.float64)
    rc = _load().pkv_oracle_merge(n, d, _ptr(m_s), _ptr(l_s), _ptr(a_s), _ptr(out), _ptr(lse))
    if rc != 0:
        raise RuntimeError("pkv_oracle_merge failed: %d" % rc)
    return out, float(lse[0])


def attention_via_splits(q, k_cache, v_cache, block_table, seq_lens, tasks, split_offsets, *, Hkv,
                         page_size, tile_tokens, scale, strides=None, num_threads: int = 0):
    """Split form end to end: states per task, then the segmented merge over each
    row's compact slot range.  ``tasks`` must be in the canonical order
    (row, kvh, split) so that the tasks of (row i, kvh g) are the contiguous run starting at
    split_offsets[i]*Hkv + g*n_i (reading A8).  Returns (out [B,Hq,d], lse [B,Hq])."""
    tasks = np.ascontiguousarray(tasks, dtype=np.int32).reshape(-1, 5)
    B, Hq, d = q.shape
    G = Hq // Hkv
    m, l, a = split_states(q, k_cache, v_cache, block_table, seq_lens, tasks, Hkv=Hkv,
                           page_size=page_size, tile_tokens=tile_tokens, scale=scale,
                           strides=strides, num_threads=num_threads)
    out = np.zeros((B, Hq, d), dtype=np.float64)
    lse = np.full((B, Hq), -np.inf, dtype=np.float64)
    for i in range(B):
        n_i = int(split_offsets[i + 1] - split_offsets[i])
        for g in range(Hkv):
            base = int(split_offsets[i]) * Hkv + g * n_i
            for hh in range(G):
                o, e = merge(m[base:base + n_i, hh], l[base:base + n_i, hh], a[base:base + n_i, hh, :])
                out[i, g * G + hh] = o
                lse[i, g * G + hh] = e
    return out, lse
