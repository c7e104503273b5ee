"""Shared test helpers: small problem construction and an independent numpy brute force.

The brute force here (dense gather in Python + softmax(q K^T * scale) V in numpy FP64) is the
third, independent statement of PAPER.md:39 Eq. (1) used to pin the C oracle (pin P1).  It
calls neither oracle/ nor the CUDA path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

import pkv_inputs
from pkv_inputs import PAD_PAGE


def default_scale(d: int) -> float:
    """1/sqrt(d) rounded to FP32 first, so the oracle and the kernel multiply by the identical
    number (reading A4)."""
    return float(np.float32(1.0 / math.sqrt(d)))


@dataclass
class Problem:
    q: np.ndarray            # [B,Hq,d] f16
    k_cache: np.ndarray      # [num_pages,P,Hkv,d] f16
    v_cache: np.ndarray
    block_table: np.ndarray  # [B,max_pages] i32
    seq_lens: np.ndarray     # [B] i32
    Hkv: int
    page_size: int
    scale: float

    @property
    def B(self):
        return self.q.shape[0]

    @property
    def Hq(self):
        return self.q.shape[1]

    @property
    def d(self):
        return self.q.shape[2]

    @property
    def G(self):
        return self.Hq // self.Hkv


def make_problem(seq_lens: Sequence[int], *, seed: int, Hq: int = 32, Hkv: int = 8, d: int = 128,
                 page_size: int = 16, hole_frac: float = 0.5, reserve_extra: int = 0,
                 max_pages: Optional[int] = None) -> Problem:
    """Random problem in the default [num_pages, P, Hkv, d] layout; whole pool filled."""
    rng = np.random.Generator(np.random.PCG64(seed))
    lens = np.asarray(seq_lens, dtype=np.int32)
    reserved = np.maximum(lens.astype(np.int64) + reserve_extra, 1)
    table, universe = pkv_inputs.make_page_table(reserved, page_size, hole_frac, rng, max_pages=max_pages)
    # rows with N=0 still got one reserved page above; keep the table entry (it is never read)
    B = len(lens)
    q = pkv_inputs.fill_normal_f16((B, Hq, d), seed * 7 + 1)
    k = pkv_inputs.fill_normal_f16((universe, page_size, Hkv, d), seed * 7 + 2)
    v = pkv_inputs.fill_normal_f16((universe, page_size, Hkv, d), seed * 7 + 3)
    return Problem(q=q, k_cache=k, v_cache=v, block_table=table, seq_lens=lens, Hkv=Hkv,
                   page_size=page_size, scale=default_scale(d))


def gather_dense(p: Problem, cache: np.ndarray, i: int) -> np.ndarray:
    """[N_i, Hkv, d] f64 copy of row i's tokens, gathered page by page in Python."""
    N = int(p.seq_lens[i])
    out = np.zeros((N, p.Hkv, p.d), dtype=np.float64)
    for j in range(N):
        page = int(p.block_table[i, j // p.page_size])
        assert page != PAD_PAGE
        out[j] = cache[page, j % p.page_size].astype(np.float64)
    return out


def dense_attention_bruteforce(p: Problem):
    """softmax(q K^T * scale) V per query head in numpy FP64 on a dense gathered copy."""
    B, Hq, d = p.q.shape
    out = np.zeros((B, Hq, d), dtype=np.float64)
    lse = np.full((B, Hq), -np.inf, dtype=np.float64)
    for i in range(B):
        N = int(p.seq_lens[i])
        if N == 0:
            continue
        Kd = gather_dense(p, p.k_cache, i)
        Vd = gather_dense(p, p.v_cache, i)
        for h in range(Hq):
            g = h // p.G
            x = (Kd[:, g, :] @ p.q[i, h].astype(np.float64)) * p.scale
            m = x.max()
            w = np.exp(x - m)
            out[i, h] = (w[:, None] * Vd[:, g, :]).sum(axis=0) / w.sum()
            lse[i, h] = m + np.log(w.sum())
    return out, lse


def permute_pool(p: Problem, seed: int) -> Problem:
    """Physically permute the page pool and map the table through the permutation (pin P2)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = p.k_cache.shape[0]
    perm = rng.permutation(n)            # new_pool[perm[a]] = old_pool[a]
    k2 = np.empty_like(p.k_cache)
    v2 = np.empty_like(p.v_cache)
    k2[perm] = p.k_cache
    v2[perm] = p.v_cache
    t2 = p.block_table.copy()
    mask = t2 != PAD_PAGE
    t2[mask] = perm[t2[mask]].astype(np.int32)
    return Problem(q=p.q, k_cache=k2, v_cache=v2, block_table=t2, seq_lens=p.seq_lens, Hkv=p.Hkv,
                   page_size=p.page_size, scale=p.scale)


def token_location(p: Problem, i: int, j: int):
    return int(p.block_table[i, j // p.page_size]), j % p.page_size


def error_metrics(got: np.ndarray, ref: np.ndarray):
    """Reading A15: max abs error, and max relative error with the per-(row, head)
    floor tau = 2^-4 * max_c |ref[row, head, c]| so FP16 subnormal-sized outputs do not decide it."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    err = np.abs(got - ref)
    tau = np.abs(ref).max(axis=-1, keepdims=True) / 16.0
    denom = np.maximum(np.abs(ref), np.maximum(tau, 1e-30))
    return {"max_abs": float(err.max()) if err.size else 0.0,
            "mean_abs": float(err.mean()) if err.size else 0.0,
            "max_rel_floored": float((err / denom).max()) if err.size else 0.0}


MAX_ABS_TOL = 2e-3      # BASELINE.json north_star
MAX_REL_TOL = 1e-2      # BASELINE.json north_star (with the A15 floor)
MEAN_ABS_TOL = 3e-4


def assert_within_tolerance(got, ref, what=""):
    m = error_metrics(got, ref)
    assert m["max_abs"] <= MAX_ABS_TOL, (what, m)
    assert m["max_rel_floored"] <= MAX_REL_TOL, (what, m)
    assert m["mean_abs"] <= MEAN_ABS_TOL, (what, m)
    return m
