"""Helpers of the -m gpu parity tests: move a host Problem to the device, call the C ABI through
the binding, bring results back.  PyTorch owns memory only."""
from __future__ import annotations

import ctypes

import numpy as np
import torch

import paper_2606_26666_b200 as pkv
from helpers import Problem
from oracle import pkv_oracle, workqueue_oracle as wq


def to_dev(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class DevProblem:
    def __init__(self, p: Problem, kv_strides=(0, 0, 0), k_dev=None, v_dev=None):
        self.p = p
        self.q = to_dev(p.q)
        self.k = to_dev(p.k_cache) if k_dev is None else k_dev
        self.v = to_dev(p.v_cache) if v_dev is None else v_dev
        self.bt = to_dev(p.block_table)
        self.sl = to_dev(p.seq_lens)
        self.shape = pkv.Shape(B=p.B, Hq=p.Hq, Hkv=p.Hkv, d=p.d, page_size=p.page_size,
                               max_pages=p.block_table.shape[1], num_pages=p.k_cache.shape[0],
                               kv_strides=kv_strides)
        self.out = torch.full((p.B, p.Hq, p.d), float("nan"), dtype=torch.float16, device="cuda")
        self.lse = torch.full((p.B, p.Hq), float("nan"), dtype=torch.float32, device="cuda")

    def decode(self, pol: pkv.Policy, ws=None, build_queue=True, scale=None):
        """One pkv_decode call; returns (out f64 [B,Hq,d], lse f64 [B,Hq], workspace)."""
        if ws is None:
            ws = pkv.alloc_workspace(self.shape, pol)
        self.out.fill_(float("nan"))
        self.lse.fill_(float("nan"))
        pkv.pkv_decode(self.shape, pol, self.q, self.k, self.v, self.bt, self.sl, self.out, self.lse,
                       scale=self.p.scale if scale is None else scale, build_queue=build_queue, workspace=ws)
        torch.cuda.synchronize()
        return (self.out.cpu().numpy().astype(np.float64), self.lse.cpu().numpy().astype(np.float64), ws)


def oracle_policy(pol: pkv.Policy) -> wq.Policy:
    """The same policy for the workqueue oracle; num_sms = 0 means the device's SM count."""
    return wq.Policy(tile_tokens=pol.tile_tokens, split_mode=pol.split_mode, num_splits=pol.num_splits,
                     chunk_tiles=pol.chunk_tiles, route=pol.route, merge_mode=pol.merge_mode,
                     num_sms=pol.num_sms if pol.num_sms > 0 else sm_count())


def oracle_attention(p: Problem, **kw):
    return pkv_oracle.attention(p.q, p.k_cache, p.v_cache, p.block_table, p.seq_lens, Hkv=p.Hkv,
                                page_size=p.page_size, scale=p.scale, **kw)


def read_partials(dp: DevProblem, pol: pkv.Policy, ws, slots: int):
    """Copies the first `slots` partial states out of the workspace: (m [slots,G], l, acc [slots,G,d])."""
    pm, pl, pa, cap = pkv.pkv_workspace_partials(dp.shape, pol, ws)
    assert slots <= cap
    G, d = dp.p.G, dp.p.d
    base = ws.data_ptr()

    def view(ptr, n):
        off = ptr - base
        return ws[off:off + 4 * n].view(torch.float32).cpu().numpy().astype(np.float64)

    m = view(pm, slots * G).reshape(slots, G)
    l = view(pl, slots * G).reshape(slots, G)
    a = view(pa, slots * G * d).reshape(slots, G, d)
    return m, l, a


def sm_count() -> int:
    return torch.cuda.get_device_properties(0).multi_processor_count
