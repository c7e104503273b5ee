"""ctypes binding of libpkv.so -- argument marshalling only.

Every function here has the name and the argument order of its C entry point in
``include/pkv.h``; tensors are passed as raw device (or host) pointers taken from
``torch.Tensor.data_ptr()`` / numpy arrays.  No step of the decode path runs in Python or in
PyTorch ops: PyTorch only owns the memory and the stream.  There is no CPU fallback: if
``libpkv.so`` cannot be loaded (or built), importing this module raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np

from . import build as _build

PKV_OK, PKV_ERR_INVALID_ARG, PKV_ERR_UNSUPPORTED, PKV_ERR_WORKSPACE, PKV_ERR_CUDA = range(5)
ROUTE_RECT, ROUTE_WORKQUEUE = 0, 1
MERGE_SEPARATE, MERGE_FUSED = 0, 1
SPLIT_FIXED_COUNT, SPLIT_FIXED_CHUNK, SPLIT_BALANCED, SPLIT_AUTO = 0, 1, 2, 3
KERNEL_AUTO, KERNEL_TMA_MMA, KERNEL_SIMT = 0, 1, 2
FLAG_VALIDATE, FLAG_NO_PDL, FLAG_SEPARATE_BUILD, FLAG_TEST_REPLAN, FLAG_OUT_PINNED = 1, 2, 4, 8, 16
DEVERR_QUEUE_OVERFLOW, DEVERR_SEQ_LEN, DEVERR_PAGE_ID = 1, 2, 4
STAGE_BUILD, STAGE_DECODE, STAGE_MERGE, STAGE_ALL = 1, 2, 4, 7
KV_F16, KV_E4M3, KV_INT8 = 0, 1, 2

_i32, _i64 = ctypes.c_int32, ctypes.c_int64
_vp = ctypes.c_void_p


class pkv_split_policy(ctypes.Structure):
    _fields_ = [("tile_tokens", _i32), ("split_mode", _i32), ("num_splits", _i32), ("chunk_tiles", _i32),
                ("route", _i32), ("merge_mode", _i32), ("num_sms", _i32), ("kernel", _i32), ("flags", _i32),
                ("heads_per_cta", _i32), ("prefetch_kb", _i32)]


class pkv_task(ctypes.Structure):
    _fields_ = [("row", _i32), ("kvh", _i32), ("split", _i32), ("t_begin", _i32), ("t_end", _i32)]


class pkv_shape(ctypes.Structure):
    _fields_ = [("B", _i32), ("Hq", _i32), ("Hkv", _i32), ("d", _i32), ("page_size", _i32), ("max_pages", _i32),
                ("num_pages", _i64), ("kv_stride_page", _i64), ("kv_stride_token", _i64), ("kv_stride_head", _i64),
                ("kv_dtype", _i32), ("reserved_", _i32), ("k_scale", _vp), ("v_scale", _vp)]


class pkv_counters(ctypes.Structure):
    _fields_ = [(n, _i64) for n in ("tasks", "empty_tasks", "decode_launches", "merge_launches", "build_launches",
                                    "useful_kv_bytes", "merge_bytes", "num_splits", "max_row_splits", "chunk_tiles", "h2d_bytes",
                                    "d2h_bytes", "launched_build", "launched_decode", "launched_merge", "error_word", "armed_step")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class pkv_calibration(ctypes.Structure):
    _fields_ = ([(n, ctypes.c_double) for n in ("read_gbps", "read_ldg_gbps", "read_bulk8k_gbps", "read_bulk16k_gbps",
                                                 "launch_us", "launch_pdl_us", "graph_launch_us", "graph_launch_pdl_us")]
                + [("buffer_bytes", _i64), ("num_sms", _i32), ("l2_bytes", _i32)])

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class pkv_cost_model(ctypes.Structure):
    _fields_ = [("beta_gbps", ctypes.c_double), ("lambda_us", ctypes.c_double), ("c_min", ctypes.c_double),
                ("num_sms", _i32), ("reserved_", _i32)]


class pkv_cost_estimate(ctypes.Structure):
    _fields_ = ([(n, ctypes.c_double) for n in ("total_us", "stream_us", "launch_us", "merge_us", "cta_work_per_sm",
                                                 "makespan_us", "makespan_total_us")]
                + [(n, _i64) for n in ("kv_bytes", "merge_bytes", "tasks", "launches", "max_share_bytes", "units")])

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class pkv_append(ctypes.Structure):
    _fields_ = [("k_new", _vp), ("v_new", _vp), ("rope_cos", _vp), ("rope_sin", _vp), ("rope_positions", _i32), ("reserved_", _i32)]


# every symbol include/pkv.h declares (tests/test_abi.py checks the header against this list)
EXPORTS = ("pkv_version", "pkv_last_error", "pkv_workspace_bytes", "pkv_workspace_init_bytes", "pkv_build_workqueue_host",
           "pkv_build_workqueue", "pkv_decode", "pkv_decode_stages", "pkv_merge", "pkv_get_counters", "pkv_read_workqueue",
           "pkv_workspace_partials", "pkv_host_scratch_bytes", "pkv_decode_host", "pkv_calibrate", "pkv_decode_indexed",
           "pkv_plan_buckets_host", "pkv_decode_buckets", "pkv_bucket_counters_host", "pkv_default_cost_model",
           "pkv_estimate_cost", "pkv_choose_policy", "pkv_decode_append", "pkv_decode_static",
           "pkv_static_workspace_bytes", "pkv_decode_host_pipelined", "pkv_decode_host_drain")


class pkv_next_step(ctypes.Structure):
    _fields_ = [("seq_lens_host", _vp), ("block_table_host", _vp), ("k_cache_dev", _vp), ("v_cache_dev", _vp), ("out_host", _vp)]


class PkvError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("pkv status %d: %s" % (status, message))
        self.status = status


def _load() -> ctypes.CDLL:
    path = _build.LIB
    if not os.path.exists(path) or os.path.getmtime(path) < _build._deps_mtime():
        _build.build()           # raises if nvcc is missing: no fallback
    lib = ctypes.CDLL(path)
    P = ctypes.POINTER
    lib.pkv_version.restype = _i32
    lib.pkv_last_error.restype = ctypes.c_char_p
    lib.pkv_workspace_bytes.restype = ctypes.c_size_t
    lib.pkv_workspace_bytes.argtypes = [P(pkv_shape), P(pkv_split_policy)]
    lib.pkv_workspace_init_bytes.restype = ctypes.c_size_t
    lib.pkv_workspace_init_bytes.argtypes = [P(pkv_shape), P(pkv_split_policy)]
    lib.pkv_host_scratch_bytes.restype = ctypes.c_size_t
    lib.pkv_host_scratch_bytes.argtypes = [P(pkv_shape), P(pkv_split_policy)]
    lib.pkv_build_workqueue_host.restype = _i32
    lib.pkv_build_workqueue_host.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _i32, _vp, P(_i32)]
    lib.pkv_build_workqueue.restype = _i32
    lib.pkv_build_workqueue.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, ctypes.c_size_t, _vp]
    lib.pkv_decode.restype = _i32
    lib.pkv_decode.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_float,
                               _i32, _vp, ctypes.c_size_t, _vp]
    lib.pkv_decode_stages.restype = _i32
    lib.pkv_decode_stages.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, _vp,
                                      ctypes.c_float, ctypes.c_uint32, _vp, ctypes.c_size_t, _vp]
    lib.pkv_static_workspace_bytes.restype = ctypes.c_size_t
    lib.pkv_static_workspace_bytes.argtypes = []
    lib.pkv_decode_static.restype = _i32
    lib.pkv_decode_static.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_float, _vp]
    lib.pkv_decode_indexed.restype = _i32
    lib.pkv_decode_indexed.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp,
                                       ctypes.c_float, _vp, ctypes.c_size_t, _vp]
    lib.pkv_plan_buckets_host.restype = _i32
    lib.pkv_plan_buckets_host.argtypes = [_vp, _i32, _i32, _vp, _vp, _vp, P(_i32)]
    lib.pkv_decode_buckets.restype = _i32
    lib.pkv_decode_buckets.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, _vp, _i32, _vp, _vp,
                                       ctypes.c_float, _vp, ctypes.c_size_t, _vp]
    lib.pkv_bucket_counters_host.restype = _i32
    lib.pkv_bucket_counters_host.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _i32, P(pkv_counters)]
    lib.pkv_default_cost_model.restype = _i32
    lib.pkv_default_cost_model.argtypes = [_i32, P(pkv_cost_model)]
    lib.pkv_estimate_cost.restype = _i32
    lib.pkv_estimate_cost.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _i32, P(pkv_cost_model), P(pkv_cost_estimate)]
    lib.pkv_choose_policy.restype = _i32
    lib.pkv_choose_policy.argtypes = [P(pkv_shape), _vp, P(pkv_cost_model), P(pkv_split_policy), P(pkv_split_policy),
                                      P(pkv_cost_estimate)]
    lib.pkv_decode_append.restype = _i32
    lib.pkv_decode_append.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, P(pkv_append), _vp, _vp,
                                      ctypes.c_float, _vp, ctypes.c_size_t, _vp]
    lib.pkv_merge.restype = _i32
    lib.pkv_merge.argtypes = [P(pkv_shape), _vp, _vp, _vp, _vp, _vp, _vp, _vp]
    lib.pkv_get_counters.restype = _i32
    lib.pkv_get_counters.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, ctypes.c_size_t, P(pkv_counters), _vp]
    lib.pkv_read_workqueue.restype = _i32
    lib.pkv_read_workqueue.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, ctypes.c_size_t, _vp, _i32, _vp,
                                       P(_i32), _vp]
    lib.pkv_workspace_partials.restype = _i32
    lib.pkv_workspace_partials.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, ctypes.c_size_t, P(_vp), P(_vp),
                                           P(_vp), P(_i64)]
    lib.pkv_decode_host.restype = _i32
    lib.pkv_decode_host.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_float,
                                    _vp, _vp, ctypes.c_size_t, _vp, ctypes.c_size_t, _vp, P(pkv_counters)]
    lib.pkv_decode_host_pipelined.restype = _i32
    lib.pkv_decode_host_pipelined.argtypes = [P(pkv_shape), P(pkv_split_policy), _vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_float,
                                              _vp, _vp, ctypes.c_size_t, _vp, ctypes.c_size_t, _vp, P(pkv_next_step), P(pkv_counters)]
    lib.pkv_decode_host_drain.restype = _i32
    lib.pkv_decode_host_drain.argtypes = [_vp, _vp]
    lib.pkv_calibrate.restype = _i32
    lib.pkv_calibrate.argtypes = [_vp, ctypes.c_size_t, _vp, P(pkv_calibration)]
    return lib


_lib = _load()


def _check(status: int):
    if status != PKV_OK:
        raise PkvError(status, _lib.pkv_last_error().decode("utf-8", "replace"))


# ------------------------------------------------------------------ argument helpers

@dataclass
class Shape:
    B: int
    Hq: int
    Hkv: int
    d: int = 128
    page_size: int = 16
    max_pages: int = 0
    num_pages: int = 0
    kv_strides: Tuple[int, int, int] = (0, 0, 0)   # (page, token, head) in elements; zeros = default layout
    kv_dtype: int = 0                              # KV_F16 / KV_E4M3
    k_scale: object = None                         # device float32 [Hkv] tensors (or raw addresses) for KV_E4M3
    v_scale: object = None

    def c(self) -> pkv_shape:
        return pkv_shape(self.B, self.Hq, self.Hkv, self.d, self.page_size, self.max_pages, self.num_pages,
                         *self.kv_strides, self.kv_dtype, 0, _ptr(self.k_scale), _ptr(self.v_scale))


@dataclass
class Policy:
    tile_tokens: int = 32
    split_mode: int = SPLIT_FIXED_COUNT
    num_splits: int = 1
    chunk_tiles: int = 0
    route: int = ROUTE_WORKQUEUE
    merge_mode: int = MERGE_SEPARATE
    num_sms: int = 0
    kernel: int = KERNEL_AUTO
    flags: int = 0
    heads_per_cta: int = 0
    prefetch_kb: int = 0

    def c(self) -> pkv_split_policy:
        return pkv_split_policy(self.tile_tokens, self.split_mode, self.num_splits, self.chunk_tiles, self.route,
                                self.merge_mode, self.num_sms, self.kernel, self.flags, self.heads_per_cta,
                                self.prefetch_kb)


def _ptr(x) -> Optional[int]:
    """Raw address of a torch tensor, a numpy array, an int, or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data
    assert x.is_contiguous(), "tensors must be contiguous"
    return x.data_ptr()


def _nbytes(x) -> int:
    if isinstance(x, np.ndarray):
        return x.nbytes
    return x.numel() * x.element_size()


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


# ------------------------------------------------------------------ the ABI, name for name

def pkv_version() -> int:
    return int(_lib.pkv_version())


def pkv_last_error() -> str:
    return _lib.pkv_last_error().decode("utf-8", "replace")


def pkv_workspace_bytes(shape: Shape, policy: Policy) -> int:
    n = int(_lib.pkv_workspace_bytes(ctypes.byref(shape.c()), ctypes.byref(policy.c())))
    if n == 0:
        raise PkvError(PKV_ERR_INVALID_ARG, "pkv_workspace_bytes: invalid shape/policy")
    return n


def pkv_workspace_init_bytes(shape: Shape, policy: Policy) -> int:
    n = int(_lib.pkv_workspace_init_bytes(ctypes.byref(shape.c()), ctypes.byref(policy.c())))
    if n == 0:
        raise PkvError(PKV_ERR_INVALID_ARG, "pkv_workspace_init_bytes: invalid shape/policy")
    return n


def pkv_host_scratch_bytes(shape: Shape, policy: Policy) -> int:
    n = int(_lib.pkv_host_scratch_bytes(ctypes.byref(shape.c()), ctypes.byref(policy.c())))
    if n == 0:
        raise PkvError(PKV_ERR_INVALID_ARG, "pkv_host_scratch_bytes: invalid shape/policy")
    return n


def pkv_build_workqueue_host(shape: Shape, policy: Policy, seq_lens_host: np.ndarray):
    """Returns (tasks int32 [num_tasks, 5], split_offsets int32 [B+1])."""
    seq = np.ascontiguousarray(seq_lens_host, dtype=np.int32)
    offsets = np.zeros(shape.B + 1, dtype=np.int32)
    n = _i32(0)
    st = _lib.pkv_build_workqueue_host(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(seq), None, 0,
                                       _ptr(offsets), ctypes.byref(n))
    _check(st)
    tasks = np.zeros((max(int(n.value), 1), 5), dtype=np.int32)
    st = _lib.pkv_build_workqueue_host(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(seq), _ptr(tasks),
                                       tasks.shape[0], _ptr(offsets), ctypes.byref(n))
    _check(st)
    return tasks[:int(n.value)], offsets


def pkv_build_workqueue(shape: Shape, policy: Policy, seq_lens_dev, workspace, stream=None) -> None:
    _check(_lib.pkv_build_workqueue(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(seq_lens_dev),
                                    _ptr(workspace), _nbytes(workspace), _stream_ptr(stream)))


def pkv_decode(shape: Shape, policy: Policy, q, k_cache, v_cache, block_table, seq_lens, out, lse=None,
               scale: float = 0.0, build_queue: bool = True, workspace=None, stream=None) -> None:
    _check(_lib.pkv_decode(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(q), _ptr(k_cache), _ptr(v_cache),
                           _ptr(block_table), _ptr(seq_lens), _ptr(out), _ptr(lse), ctypes.c_float(scale),
                           1 if build_queue else 0, _ptr(workspace), _nbytes(workspace), _stream_ptr(stream)))


def pkv_static_workspace_bytes() -> int:
    return int(_lib.pkv_static_workspace_bytes())


def pkv_decode_static(shape: Shape, policy: Policy, q, k_cache, v_cache, block_table, seq_lens, out, lse=None,
                      scale: float = 0.0, stream=None) -> None:
    """pkv_decode without a caller workspace: the scratch is the library's static device array."""
    _check(_lib.pkv_decode_static(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(q), _ptr(k_cache), _ptr(v_cache),
                                  _ptr(block_table), _ptr(seq_lens), _ptr(out), _ptr(lse), ctypes.c_float(scale),
                                  _stream_ptr(stream)))


def pkv_decode_stages(shape: Shape, policy: Policy, q, k_cache, v_cache, block_table, seq_lens, out, lse=None,
                      scale: float = 0.0, stages: int = STAGE_ALL, workspace=None, stream=None) -> None:
    _check(_lib.pkv_decode_stages(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(q), _ptr(k_cache),
                                  _ptr(v_cache), _ptr(block_table), _ptr(seq_lens), _ptr(out), _ptr(lse),
                                  ctypes.c_float(scale), int(stages), _ptr(workspace), _nbytes(workspace),
                                  _stream_ptr(stream)))


def pkv_decode_indexed(shape: Shape, policy: Policy, q, k_cache, v_cache, block_table, seq_lens, row_index, out, lse=None,
                       scale: float = 0.0, workspace=None, stream=None) -> None:
    _check(_lib.pkv_decode_indexed(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(q), _ptr(k_cache),
                                   _ptr(v_cache), _ptr(block_table), _ptr(seq_lens), _ptr(row_index), _ptr(out), _ptr(lse),
                                   ctypes.c_float(scale), _ptr(workspace), _nbytes(workspace), _stream_ptr(stream)))


def pkv_plan_buckets_host(seq_lens_host: np.ndarray, bucket_tokens: int):
    """Returns (row_index int32 [B], bucket_offsets int32 [num_buckets+1], bucket_lengths int32 [num_buckets])."""
    seq = np.ascontiguousarray(seq_lens_host, dtype=np.int32)
    B = len(seq)
    index = np.zeros(max(B, 1), dtype=np.int32)
    offs = np.zeros(B + 1, dtype=np.int32)
    lens = np.zeros(max(B, 1), dtype=np.int32)
    nb = _i32(0)
    _check(_lib.pkv_plan_buckets_host(_ptr(seq), B, int(bucket_tokens), _ptr(index), _ptr(offs), _ptr(lens), ctypes.byref(nb)))
    return index[:B], offs[:nb.value + 1], lens[:nb.value]


def pkv_decode_buckets(shape: Shape, policy: Policy, q, k_cache, v_cache, block_table, seq_lens, row_index,
                       bucket_offsets_host: np.ndarray, out, lse=None, scale: float = 0.0, workspace=None, stream=None) -> None:
    offs = np.ascontiguousarray(bucket_offsets_host, dtype=np.int32)
    _check(_lib.pkv_decode_buckets(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(q), _ptr(k_cache),
                                   _ptr(v_cache), _ptr(block_table), _ptr(seq_lens), _ptr(row_index), _ptr(offs),
                                   len(offs) - 1, _ptr(out), _ptr(lse), ctypes.c_float(scale), _ptr(workspace),
                                   _nbytes(workspace), _stream_ptr(stream)))


def pkv_bucket_counters_host(shape: Shape, policy: Policy, seq_lens_host: np.ndarray, bucket_tokens: int) -> dict:
    seq = np.ascontiguousarray(seq_lens_host, dtype=np.int32)
    c = pkv_counters()
    _check(_lib.pkv_bucket_counters_host(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(seq), int(bucket_tokens),
                                         ctypes.byref(c)))
    return c.as_dict()


@dataclass
class CostModel:
    beta_gbps: float
    lambda_us: float
    c_min: float
    num_sms: int

    def c(self) -> pkv_cost_model:
        return pkv_cost_model(self.beta_gbps, self.lambda_us, self.c_min, self.num_sms, 0)


def pkv_default_cost_model(num_sms: int) -> CostModel:
    m = pkv_cost_model()
    _check(_lib.pkv_default_cost_model(int(num_sms), ctypes.byref(m)))
    return CostModel(m.beta_gbps, m.lambda_us, m.c_min, m.num_sms)


def pkv_estimate_cost(shape: Shape, policy: Policy, seq_lens_host: np.ndarray, bucket_tokens: int, model: CostModel) -> dict:
    seq = np.ascontiguousarray(seq_lens_host, dtype=np.int32)
    e = pkv_cost_estimate()
    _check(_lib.pkv_estimate_cost(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(seq), int(bucket_tokens),
                                  ctypes.byref(model.c()), ctypes.byref(e)))
    return e.as_dict()


def pkv_choose_policy(shape: Shape, seq_lens_host: np.ndarray, model: CostModel, base: Policy):
    """Returns (Policy, estimate dict)."""
    seq = np.ascontiguousarray(seq_lens_host, dtype=np.int32)
    out, e = pkv_split_policy(), pkv_cost_estimate()
    _check(_lib.pkv_choose_policy(ctypes.byref(shape.c()), _ptr(seq), ctypes.byref(model.c()), ctypes.byref(base.c()),
                                  ctypes.byref(out), ctypes.byref(e)))
    return Policy(**{n: int(getattr(out, n)) for n, _ in pkv_split_policy._fields_}), e.as_dict()


@dataclass
class Append:
    """The new token of every row for pkv_decode_append: device tensors (or raw addresses)."""
    k_new: object
    v_new: object
    rope_cos: object = None
    rope_sin: object = None
    rope_positions: int = 0

    def c(self) -> pkv_append:
        return pkv_append(_ptr(self.k_new), _ptr(self.v_new), _ptr(self.rope_cos), _ptr(self.rope_sin), int(self.rope_positions), 0)


def pkv_decode_append(shape: Shape, policy: Policy, q, k_cache, v_cache, block_table, seq_lens, row_index, append: Append, out,
                      lse=None, scale: float = 0.0, workspace=None, stream=None) -> None:
    _check(_lib.pkv_decode_append(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(q), _ptr(k_cache), _ptr(v_cache),
                                  _ptr(block_table), _ptr(seq_lens), _ptr(row_index), ctypes.byref(append.c()), _ptr(out),
                                  _ptr(lse), ctypes.c_float(scale), _ptr(workspace), _nbytes(workspace), _stream_ptr(stream)))


def pkv_merge(shape: Shape, part_m, part_l, part_acc, split_offsets, out, lse=None, stream=None) -> None:
    _check(_lib.pkv_merge(ctypes.byref(shape.c()), _ptr(part_m), _ptr(part_l), _ptr(part_acc), _ptr(split_offsets),
                          _ptr(out), _ptr(lse), _stream_ptr(stream)))


def pkv_get_counters(shape: Shape, policy: Policy, workspace, stream=None) -> dict:
    c = pkv_counters()
    _check(_lib.pkv_get_counters(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(workspace),
                                 _nbytes(workspace), ctypes.byref(c), _stream_ptr(stream)))
    return c.as_dict()


def pkv_read_workqueue(shape: Shape, policy: Policy, workspace, stream=None):
    """Returns (tasks int32 [num_tasks, 5], split_offsets int32 [B+1]) copied from the device."""
    offsets = np.zeros(shape.B + 1, dtype=np.int32)
    n = _i32(0)
    sp = _stream_ptr(stream)
    _check(_lib.pkv_read_workqueue(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(workspace),
                                   _nbytes(workspace), None, 0, _ptr(offsets), ctypes.byref(n), sp))
    tasks = np.zeros((max(int(n.value), 1), 5), dtype=np.int32)
    _check(_lib.pkv_read_workqueue(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(workspace),
                                   _nbytes(workspace), _ptr(tasks), tasks.shape[0], _ptr(offsets), ctypes.byref(n), sp))
    return tasks[:int(n.value)], offsets


def pkv_workspace_partials(shape: Shape, policy: Policy, workspace):
    """Returns (ptr_m, ptr_l, ptr_acc, slots_cap): device addresses inside the workspace."""
    pm, pl, pa, cap = _vp(), _vp(), _vp(), _i64(0)
    _check(_lib.pkv_workspace_partials(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(workspace),
                                       _nbytes(workspace), ctypes.byref(pm), ctypes.byref(pl), ctypes.byref(pa),
                                       ctypes.byref(cap)))
    return int(pm.value), int(pl.value), int(pa.value), int(cap.value)


def pkv_decode_host(shape: Shape, policy: Policy, q_host, k_cache_dev, v_cache_dev, block_table_host, seq_lens_host,
                    out_host, scale: float, host_staging, dev_scratch, workspace, stream=None) -> dict:
    c = pkv_counters()
    _check(_lib.pkv_decode_host(ctypes.byref(shape.c()), ctypes.byref(policy.c()), _ptr(q_host), _ptr(k_cache_dev),
                                _ptr(v_cache_dev), _ptr(block_table_host), _ptr(seq_lens_host), _ptr(out_host),
                                ctypes.c_float(scale), _ptr(host_staging), _ptr(dev_scratch),
                                min(_nbytes(host_staging), _nbytes(dev_scratch)), _ptr(workspace), _nbytes(workspace),
                                _stream_ptr(stream), ctypes.byref(c)))
    return c.as_dict()


class HostDecoder:
    """pkv_decode_host with everything that does not change from step to step marshalled ONCE
    (shape, policy, caches, staging / scratch / workspace, stream): a serving loop then pays one
    ctypes call per decode step.  Still argument marshalling only.  Per step pass raw addresses
    (``tensor.data_ptr()`` / ``array.ctypes.data``) of q, block_table, seq_lens and out."""

    def __init__(self, shape: Shape, policy: Policy, k_cache_dev, v_cache_dev, host_staging, dev_scratch, workspace,
                 scale: float, stream=None):
        self._keep = (k_cache_dev, v_cache_dev, host_staging, dev_scratch, workspace, stream)
        self._shape, self._policy, self._counters = shape.c(), policy.c(), pkv_counters()
        self._head = (ctypes.byref(self._shape), ctypes.byref(self._policy))
        self._k, self._v = _vp(_ptr(k_cache_dev)), _vp(_ptr(v_cache_dev))
        self._tail = (ctypes.c_float(scale), _vp(_ptr(host_staging)), _vp(_ptr(dev_scratch)),
                      ctypes.c_size_t(min(_nbytes(host_staging), _nbytes(dev_scratch))), _vp(_ptr(workspace)),
                      ctypes.c_size_t(_nbytes(workspace)), _vp(_stream_ptr(stream)), ctypes.byref(self._counters))
        self._fn = _lib.pkv_decode_host

    def __call__(self, q_host: int, block_table_host: int, seq_lens_host: int, out_host: int) -> None:
        st = self._fn(*self._head, q_host, self._k, self._v, block_table_host, seq_lens_host, out_host, *self._tail)
        if st != PKV_OK:
            _check(st)

    @property
    def counters(self) -> dict:
        return self._counters.as_dict()


class PipelinedHostDecoder(HostDecoder):
    """pkv_decode_host_pipelined, marshalled once like HostDecoder.  Per step pass raw addresses of this
    step's q, block_table, seq_lens and out and -- to take the next step's submission off the critical
    path -- of the NEXT step's seq_lens and block_table (0 = arm nothing), optionally its caches / out.
    While a step is armed the stream is blocked: call drain() before anything that waits for the stream
    or the device (torch.cuda.synchronize(), freeing memory, ...)."""

    def __init__(self, shape: Shape, policy: Policy, k_cache_dev, v_cache_dev, host_staging, dev_scratch, workspace,
                 scale: float, stream=None):
        super().__init__(shape, policy, k_cache_dev, v_cache_dev, host_staging, dev_scratch, workspace, scale, stream)
        self._fn = _lib.pkv_decode_host_pipelined
        self._next = pkv_next_step()
        self._next_ref = ctypes.byref(self._next)
        self._tail_a, self._tail_b = self._tail[:-1], self._tail[-1]     # ... stream | counters
        self._staging, self._stream = _vp(_ptr(host_staging)), _vp(_stream_ptr(stream))

    def __call__(self, q_host: int, block_table_host: int, seq_lens_host: int, out_host: int, next_seq_lens_host: int = 0,
                 next_block_table_host: int = 0, k_cache_dev: int = 0, v_cache_dev: int = 0, next_k_cache_dev: int = 0,
                 next_v_cache_dev: int = 0, next_out_host: int = 0) -> None:
        n = self._next
        n.seq_lens_host, n.block_table_host = next_seq_lens_host or None, next_block_table_host or None
        n.k_cache_dev, n.v_cache_dev, n.out_host = next_k_cache_dev or None, next_v_cache_dev or None, next_out_host or None
        st = self._fn(*self._head, q_host, k_cache_dev or self._k, v_cache_dev or self._v, block_table_host, seq_lens_host, out_host,
                      *self._tail_a, self._next_ref, self._tail_b)
        if st != PKV_OK:
            _check(st)

    def prepare(self, q_host: int, block_table_host: int, seq_lens_host: int, out_host: int, next_seq_lens_host: int = 0,
                next_block_table_host: int = 0, k_cache_dev: int = 0, v_cache_dev: int = 0, next_k_cache_dev: int = 0,
                next_v_cache_dev: int = 0, next_out_host: int = 0):
        """The marshalled argument list of one step, for run(): a decode loop passes the same few buffers
        again and again, so the per-step cost of building a struct and seventeen arguments can be paid once."""
        n = pkv_next_step()
        n.seq_lens_host, n.block_table_host = next_seq_lens_host or None, next_block_table_host or None
        n.k_cache_dev, n.v_cache_dev, n.out_host = next_k_cache_dev or None, next_v_cache_dev or None, next_out_host or None
        return (*self._head, _vp(q_host), _vp(k_cache_dev) if k_cache_dev else self._k, _vp(v_cache_dev) if v_cache_dev else self._v,
                _vp(block_table_host), _vp(seq_lens_host), _vp(out_host), *self._tail_a, ctypes.byref(n), self._tail_b, n)

    def run(self, prepared) -> None:
        st = self._fn(*prepared[:-1])       # the last element keeps the pkv_next_step alive
        if st != PKV_OK:
            _check(st)

    def drain(self) -> None:
        _check(_lib.pkv_decode_host_drain(self._staging, self._stream))


def pkv_calibrate(dev_buffer, stream=None) -> dict:
    """Measures beta (read bandwidth) and lambda (launch overhead) on the current device."""
    c = pkv_calibration()
    _check(_lib.pkv_calibrate(_ptr(dev_buffer), _nbytes(dev_buffer), _stream_ptr(stream), ctypes.byref(c)))
    return c.as_dict()
