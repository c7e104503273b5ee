"""paper_2606_26666_b200 -- B200-native paged GQA decode attention (PersistentKV hot path).

The product is ``libpkv.so`` (hand-written CUDA for sm_100a behind the C ABI of
``include/pkv.h``); this package is its thin ctypes binding.  PyTorch is used by callers only
for device memory, streams and CUDA graphs.  Importing the package loads (building if needed)
the shared library and raises if that fails -- there is no CPU or PyTorch fallback.
"""
from .binding import (  # noqa: F401
    PKV_OK, PKV_ERR_INVALID_ARG, PKV_ERR_UNSUPPORTED, PKV_ERR_WORKSPACE, PKV_ERR_CUDA,
    ROUTE_RECT, ROUTE_WORKQUEUE, MERGE_SEPARATE, MERGE_FUSED, SPLIT_FIXED_COUNT, SPLIT_FIXED_CHUNK, SPLIT_BALANCED, SPLIT_AUTO,
    KERNEL_AUTO, KERNEL_TMA_MMA, KERNEL_SIMT, FLAG_VALIDATE, FLAG_NO_PDL, FLAG_SEPARATE_BUILD, FLAG_TEST_REPLAN, FLAG_OUT_PINNED,
    DEVERR_QUEUE_OVERFLOW, DEVERR_SEQ_LEN, DEVERR_PAGE_ID, STAGE_BUILD, STAGE_DECODE, STAGE_MERGE, STAGE_ALL, KV_F16, KV_E4M3, KV_INT8, EXPORTS,
    PkvError, Shape, Policy, CostModel, HostDecoder, PipelinedHostDecoder, Append, pkv_decode_append, pkv_default_cost_model, pkv_estimate_cost, pkv_choose_policy,
    pkv_version, pkv_last_error, pkv_workspace_bytes, pkv_workspace_init_bytes, pkv_host_scratch_bytes, pkv_build_workqueue_host,
    pkv_build_workqueue, pkv_decode, pkv_decode_stages, pkv_merge, pkv_get_counters, pkv_read_workqueue, pkv_workspace_partials,
    pkv_decode_host, pkv_calibrate, pkv_decode_indexed, pkv_plan_buckets_host, pkv_decode_buckets, pkv_bucket_counters_host,
    pkv_decode_static, pkv_static_workspace_bytes,
)


def alloc_workspace(shape, policy, device="cuda"):
    """A torch uint8 buffer of pkv_workspace_bytes(shape, policy) on ``device`` (plumbing only).
    Its first pkv_workspace_init_bytes() bytes (queue header, completion counters) are zeroed, as include/pkv.h asks for a fresh workspace."""
    import torch

    ws = torch.empty(pkv_workspace_bytes(shape, policy), dtype=torch.uint8, device=device)
    ws[:pkv_workspace_init_bytes(shape, policy)].zero_()
    return ws
