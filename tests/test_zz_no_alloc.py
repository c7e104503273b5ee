"""pkv_decode_static (include/pkv.h "Allocation-free entry point"): the decode step whose scratch is
the library's static device array instead of a caller workspace.  Its output is compared with the
existing path's (pkv_decode on a workspace of the caller) on the same inputs, within the parity
tolerance of the other GPU tests (helpers.assert_within_tolerance: max abs 2e-3, floored max rel
1e-2, mean abs 3e-4), on calls in a row that share the array.

Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
from helpers import assert_within_tolerance, make_problem

RAGGED = [1, 2, 15, 16, 17, 31, 32, 33, 100, 0, 257, 700]


def test_static_workspace_limit_is_stated_and_enforced():
    """Sizes beyond the maximum are refused with both numbers in the message -- before any CUDA call,
    so this runs without a device and with null buffers (stream 0 given explicitly: the binding's default
    asks torch for the current CUDA stream)."""
    assert pkv.pkv_static_workspace_bytes() == 8 << 20
    shape = pkv.Shape(B=128, Hq=32, Hkv=8, d=128, page_size=16, max_pages=4100, num_pages=270000)
    pol = pkv.Policy(tile_tokens=32, num_splits=8)
    need = pkv.pkv_workspace_bytes(shape, pol)
    assert need > pkv.pkv_static_workspace_bytes()
    with pytest.raises(pkv.PkvError) as ei:
        pkv.pkv_decode_static(shape, pol, None, None, None, None, None, None, stream=0)
    assert ei.value.status == pkv.PKV_ERR_WORKSPACE
    assert str(need) in str(ei.value) and str(8 << 20) in str(ei.value)
    # an invalid shape is reported as such, not as a size problem
    with pytest.raises(pkv.PkvError) as ei:
        pkv.pkv_decode_static(pkv.Shape(B=1, Hq=32, Hkv=5, d=128, page_size=16, max_pages=1, num_pages=1), pol,
                              None, None, None, None, None, None, stream=0)
    assert ei.value.status in (pkv.PKV_ERR_INVALID_ARG, pkv.PKV_ERR_UNSUPPORTED)


class _Case:
    """One problem on the device with the existing path's result (caller-owned workspace)."""

    def __init__(self, lens, seed, pol, Hkv=8):
        from gpu_helpers import DevProblem
        self.pol = pol
        self.dp = DevProblem(make_problem(lens, seed=seed, Hkv=Hkv))
        self.ref_out, self.ref_lse, _ = self.dp.decode(pol)
        p = self.dp.p
        self.out = torch.full((p.B, p.Hq, p.d), float("nan"), dtype=torch.float16, device="cuda")
        self.lse = torch.full((p.B, p.Hq), float("nan"), dtype=torch.float32, device="cuda")

    def launch_static(self):
        dp = self.dp
        self.out.fill_(float("nan"))
        self.lse.fill_(float("nan"))
        pkv.pkv_decode_static(dp.shape, self.pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, self.out, self.lse, scale=dp.p.scale)

    def check(self, what):
        out = self.out.cpu().numpy().astype(np.float64)
        lse = self.lse.cpu().numpy().astype(np.float64)
        assert not np.isnan(out).any(), what
        assert_within_tolerance(out, self.ref_out, what)
        fin = np.isfinite(self.ref_lse)
        assert np.array_equal(np.isneginf(lse), np.isneginf(self.ref_lse)), what
        assert np.abs(lse[fin] - self.ref_lse[fin]).max(initial=0.0) <= 2e-3, what


@pytest.mark.gpu
def test_static_matches_existing_path_on_calls_in_a_row():
    # different batch sizes, split counts, merge modes and kernels: the shared array is laid out
    # differently from call to call and holds the previous call's queue and partial states
    a = _Case(RAGGED, 901, pkv.Policy(tile_tokens=32, num_splits=4))
    b = _Case([3000, 40, 0, 1025, 5000], 902, pkv.Policy(tile_tokens=32, num_splits=16, merge_mode=pkv.MERGE_FUSED), Hkv=4)
    c = _Case([777, 12, 2049], 903, pkv.Policy(tile_tokens=32, num_splits=3, kernel=pkv.KERNEL_SIMT))
    # two calls in a row on one stream, no synchronisation between them
    a.launch_static()
    b.launch_static()
    torch.cuda.synchronize()
    a.check("call 1 (S=4, separate merge)")
    b.check("call 2 (S=16, fused merge) right behind call 1")
    c.launch_static()
    a.launch_static()
    torch.cuda.synchronize()
    c.check("call 3 (SIMT kernel)")
    a.check("call 4 = call 1 again, after other layouts used the array")


@pytest.mark.gpu
def test_static_largest_supported_split_count():
    """B = 1 with S = 256 (4.1 MiB of scratch) fits the 8 MiB array; N just past a tile boundary."""
    pol = pkv.Policy(tile_tokens=32, num_splits=256)
    case = _Case([32768 + 17], 904, pol)
    assert pkv.pkv_workspace_bytes(case.dp.shape, pol) <= pkv.pkv_static_workspace_bytes()
    case.launch_static()
    case.launch_static()
    torch.cuda.synchronize()
    case.check("S=256, two calls in a row")
