"""dt_select_topm_static: the top-M select for callers that cannot allocate (no handle, scratch in a static device
array of the library, include/dominotree.h).  The GPU tests check its output against the existing path
(dt_select_topm on a handle) on two calls in a row that share the array: bit-exact, the bar of every select test
(BASELINE.json north_star: select bit-exact).  Collected last on purpose (file name): the suite runs with pytest -x.
"""
import ctypes

import numpy as np
import pytest
import torch

import oracle
import paper_2607_08642_b200 as dtb
from paper_2607_08642_b200 import workloads as wl


def _gu():
    import gpu_util
    return gpu_util


def test_static_limits_need_no_gpu():
    """Sizes beyond the static array are refused with their own error code before any CUDA call."""
    from paper_2607_08642_b200 import build
    build.build()
    lib = dtb.load_library()
    one = ctypes.c_void_p(16)
    assert lib.dt_select_topm_static(one, dtb.DT_BF16, dtb.STATIC_MAX_ROWS + 1, 4096, 8, one, one, None) == -5
    assert lib.dt_select_topm_static(one, dtb.DT_BF16, 4, 4096, 257, one, one, None) == -5
    assert lib.dt_select_topm_static(one, 7, 4, 4096, 8, one, one, None) == -1            # dtype
    assert lib.dt_select_topm_static(one, dtb.DT_F32, 4, 4, 8, one, one, None) == -1      # M > V
    assert lib.dt_select_topm_static(one, dtb.DT_F32, -1, 64, 8, one, one, None) == -1
    assert lib.dt_select_topm_static(None, dtb.DT_F32, 0, 64, 8, None, None, None) == 0   # rows == 0: no-op
    assert b"static" in lib.dt_error_string(-5)


def _static(lg_gpu, M):
    rows = lg_gpu.reshape(-1, lg_gpu.shape[-1]).shape[0]
    ids = torch.full((rows, M), -7, dtype=torch.int32, device="cuda")
    vals = torch.full((rows, M), float("nan"), dtype=torch.float32, device="cuda")
    dtb.select_topm_static(lg_gpu, M, ids, vals)
    return ids, vals


def _same(a, b):
    return torch.equal(a[0], b[0]) and torch.equal(a[1].view(torch.int32), b[1].view(torch.int32))


@pytest.mark.gpu
def test_static_select_matches_handle_path_twice_in_a_row_bf16():
    """Qwen-sized bf16 rows through the bulk-copy kernel.  Call 1: 64 rows split into chunks (the partial lists, tickets
    and thresholds of the static array are all in use); call 2, enqueued right behind it with no synchronisation:
    fewer rows, another M, other data, so the array still holds call 1's contents where call 2 does not overwrite."""
    case = _gu().qwen8b_case()
    lg1 = wl.make_inputs(case.cfg, batch=4, regime="flat")["logits"].cuda()
    lg2 = wl.make_inputs(case.cfg, batch=1, regime="peaked")["logits"].cuda()
    ref1 = case.builder.select_topm(lg1, 64)
    ref2 = case.builder.select_topm(lg2, 32)
    torch.cuda.synchronize()
    got1 = _static(lg1, 64)          # also the one-time set-up of this device
    got2 = _static(lg2, 32)
    torch.cuda.synchronize()
    assert _same(got1, ref1) and _same(got2, ref2)
    # the same pair again: now every word of the scratch that the calls touch is stale, and nothing may be allocated
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    again1 = _static(lg1, 64)
    again2 = _static(lg2, 32)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "the static entry point must not allocate device memory"
    assert _same(again1, ref1) and _same(again2, ref2)
    # and against the oracle on a few rows (the handle path is itself checked against it in test_gpu_parity.py)
    lgc = lg2.reshape(-1, lg2.shape[-1]).cpu()
    for r in (0, 7, 15):
        oi, ov = oracle.select_topm(lgc[r], 32)
        assert np.array_equal(got2[0][r].cpu().numpy(), oi)
        assert np.array_equal(got2[1][r].cpu().numpy().astype(np.float64), ov)


@pytest.mark.gpu
def test_static_select_full_size_and_limit():
    """BASELINE configs[4] select at full size (512 rows x 151,936 bf16, one chunk per row) and the largest row count the
    static array takes (1024 rows, fp32, V = 8192 + 64)."""
    case = _gu().qwen8b_case()
    lg = wl.make_inputs(wl.CONFIGS["concurrent8b"], batch=32, regime="flat")["logits"].cuda()
    ref = case.builder.select_topm(lg, 64)
    got = _static(lg, 64)
    torch.cuda.synchronize()
    assert _same(got, ref)
    del lg
    tiny = _gu().tiny_case(name="tiny", V=8192 + 64)
    g = torch.Generator().manual_seed(5)
    big = torch.randn((dtb.STATIC_MAX_ROWS, 8192 + 64), generator=g, dtype=torch.float32).cuda()
    got = _static(big, 64)
    torch.cuda.synchronize()
    for lo in range(0, dtb.STATIC_MAX_ROWS, 64):            # the handle path takes max_batch * L = 128 rows per call
        ref = tiny.builder.select_topm(big[lo:lo + 64], 64)
        torch.cuda.synchronize()
        assert _same((got[0][lo:lo + 64], got[1][lo:lo + 64]), ref), lo
    with pytest.raises(dtb.DominoTreeError, match="static scratch"):
        _static(torch.zeros((dtb.STATIC_MAX_ROWS + 1, 64), dtype=torch.float32, device="cuda"), 8)


@pytest.mark.gpu
@pytest.mark.parametrize("V", [1001, 4099])
def test_static_select_unaligned_fp32_twice(V):
    """Rows that are not 16-byte aligned take the register-tile kernel; two calls in a row, adversarial rows second."""
    case = _gu().tiny_case(name="tiny", V=V, max_M=8)
    lg1 = wl.make_inputs(case.cfg, batch=3)["logits"].cuda()
    adv = torch.stack(list(wl.adversarial_select_rows(V, case.cfg.torch_dtype).values())).cuda()
    ref1 = case.builder.select_topm(lg1, 8)
    ref2 = case.builder.select_topm(adv, 8)
    got1 = _static(lg1, 8)
    got2 = _static(adv, 8)
    torch.cuda.synchronize()
    assert _same(got1, ref1) and _same(got2, ref2)
