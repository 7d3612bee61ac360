"""Depth-synchronous frontier builder: with W = B lanes it selects
the same nodes as the best-first heap ("the equivalence suite asserts exact tree equality on tie-free random inputs at
batch sizes 1 through 32").  GPU tests: frontier schedule vs the float64 oracle of Algorithm 1 (the
tolerant comparator) and vs the CUDA heap schedule (bit-equal trees on these tie-free inputs)."""
import os
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2607_08642_b200 import workloads as wl  # noqa: E402


def _frontier(case, inp, M, B, T):
    case.builder.set_option("schedule", 1)
    try:
        out = case.run_gpu(inp, M, B, T)
        torch.cuda.synchronize()
        launches = case.builder.kernel_launches
    finally:
        case.builder.set_option("schedule", 0)
    return out, launches


@pytest.mark.gpu
@pytest.mark.parametrize("batch", [1, 2, 7, 32])
def test_frontier_equals_heap_tiny_fp32(batch):
    import gpu_util as gu
    case = gu.tiny_case()
    for B, T, regime in ((8, 0.0, "flat"), (24, 0.6, "peaked"), (64, 1.0, "flat")):
        inp = wl.make_inputs(case.cfg, batch=batch, seed=8000 + B + batch, regime=regime)
        out, launches = _frontier(case, inp, 8, B, T)
        assert launches == 2 + case.cfg.L + 1          # select, precompute, L depths, selection: fixed shape
        ne, nt = gu.check_batch(case, inp, 8, B, T, 1e-5, out=out)
        assert ne + nt == batch
        heap = case.run_gpu(inp, 8, B, T)
        for name in ("tokens", "parents", "depths", "positions", "mask", "n_nodes"):
            assert torch.equal(getattr(heap, name), getattr(out, name)), name
        assert torch.allclose(heap.scores, out.scores, atol=1e-5, rtol=0)


@pytest.mark.gpu
def test_frontier_short_trees_and_k1():
    """k = 1 chain longer than L (ledger exhausted -> dead-leaf padding) and leaves at depth L."""
    import gpu_util as gu
    case = gu.tiny_case(k=1)
    inp = wl.make_inputs(case.cfg, batch=3, seed=77)
    out, _ = _frontier(case, inp, 4, 12, 0.0)
    assert out.n_nodes.tolist() == [case.cfg.L + 1] * 3
    ne, nt = gu.check_batch(case, inp, 4, 12, 0.0, 1e-5, out=out)
    assert ne + nt == 3


@pytest.mark.gpu
def test_frontier_bf16_matches_oracle_and_heap_nodes():
    """bf16 weights (small shape): frontier vs oracle by the tolerant comparator; same node set as the fused heap."""
    import gpu_util as gu
    cfg = wl.CONFIGS["tiny"].replace(dtype="bf16", g=64, r=40, d=96, V=2000, L=5, embed_std=1.0)
    case = gu.get_case("frontier-bf16", cfg, max_batch=8, max_M=32, max_B=48, k=4)
    inp = wl.make_inputs(case.cfg, batch=5, seed=4242)
    out, _ = _frontier(case, inp, 20, 17, 0.6)
    ne, nt = gu.check_batch(case, inp, 20, 17, 0.6, 2e-3, out=out)
    assert ne + nt == 5


@pytest.mark.gpu
def test_frontier_qwen8b_shape_equals_heap():
    """Qwen3-8B shape (BASELINE configs[2]), batch 2, B = 16: frontier schedule vs the oracle and vs the fused heap."""
    import gpu_util as gu
    case = gu.qwen8b_case()
    inp = wl.make_inputs(case.cfg, batch=2, seed=515, regime="flat")
    out, launches = _frontier(case, inp, 64, 16, 0.0)
    assert launches <= 4            # select, precompute GEMM (2), ONE persistent kernel: the wavefront kernel at full width
    ne, nt = gu.check_batch(case, inp, 64, 16, 0.0, 2e-3, out=out)
    assert ne + nt == 2
    heap = case.run_gpu(inp, 64, 16, 0.0)
    assert torch.equal(heap.tokens, out.tokens) and torch.equal(heap.parents, out.parents)
