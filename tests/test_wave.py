"""Wavefront expansion kernel (dt_wave.cuh) and the adaptive schedule, -m gpu, through the C-ABI.

* every wave width against the float64 oracle on small bf16 shapes (ragged batch / M / B / k, short trees);
* the wavefront schedule returns the SAME tree as the lock-step heap schedule (the node set does not depend on
  the order in which CHILDREN(.) is evaluated);
* FULL-SIZE shapes with REAL path dependence (SURVEY.md 8(c) stress row: E ~ N(0, 1) at V = 151 936, d = 4096, g = 1024,
  r = 256): a kernel that mixed up parent state slots, or shared one state across sibling paths, changes these trees --
  asserted with the oracle: the Cond-static tree (states shared along the greedy chain) differs from the
  DominoTree tree on these inputs;
* batch 128 at g = 1024 (more requests than one cooperative launch holds): consecutive launches, no per-step fallback;
* adaptive schedule: the device picks the wavefront kernel on flat inputs and the lock-step kernel on peaked ones.
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import scorers
from paper_2607_08642_b200 import workloads as wl

pytestmark = pytest.mark.gpu
BF16_TOL = 2e-3


def _gu():
    import gpu_util
    return gpu_util


def _small(gu, g, r, k, max_batch=40):
    cfg = wl.CONFIGS["tiny"].replace(dtype="bf16", g=g, r=r, d=96, V=2000, L=5, embed_std=1.0)
    return gu.get_case(f"wave-{g}-{r}-{k}-{max_batch}", cfg, max_batch=max_batch, max_M=32, max_B=48, k=k)


def _with(case, **opts):
    class _Ctx:
        def __enter__(self_):
            for n, v in opts.items():
                case.builder.set_option(n, v)

        def __exit__(self_, *exc):
            for n in opts:
                case.builder.set_option(n, 1 if n == "adaptive_schedule" else 0)
    return _Ctx()


@pytest.mark.parametrize("W", [1, 2, 5, 15])
@pytest.mark.parametrize("g,batch,M,B,k", [(128, 1, 8, 8, 8), (256, 5, 20, 17, 3), (128, 33, 24, 40, 8), (256, 40, 9, 6, 1),
                                           (256, 7, 32, 48, 4)])
def test_wave_small_bf16_vs_oracle(W, g, batch, M, B, k):
    gu = _gu()
    case = _small(gu, g, 40, k)
    inp = wl.make_inputs(case.cfg, batch=batch, seed=1900 + batch + W, regime="flat" if (batch + W) % 2 else "peaked")
    with _with(case, expand_path=5, wave_width=W):
        ne, nt = gu.check_batch(case, inp, M, B, 0.6, BF16_TOL)
        assert case.builder.get_option("expand_path_taken") == 5
        assert case.builder.get_option("device_error") == 0
    print(f"exact {ne} tolerant {nt}")
    assert ne + nt == batch


@pytest.mark.parametrize("regime", ["flat", "peaked"])
def test_wave_equals_lockstep_schedule(regime):
    """Same tokens / parents / depths / mask from both schedules (tie-free inputs); scores to fp32 rounding."""
    gu = _gu()
    case = _small(gu, 256, 40, 8)
    inp = wl.make_inputs(case.cfg, batch=12, seed=2100, regime=regime)
    outs = {}
    for path in (4, 5):
        with _with(case, expand_path=path):
            outs[path] = case.run_gpu(inp, 24, 40, 0.6)
            assert case.builder.get_option("expand_path_taken") == path
    for name in ("tokens", "parents", "depths", "positions", "mask", "n_nodes"):
        assert torch.equal(getattr(outs[4], name), getattr(outs[5], name)), name
    assert torch.allclose(outs[4].scores, outs[5].scores, atol=1e-5, rtol=0)


def test_wave_batch_invariance_bitwise():
    """With the schedule pinned, a request's output does not depend on the batch it ran in."""
    gu = _gu()
    case = _small(gu, 256, 40, 8)
    inp = wl.make_inputs(case.cfg, batch=33, seed=2200)
    with _with(case, expand_path=5, wave_width=3):
        full = case.run_gpu(inp, 24, 40, 0.6)
        for b in (0, 17, 32):
            one = {k_: v[b:b + 1] for k_, v in inp.items()}
            o1 = case.run_gpu(one, 24, 40, 0.6)
            for name in ("tokens", "parents", "depths", "positions", "scores", "mask", "n_nodes"):
                assert torch.equal(getattr(o1, name)[0], getattr(full, name)[b]), (b, name)


# ---------------------------------------------------------------------------------------- full-size stress
def _stress_case(gu):
    cfg = wl.CONFIGS["qwen8b"].replace(embed_std=1.0)
    return gu.get_case("qwen8b-stress", cfg, max_batch=40, max_M=128, max_B=128, k=8)


@pytest.mark.parametrize("path,batch,M,B,regime", [(4, 40, 64, 32, "flat"), (5, 40, 64, 32, "flat"), (5, 32, 128, 128, "peaked"),
                                                    (4, 32, 128, 128, "flat"), (5, 1, 64, 128, "flat"), (4, 1, 64, 32, "peaked"),
                                                    (0, 32, 64, 32, "peaked")])
def test_full_size_stress_path_dependence(path, batch, M, B, regime):
    gu = _gu()
    case = _stress_case(gu)
    T = 0.6
    inp = wl.make_inputs(case.cfg, batch=batch, seed=3100 + B, regime=regime)
    trees = case.run_oracle(inp, M, B, T)
    # the inputs must tell DominoTree from a scorer that shares states across sibling paths (checked on 3 requests)
    differs = 0
    for b in range(min(batch, 3)):
        root, rp = int(inp["root_tokens"][b]), int(inp["root_positions"][b])
        menus = scorers.cond_static_menus(case.w_orc, inp["logits"][b], inp["hidden"][b], root, M, case.k, T)
        cs_tok, cs_par = scorers.factorized_tree(menus, root, rp, B)[:2]
        differs += not (np.array_equal(np.asarray(cs_tok), trees[b].tokens) and np.array_equal(np.asarray(cs_par), trees[b].parents))
    # (peaked rows are decided by the base logits alone, whatever the embedding scale: those cases cover the long chains)
    assert differs >= 1 or regime == "peaked", "Cond-static and DominoTree agree on these inputs: the case has no power"
    with _with(case, expand_path=path):
        # one CUDA graph, as bench.py times it
        lg, hd = inp["logits"].cuda(), inp["hidden"].cuda()
        rt, rp_ = inp["root_tokens"].cuda(), inp["root_positions"].cuda()
        import paper_2607_08642_b200 as dtb
        out = dtb.alloc_outputs(batch, B)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            case.builder.build_trees(lg, hd, rt, rp_, M, B, T, out=out, stream=st)
            st.synchronize()
            taken = case.builder.get_option("expand_path_taken")
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=st):
                case.builder.build_trees(lg, hd, rt, rp_, M, B, T, out=out, stream=st)
        for t in (out.tokens, out.parents, out.scores, out.mask):
            t.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert taken == (path if path else 6)
        assert case.builder.get_option("device_error") == 0
        ne, nt = gu.check_batch(case, inp, M, B, T, BF16_TOL, out=out, trees=trees)
    print(f"path {taken}: exact {ne} tolerant {nt}")
    assert ne + nt == batch


def test_batch_128_runs_on_the_persistent_kernels():
    """batch 128 at g = 1024 does not fit one cooperative launch beside the 64 GRU CTAs: consecutive launches of the
    wavefront kernel, never the 2 B + 3 launches of the per-step fallback."""
    gu = _gu()
    cfg = wl.CONFIGS["qwen8b"]
    base = gu.qwen8b_case()
    case = gu.get_case("qwen8b-b128", cfg, max_batch=128, max_M=64, max_B=16, k=8, weights=base.w_cpu)
    inp = wl.make_inputs(cfg, batch=128, seed=4100, regime="flat")
    out = case.run_gpu(inp, 64, 8, 0.6)
    assert case.builder.get_option("expand_path_taken") == 5
    assert case.builder.kernel_launches <= 6
    assert case.builder.get_option("device_error") == 0
    # oracle on a sample of the requests (both launches)
    from compare import compare_tree, tree_to_numpy
    hid = oracle.to_numpy(inp["hidden"])
    for b in (0, 63, 64, 90, 127):
        tr = oracle.build_tree(case.w_orc, inp["logits"][b], inp["hidden"][b], int(inp["root_tokens"][b]),
                               int(inp["root_positions"][b]), 64, 8, 8, 0.6)
        compare_tree(tree_to_numpy(out, b), tr, case.w_orc, hid[b], int(inp["root_tokens"][b]),
                     int(inp["root_positions"][b]), cfg.L, 8, 8, 0.6, BF16_TOL)


def test_adaptive_schedule_picks_by_regime():
    gu = _gu()
    case = gu.qwen8b_case()
    cfg = wl.CONFIGS["concurrent8b"]
    chosen = {}
    for regime in ("flat", "peaked"):
        inp = wl.make_inputs(cfg, batch=8, seed=5100, regime=regime)
        case.run_gpu(inp, cfg.M, cfg.B, cfg.T)
        assert case.builder.get_option("expand_path_taken") == 6
        chosen[regime] = case.builder.get_option("schedule_chosen")
    assert chosen == {"flat": 1, "peaked": 0}, chosen


@pytest.mark.parametrize("path,schedule", [(5, 0), (4, 0), (0, 1)])
def test_exact_fp32_ties_give_a_valid_tree(path, schedule):
    """Saturated slices (a planted token 40 nats above the row): log p of the top child is exactly 0 in fp32, so a child's
    score EQUALS its parent's and sibling subtrees tie bit for bit.  Every schedule must still return a valid best-first tree
    (parents before children, the same node set up to the comparator's margin): reading A17 / ADVICE r1."""
    gu = _gu()
    case = _small(gu, 256, 40, 8)
    inp = wl.make_inputs(case.cfg, batch=6, seed=2300, regime="peaked")
    lg = inp["logits"].float()
    rows = torch.arange(case.cfg.L)
    for b in range(6):
        lg[b, rows, inp["planted"][b]] = lg[b].max(dim=1).values + 40.0
    inp["logits"] = lg.to(inp["logits"].dtype)
    case.builder.set_option("schedule", schedule)
    try:
        with _with(case, expand_path=path):
            out = case.run_gpu(inp, 24, 40, 1.0)
            ne, nt = gu.check_batch(case, inp, 24, 40, 1.0, BF16_TOL, out=out)
    finally:
        case.builder.set_option("schedule", 0)
    sc = out.scores[:, 1:6].cpu().numpy()
    assert (sc[:, 0] == 0.0).all(), "the inputs were meant to saturate: top child log p == 0"
    print(f"exact {ne} tolerant {nt}")
    assert ne + nt == 6


def test_handles_on_the_same_weights_share_the_input_table():
    """P = E W_ih^T is reference-counted across handles created on the same borrowed weight tensors: the second handle
    gives the same trees, and closing either leaves the other working."""
    import paper_2607_08642_b200 as dtb
    gu = _gu()
    case = _small(gu, 256, 40, 8)
    inp = wl.make_inputs(case.cfg, batch=4, seed=2400)
    ref = case.run_gpu(inp, 24, 20, 0.6)
    b2 = dtb.DominoTreeBuilder(case.w_gpu, max_batch=4, L=case.cfg.L, max_M=32, max_B=48, k=8)
    out2 = b2.build_trees(inp["logits"].cuda(), inp["hidden"].cuda(), inp["root_tokens"].cuda(), inp["root_positions"].cuda(), 24, 20, 0.6)
    torch.cuda.synchronize()
    for name in ("tokens", "parents", "scores", "mask"):
        assert torch.equal(getattr(ref, name), getattr(out2, name)), name
    b2.close()
    again = case.run_gpu(inp, 24, 20, 0.6)
    assert torch.equal(ref.tokens, again.tokens) and torch.equal(ref.scores, again.scores)
