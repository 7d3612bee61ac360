"""Marg and Cond-static scorer arms: oracle pins (CPU) and GPU parity."""
import os
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from oracle import scorers  # noqa: E402
from paper_2607_08642_b200 import workloads as wl  # noqa: E402


def _case(**kw):
    cfg = wl.CONFIGS["tiny"].replace(**kw) if kw else wl.CONFIGS["tiny"]
    w = wl.make_weights(cfg)
    return cfg, w


def _paths(tokens, parents, n):
    out = {}
    for i in range(1, n):
        p, u = [], i
        while u > 0:
            p.append(int(tokens[u])); u = int(parents[u])
        out[tuple(p[::-1])] = i
    return out


def _same_tree(t, ref, tol=1e-9):
    """Bit-equal structure, or -- when two float64 formulations round mathematically equal sums differently -- the
    same node set and scores, with free order among scores closer than `tol` (boundary ties excluded)."""
    tokens, parents, depths, positions, scores, mask, n = t
    assert n == ref.n_nodes
    assert np.allclose(scores[:n], ref.scores[:n], atol=tol, rtol=0)
    if (np.array_equal(tokens, ref.tokens) and np.array_equal(parents, ref.parents)
            and np.array_equal(depths, ref.depths) and np.array_equal(mask, ref.mask)):
        assert np.array_equal(positions, ref.positions)
        return
    pa, pb = _paths(tokens, parents, n), _paths(ref.tokens, ref.parents, n)
    last = min(scores[n - 1], ref.scores[n - 1])
    for path, i in pa.items():
        if scores[i] > last + tol:
            assert path in pb and abs(ref.scores[pb[path]] - scores[i]) <= tol, path
    for path, i in pb.items():
        if ref.scores[i] > last + tol:
            assert path in pa, path
    assert all(parents[i] < i and depths[i] == depths[parents[i]] + 1 for i in range(1, n))


@pytest.mark.parametrize("regime", ["flat", "peaked"])
@pytest.mark.parametrize("T", [0.0, 0.6])
def test_marg_equals_algorithm1_with_the_correction_zeroed(regime, T):
    # PAPER.md:553 "ignoring the GRU correction entirely": the C oracle of Alg. 1 with W2 = 0 is that arm
    cfg, w = _case()
    w0 = dict(w); w0["corr_w2"] = torch.zeros_like(w["corr_w2"])
    worc = oracle.Weights.from_dict(w0)
    inp = wl.make_inputs(cfg, batch=3, regime=regime)
    for b in range(3):
        for B, k in ((8, 8), (20, 3), (5, 1)):
            ref = oracle.build_tree(worc, inp["logits"][b], inp["hidden"][b], int(inp["root_tokens"][b]),
                                    int(inp["root_positions"][b]), 8, B, k, T)
            menus = scorers.marg_menus(inp["logits"][b], 8, k, T)
            _same_tree(scorers.factorized_tree(menus, int(inp["root_tokens"][b]), int(inp["root_positions"][b]), B), ref)


def test_cond_static_with_path_independent_states_equals_dominotree():
    # all embedding rows equal => the GRU state depends on the depth only, never on the realized tokens, so the
    # per-node correction (DominoTree) and the greedy-path correction (Cond-static) coincide
    cfg, w = _case(embed_std=1.0)
    w1 = dict(w); w1["embed"] = w["embed"][:1].expand_as(w["embed"]).contiguous()
    worc = oracle.Weights.from_dict(w1)
    inp = wl.make_inputs(cfg, batch=3)
    for b in range(3):
        root, rp = int(inp["root_tokens"][b]), int(inp["root_positions"][b])
        ref = oracle.build_tree(worc, inp["logits"][b], inp["hidden"][b], root, rp, 8, 16, 4, 0.6)
        menus = scorers.cond_static_menus(worc, inp["logits"][b], inp["hidden"][b], root, 8, 4, 0.6)
        _same_tree(scorers.factorized_tree(menus, root, rp, 16), ref)


def test_cond_static_chain_is_dominos_greedy_chain():
    # k = 1, B = L: the tree is the greedy trajectory itself, for which Alg. 1 and Cond-static agree
    cfg, w = _case(embed_std=1.0)
    worc = oracle.Weights.from_dict(w)
    inp = wl.make_inputs(cfg, batch=2, regime="peaked")
    for b in range(2):
        root, rp = int(inp["root_tokens"][b]), int(inp["root_positions"][b])
        ref = oracle.build_tree(worc, inp["logits"][b], inp["hidden"][b], root, rp, 8, cfg.L, 1, 0.0)
        menus = scorers.cond_static_menus(worc, inp["logits"][b], inp["hidden"][b], root, 8, 1, 0.0)
        _same_tree(scorers.factorized_tree(menus, root, rp, cfg.L), ref)


def test_cond_static_differs_from_marg_and_from_dominotree_on_the_stress_config():
    # the ladder has three distinct rungs when the path actually matters (E ~ N(0,1))
    cfg, w = _case(embed_std=1.0)
    worc = oracle.Weights.from_dict(w)
    inp = wl.make_inputs(cfg, batch=6)
    diff_marg = diff_dt = 0
    for b in range(6):
        root, rp = int(inp["root_tokens"][b]), int(inp["root_positions"][b])
        cs = scorers.factorized_tree(scorers.cond_static_menus(worc, inp["logits"][b], inp["hidden"][b], root, 8, 8, 0.0), root, rp, 32)
        mg = scorers.factorized_tree(scorers.marg_menus(inp["logits"][b], 8, 8, 0.0), root, rp, 32)
        dt = oracle.build_tree(worc, inp["logits"][b], inp["hidden"][b], root, rp, 8, 32, 8, 0.0)
        diff_marg += not (np.array_equal(cs[0], mg[0]) and np.array_equal(cs[1], mg[1]))
        diff_dt += not (np.array_equal(cs[0], dt.tokens) and np.array_equal(cs[1], dt.parents))
        # the first level is the same menu in Cond-static and DominoTree: CHILDREN(S_0, 1)
        lvl1_cs = sorted(int(cs[0][i]) for i in range(1, cs[6]) if cs[2][i] == 1)
        lvl1_dt = sorted(int(dt.tokens[i]) for i in range(1, dt.n_nodes) if dt.depths[i] == 1)
        assert set(lvl1_cs) <= set(int(x) for x in scorers.cond_static_menus(worc, inp["logits"][b], inp["hidden"][b], root, 8, 8, 0.0)[0][0])
        assert lvl1_dt  # non-empty
    assert diff_marg > 0 and diff_dt > 0


def test_factorized_tree_invariants_and_closed_form():
    cfg, _ = _case()
    inp = wl.make_inputs(cfg, batch=1)
    menus = scorers.marg_menus(inp["logits"][0], 8, 3, 1.0)
    tokens, parents, depths, positions, scores, mask, n = scorers.factorized_tree(menus, 5, 100, 20)
    assert all(scores[i] <= scores[i - 1] + 1e-12 for i in range(2, n))           # pop order non-increasing
    for i in range(1, n):
        p = parents[i]
        assert p < i and depths[i] == depths[p] + 1 and positions[i] == 100 + depths[i]
        d = depths[i] - 1
        j = list(menus[d][0]).index(tokens[i])
        assert abs(scores[i] - (scores[p] + menus[d][1][j])) < 1e-12               # g = sum of menu entries
        assert mask[i].sum() == depths[i] + 1
    # top-B of all factorized sums: brute force over the 3-ary tree of depth L
    allg = []
    def rec(g, d):
        if d == cfg.L:
            return
        for j in range(3):
            allg.append(g + menus[d][1][j]); rec(g + menus[d][1][j], d + 1)
    rec(0.0, 0)
    want = sorted(allg, reverse=True)[:n - 1]
    assert np.allclose(sorted(scores[1:n], reverse=True), want, atol=1e-12)


# ------------------------------------------------------------------------------------------- GPU parity
class _Ref:
    def __init__(self, t):
        self.tokens, self.parents, self.depths, self.positions, self.scores, self.mask, self.n_nodes = t


def _gpu_tree(out, b):
    n = int(out.n_nodes[b])
    return (out.tokens[b].cpu().numpy().astype(np.int64), out.parents[b].cpu().numpy().astype(np.int64),
            out.depths[b].cpu().numpy().astype(np.int64), out.positions[b].cpu().numpy().astype(np.int64),
            out.scores[b].cpu().numpy().astype(np.float64), out.mask[b].cpu().numpy(), n)


def _run_scorer(case, inp, M, B, T, scorer):
    case.builder.set_option("scorer", scorer)
    try:
        out = case.run_gpu(inp, M, B, T)
        torch.cuda.synchronize()
        launches = case.builder.kernel_launches
    finally:
        case.builder.set_option("scorer", 0)
    return out, launches


@pytest.mark.gpu
@pytest.mark.parametrize("cfgname,dtype_kw", [("tiny", {}), ("tiny", {"dtype": "bf16", "V": 2000})])
def test_gpu_marg_matches_oracle(cfgname, dtype_kw):
    import gpu_util as gu
    case = gu.tiny_case(**dtype_kw) if dtype_kw else gu.tiny_case()
    for batch, M, B, T, regime in ((5, 8, 8, 0.0, "flat"), (32, 8, 31, 0.6, "peaked"), (3, 9, 64, 1.0, "flat")):
        inp = wl.make_inputs(case.cfg, batch=batch, seed=6000 + B, regime=regime)
        out, launches = _run_scorer(case, inp, M, B, T, 1)
        assert launches <= 4
        for b in range(batch):
            menus = scorers.marg_menus(inp["logits"][b], M, case.k, T)
            ref = _Ref(scorers.factorized_tree(menus, int(inp["root_tokens"][b]), int(inp["root_positions"][b]), B))
            _same_tree(_gpu_tree(out, b), ref, tol=1e-4)
            n = ref.n_nodes
            assert np.max(np.abs(_gpu_tree(out, b)[4][:n] - ref.scores[:n])) < 2e-3


@pytest.mark.gpu
@pytest.mark.parametrize("g,path", [(256, 0), (64, 0)])
def test_gpu_cond_static_matches_oracle(g, path):
    """Cond-static through the fused kernel in static mode (tcgen05 GRU role at g = 256, mma.sync at g = 64)."""
    import gpu_util as gu
    cfg = wl.CONFIGS["tiny"].replace(dtype="bf16", g=g, r=40, d=96, V=2000, L=5, embed_std=1.0)
    case = gu.get_case(f"cs-{g}", cfg, max_batch=40, max_M=32, max_B=48, k=4)
    worc = oracle.Weights.from_dict(case.w_cpu) if hasattr(case, "w_cpu") else case.w_orc
    for batch, M, B, T in ((1, 8, 8, 0.0), (7, 20, 17, 0.6), (33, 24, 40, 1.0)):
        inp = wl.make_inputs(case.cfg, batch=batch, seed=7000 + B)
        out, launches = _run_scorer(case, inp, M, B, T, 2)
        assert launches <= 6
        for b in range(batch):
            root, rp = int(inp["root_tokens"][b]), int(inp["root_positions"][b])
            menus = scorers.cond_static_menus(worc, inp["logits"][b], inp["hidden"][b], root, M, case.k, T)
            ref = _Ref(scorers.factorized_tree(menus, root, rp, B))
            _same_tree(_gpu_tree(out, b), ref, tol=1e-4)
        # and it is a different tree from DominoTree's on this path-sensitive config for at least one request
        dt_out = case.run_gpu(inp, M, B, T)
        if batch >= 7:
            assert not (torch.equal(dt_out.tokens, out.tokens) and torch.equal(dt_out.parents, out.parents))


@pytest.mark.gpu
def test_gpu_cond_static_unsupported_for_fp32():
    import gpu_util as gu
    import paper_2607_08642_b200 as dtb
    case = gu.tiny_case()
    inp = wl.make_inputs(case.cfg, batch=1)
    with pytest.raises(dtb.DominoTreeError):
        _run_scorer(case, inp, 8, 8, 0.0, 2)
