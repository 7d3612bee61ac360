"""Unit tests of the tolerant comparator itself (tests/compare.py, BASELINE.json north_star): a
comparator that accepted anything in its tolerant branch would keep the whole GPU suite green, so it is fed hand-made
"GPU" trees: a constructed 5e-5 near-tie swap must pass as "tolerant"; a 2e-4 swap, a missing oracle node, a node
below the B-th score, a 3e-3 score error and a broken structure must each raise.  CPU only: the trees come from the
float64 oracle and are edited by hand."""
import numpy as np
import pytest
import torch

import oracle
from compare import compare_tree
from paper_2607_08642_b200 import workloads as wl

K, M, T = 4, 8, 0.0


def _setup(gap):
    """Tiny fp32 case whose two best depth-1 candidates are an exact copy of one another except for a base-logit gap
    `gap` (same W2 row, so the correction is the same): they are the root's two best children and their scores differ
    by `gap` (up to the softmax normalisation, which moves both alike)."""
    cfg = wl.CONFIGS["tiny"]
    w = {n: t.clone() for n, t in wl.make_weights(cfg).items()}
    inp = wl.make_inputs(cfg, batch=1)
    lg = inp["logits"][0]
    a, b = 17, 911
    lg[0, :] = lg[0, :].clamp(max=5.0)
    lg[0, a] = 20.0
    lg[0, b] = 20.0 - gap
    w["corr_w2"][b] = w["corr_w2"][a]
    worc = oracle.Weights.from_dict(w)
    hid = oracle.to_numpy(inp["hidden"])[0]
    root, rpos = int(inp["root_tokens"][0]), int(inp["root_positions"][0])
    return cfg, worc, hid, root, rpos, lg, inp, a, b


def _tree_B2(gap):
    cfg, worc, hid, root, rpos, lg, inp, a, b = _setup(gap)
    tr = oracle.build_tree(worc, lg, inp["hidden"][0], root, rpos, M, 2, K, T)
    assert list(tr.tokens[:3]) == [root, a, b], tr.tokens
    assert abs((tr.scores[1] - tr.scores[2]) - gap) < 0.2 * gap
    return cfg, worc, hid, root, rpos, tr


def _as_gpu(tr):
    return {"tokens": tr.tokens.copy(), "parents": tr.parents.copy(), "depths": tr.depths.copy(),
            "positions": tr.positions.copy(), "scores": tr.scores.astype(np.float32).copy(), "mask": tr.mask.copy(),
            "n_nodes": np.int32(tr.n_nodes)}


def _cmp(gpu, tr, cfg, worc, hid, root, rpos, B, tol=1e-5):
    return compare_tree(gpu, tr, worc, hid, root, rpos, cfg.L, B, K, T, tol)


def test_exact_copy_is_exact():
    cfg, worc, hid, root, rpos, tr = _tree_B2(5e-5)
    assert _cmp(_as_gpu(tr), tr, cfg, worc, hid, root, rpos, 2) == "exact"


def test_near_tie_swap_is_tolerant():
    cfg, worc, hid, root, rpos, tr = _tree_B2(5e-5)
    gpu = _as_gpu(tr)
    gpu["tokens"][[1, 2]] = gpu["tokens"][[2, 1]]
    gpu["scores"][[1, 2]] = gpu["scores"][[2, 1]]
    assert _cmp(gpu, tr, cfg, worc, hid, root, rpos, 2) == "tolerant"


def test_swap_beyond_the_margin_raises():
    cfg, worc, hid, root, rpos, tr = _tree_B2(2e-4)
    gpu = _as_gpu(tr)
    gpu["tokens"][[1, 2]] = gpu["tokens"][[2, 1]]
    gpu["scores"][[1, 2]] = gpu["scores"][[2, 1]]
    with pytest.raises(AssertionError, match="pop order"):
        _cmp(gpu, tr, cfg, worc, hid, root, rpos, 2)


def test_missing_oracle_node_and_node_below_the_budget_raise():
    """The second node is replaced by the root's third-best child (more than 1e-4 worse): the oracle's node is missing
    and the intruder lies below the B-th score."""
    cfg, worc, hid, root, rpos, tr = _tree_B2(5e-5)
    third = int(tr.cand_ids[0][2])                             # third-best base logit of depth 1: ~15 nats below the pair
    gpu = _as_gpu(tr)
    gpu["tokens"][2] = third
    with pytest.raises(AssertionError):
        _cmp(gpu, tr, cfg, worc, hid, root, rpos, 2)


def test_score_error_raises_on_both_branches():
    cfg, worc, hid, root, rpos, tr = _tree_B2(5e-5)
    gpu = _as_gpu(tr)
    gpu["scores"][1] += 3e-3
    with pytest.raises(AssertionError, match="score error"):
        _cmp(gpu, tr, cfg, worc, hid, root, rpos, 2, tol=2e-3)
    gpu = _as_gpu(tr)
    gpu["tokens"][[1, 2]] = gpu["tokens"][[2, 1]]          # tolerant branch, scores NOT swapped: off by the gap only
    gpu["scores"][2] += 3e-3
    with pytest.raises(AssertionError, match="score error"):
        _cmp(gpu, tr, cfg, worc, hid, root, rpos, 2, tol=2e-3)


def test_broken_structure_raises():
    cfg, worc, hid, root, rpos, lg, inp, a, b = _setup(5e-5)
    tr = oracle.build_tree(worc, lg, inp["hidden"][0], root, rpos, M, 8, K, T)
    for field, edit in (("parents", lambda g: g["parents"].__setitem__(3, 5)),
                        ("mask", lambda g: g["mask"].__setitem__((4, 0), 0)),
                        ("positions", lambda g: g["positions"].__setitem__(2, g["positions"][2] + 1)),
                        ("depths", lambda g: g["depths"].__setitem__(5, g["depths"][5] + 1))):
        gpu = _as_gpu(tr)
        edit(gpu)
        with pytest.raises(AssertionError):
            _cmp(gpu, tr, cfg, worc, hid, root, rpos, 8)


def test_duplicate_node_raises():
    cfg, worc, hid, root, rpos, tr = _tree_B2(5e-5)
    gpu = _as_gpu(tr)
    gpu["tokens"][2] = gpu["tokens"][1]
    with pytest.raises(AssertionError):
        _cmp(gpu, tr, cfg, worc, hid, root, rpos, 2)
