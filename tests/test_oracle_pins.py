"""Pins for the float64 CPU oracle (oracle/dominotree_oracle.c) against what the paper and the
mathematics fix -- none of them re-types the oracle's own formula or re-calls its own routine:

* library routines (torch.nn.GRUCell(bias=False), F.silu, F.linear, torch.log_softmax, stable sort)
* zero-correction reduction to DDTree's factorized best-first tree
* k=1 reduction to Domino's greedy chain over the FULL vocabulary
* brute force: best-first == the B highest-scoring nodes of the candidate tree
* exhaustive prefix-closed subtrees maximise Phi(n) = sum exp(g)
* candidate restriction M = V equals the unrestricted scorer
* structural invariants of the output
"""
import heapq
import itertools
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2607_08642_b200 import workloads as wl
from ref_torch import TorchRef, order_desc


def _setup(cfg, regime="flat", seed=None, batch=None, embed_std=None):
    if embed_std is not None:
        cfg = cfg.replace(embed_std=embed_std)
    w = wl.make_weights(cfg, seed)
    x = wl.make_inputs(cfg, batch=batch, seed=seed, regime=regime)
    return cfg, w, x, oracle.Weights.from_dict(w)


def _tree(cfg, ow, x, b=0, **kw):
    args = dict(M=cfg.M, B=cfg.B, k=cfg.k, temperature=cfg.T)
    args.update(kw)
    return oracle.build_tree(ow, x["logits"][b], x["hidden"][b], int(x["root_tokens"][b]),
                             int(x["root_positions"][b]), **args)


# ----------------------------------------------------------------------------- library pins
def test_select_matches_stable_library_sort():
    gen = torch.Generator().manual_seed(1)
    for V, M in [(1024, 8), (1000, 64), (16, 16), (4097, 128)]:
        row = torch.randn(V, generator=gen).mul(3).to(torch.bfloat16)    # bf16 => many exact ties
        ids, vals = oracle.select_topm(row, M)
        ref = torch.sort(row.double(), descending=True, stable=True)     # stable => token asc among ties
        assert np.array_equal(ids, ref.indices[:M].numpy().astype(np.int32))
        assert np.array_equal(vals, ref.values[:M].numpy())


def test_select_adversarial_rows():
    for name, row in wl.adversarial_select_rows(2048, torch.bfloat16).items():
        ids, vals = oracle.select_topm(row, 64)
        ref = torch.sort(row.double(), descending=True, stable=True)
        assert np.array_equal(ids, ref.indices[:64].numpy().astype(np.int32)), name
        assert np.array_equal(vals, ref.values[:64].numpy()), name


@pytest.mark.parametrize("cfgname", ["tiny", "brute"])
def test_gru_cell_matches_torch_grucell(cfgname):
    cfg, w, x, ow = _setup(wl.CONFIGS[cfgname], embed_std=1.0)
    ref = TorchRef(w)
    gen = torch.Generator().manual_seed(2)
    h = torch.randn(cfg.g, generator=gen, dtype=torch.float64)
    for tok in [0, 3, cfg.V - 1]:
        got = oracle.gru_cell(ow, h.numpy(), tok)
        want = ref.advance(h, tok).numpy()
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-14)
        h = torch.from_numpy(got)
    # S_0 from the zero state (A4)
    np.testing.assert_allclose(oracle.gru_cell(ow, np.zeros(cfg.g), 5), ref.s0(5).numpy(), atol=1e-15)


def test_gru_cell_bf16_weights_widened_exactly():
    cfg = wl.CONFIGS["tiny"].replace(dtype="bf16", embed_std=1.0)
    w = wl.make_weights(cfg)
    ow = oracle.Weights.from_dict(w)
    ref = TorchRef(w)
    h = torch.linspace(-1, 1, cfg.g, dtype=torch.float64)
    np.testing.assert_allclose(oracle.gru_cell(ow, h.numpy(), 7), ref.advance(h, 7).numpy(), atol=1e-14)


@pytest.mark.parametrize("T_eff", [1.0, 0.6])
def test_children_match_library_correction_and_log_softmax(T_eff):
    """dL = W2 SiLU(W1 [H; S]) on the slice, log-softmax over the slice, top-k (value desc, token asc)."""
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"], embed_std=1.0)
    ref = TorchRef(w)
    S = ref.s0(int(x["root_tokens"][0]))
    for i in range(cfg.L):
        row = x["logits"][0, i]
        ids, vals = oracle.select_topm(row, cfg.M)
        tok, lp, allp = oracle.children(ow, x["hidden"][0, i], S.numpy(), ids, vals, cfg.k, T_eff)
        want = ref.slice_logprobs(row, x["hidden"][0, i], S, torch.from_numpy(ids), T_eff)
        np.testing.assert_allclose(allp, want.numpy(), atol=1e-12)
        assert abs(np.exp(allp).sum() - 1.0) < 1e-12
        o = order_desc(want, torch.from_numpy(ids).long())[: cfg.k]
        assert np.array_equal(tok, ids[o.numpy()])
        np.testing.assert_allclose(lp, want[o].numpy(), atol=1e-12)
        S = ref.advance(S, int(tok[0]))


def test_restriction_with_M_equal_V_is_the_unrestricted_scorer():
    """restriction only shrinks the operand; with M=V it is softmax(L_base + dL) over V."""
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"].replace(V=64, M=64, k=8), embed_std=1.0)
    ref = TorchRef(w)
    S = ref.s0(int(x["root_tokens"][0]))
    row = x["logits"][0, 1]
    ids, vals = oracle.select_topm(row, cfg.V)
    _, _, allp = oracle.children(ow, x["hidden"][0, 1], S.numpy(), ids, vals, cfg.k)
    full = torch.log_softmax(ref.corrected_logits(row, x["hidden"][0, 1], S), dim=0)
    np.testing.assert_allclose(allp, full[torch.from_numpy(ids).long()].numpy(), atol=1e-12)


# ----------------------------------------------------------------------------- DDTree reduction
def _ddtree_factorized(table_lp, table_tok, B, k, L):
    """Independent best-first tree over a factorized table (DDTree): heapq keyed by
    (-g, token, parent)."""
    heap, out = [], []
    for c in range(k):
        heapq.heappush(heap, (-table_lp[0][c], int(table_tok[0][c]), 0, 1))
    while len(out) < B and heap:
        ng, tok, par, dep = heapq.heappop(heap)
        out.append((tok, par, dep, -ng))
        slot = len(out)
        if dep < L:
            for c in range(k):
                heapq.heappush(heap, (ng - table_lp[dep][c], int(table_tok[dep][c]), slot, dep + 1))
    return out


@pytest.mark.parametrize("zero", ["W2", "W1"])
@pytest.mark.parametrize("regime", ["flat", "peaked"])
def test_zero_correction_reduces_to_ddtree(zero, regime):
    cfg = wl.CONFIGS["tiny"].replace(B=24, k=4)
    cfg, w, x, _ = _setup(cfg, regime=regime)
    if zero == "W2":
        w["corr_w2"].zero_()
    else:
        w["corr_w1"].zero_()           # SiLU(0) = 0
    ow = oracle.Weights.from_dict(w)
    t = _tree(cfg, ow, x)
    # factorized table: log-softmax of the raw top-M logits per depth (reading A1), via library calls
    tab_lp, tab_tok = [], []
    for i in range(cfg.L):
        srt = torch.sort(x["logits"][0, i].double(), descending=True, stable=True)
        lp = torch.log_softmax(srt.values[: cfg.M], dim=0)
        tab_lp.append(lp[: cfg.k].tolist())
        tab_tok.append(srt.indices[: cfg.k].tolist())
    want = _ddtree_factorized(tab_lp, tab_tok, cfg.B, cfg.k, cfg.L)
    assert t.n_nodes == len(want) + 1
    for s, (tok, par, dep, g) in enumerate(want, start=1):
        assert (int(t.tokens[s]), int(t.parents[s]), int(t.depths[s])) == (tok, par, dep)
        assert abs(t.scores[s] - g) < 1e-12
    # closed form: every node's g is a sum of per-depth table entries; the result is the top-B of all sums
    sums = []
    for dep in range(1, cfg.L + 1):
        for ranks in itertools.product(range(cfg.k), repeat=dep):
            sums.append(sum(tab_lp[i][rk] for i, rk in enumerate(ranks)))
    sums.sort(reverse=True)
    np.testing.assert_allclose(t.scores[1: cfg.B + 1], sums[: cfg.B], atol=1e-12)


# ----------------------------------------------------------------------------- chain reduction
def test_k1_reduces_to_domino_greedy_chain_over_full_vocab():
    """k=1, B=L, M=V: one token per position, one GRU state (Fact A); the token at
    position i is argmax over the FULL vocabulary of L_i^base + dL_i."""
    cfg = wl.CONFIGS["tiny"].replace(V=256, M=256, k=1, B=4)
    cfg, w, x, ow = _setup(cfg, embed_std=1.0)
    ref = TorchRef(w)
    t = _tree(cfg, ow, x)
    S = ref.s0(int(x["root_tokens"][0]))
    g = 0.0
    assert t.n_nodes == cfg.L + 1
    for i in range(cfg.L):
        full = ref.corrected_logits(x["logits"][0, i], x["hidden"][0, i], S)
        tok = int(torch.argmax(full))
        g += float(torch.log_softmax(full, dim=0)[tok])
        assert int(t.tokens[i + 1]) == tok and int(t.parents[i + 1]) == i and int(t.depths[i + 1]) == i + 1
        assert abs(t.scores[i + 1] - g) < 1e-12
        S = ref.advance(S, tok)


def test_M1_degenerate_chain_all_scores_zero():
    """Literal 'M=1': a slice of one => every logp = 0 => marginal-argmax chain, all scores 0."""
    cfg = wl.CONFIGS["tiny"].replace(M=1, k=1, B=4)
    cfg, w, x, ow = _setup(cfg)
    t = _tree(cfg, ow, x)
    for i in range(cfg.L):
        assert int(t.tokens[i + 1]) == int(torch.argmax(x["logits"][0, i].double()))
        assert t.scores[i + 1] == 0.0
    assert t.n_nodes == cfg.L + 1


# ----------------------------------------------------------------------------- brute force
def _enumerate_candidate_tree(ref, x, cand, k, L, T_eff=1.0):
    """Every node of the k-ary depth-L candidate tree with its path score, scored with library ops."""
    nodes = []   # (g, path tuple)

    def rec(S, path, g):
        i = len(path)
        if i == L:
            return
        ids = cand[i]
        lp = ref.slice_logprobs(x["logits"][0, i], x["hidden"][0, i], S, torch.from_numpy(ids), T_eff)
        o = order_desc(lp, torch.from_numpy(ids).long())[:k]
        for j in o.tolist():
            tok = int(ids[j])
            gg = g + float(lp[j])
            nodes.append((gg, path + (tok,)))
            rec(ref.advance(S, tok), path + (tok,), gg)

    rec(ref.s0(int(x["root_tokens"][0])), (), 0.0)
    return nodes


@pytest.mark.parametrize("k,L,B", [(16, 3, 8), (4, 4, 20), (3, 4, 40)])
def test_bruteforce_best_first_is_top_B_of_candidate_tree(k, L, B):
    cfg = wl.CONFIGS["brute"].replace(k=k, L=L, B=B)
    cfg, w, x, ow = _setup(cfg, embed_std=1.0)
    ref = TorchRef(w)
    t = _tree(cfg, ow, x)
    nodes = _enumerate_candidate_tree(ref, x, t.cand_ids, k, L)
    nodes.sort(key=lambda n: -n[0])
    gaps = np.diff([n[0] for n in nodes[: B + 1]])
    assert np.all(gaps < -1e-9), "inputs must be tie-free for this pin"
    assert t.n_nodes == B + 1
    for s in range(1, B + 1):
        assert tuple(t.path(s)) == nodes[s - 1][1]
        assert abs(t.scores[s] - nodes[s - 1][0]) < 1e-10


def test_exhaustive_prefix_closed_subtrees_maximise_phi():
    """Micro size: enumerate EVERY prefix-closed subtree with B nodes; ours maximises sum exp(g)."""
    k, L, B = 3, 3, 5
    cfg = wl.CONFIGS["brute"].replace(k=k, L=L, B=B)
    cfg, w, x, ow = _setup(cfg, embed_std=1.0)
    ref = TorchRef(w)
    t = _tree(cfg, ow, x)
    nodes = _enumerate_candidate_tree(ref, x, t.cand_ids, k, L)
    score = {p: g for g, p in nodes}
    paths = list(score)
    best = -1.0
    for sub in itertools.combinations(paths, B):
        s = set(sub)
        if all(len(p) == 1 or p[:-1] in s for p in sub):
            best = max(best, sum(math.exp(score[p]) for p in sub))
    ours = sum(math.exp(t.scores[s]) for s in range(1, B + 1))
    assert abs(ours - best) < 1e-12


# ----------------------------------------------------------------------------- invariants
def _check_invariants(t, cfg, root_token, root_pos):
    N = cfg.B + 1
    n = t.n_nodes
    assert t.tokens[0] == root_token and t.parents[0] == -1 and t.depths[0] == 0 and t.scores[0] == 0
    for s in range(1, n):
        p = int(t.parents[s])
        assert 0 <= p < s                                        # parents precede children
        assert t.depths[s] == t.depths[p] + 1 <= cfg.L
        assert t.scores[s] <= t.scores[p] + 1e-15                 # child <= parent
        if s > 1:
            assert t.scores[s] <= t.scores[s - 1] + 1e-15         # pop order non-increasing
        assert t.tokens[s] in t.cand_ids[t.depths[s] - 1]
    assert np.array_equal(t.positions, root_pos + t.depths)
    for s in range(N):
        row = t.mask[s]
        assert row[s] == 1 and not row[s + 1:].any()              # lower-triangular
        anc, a = set(), s
        while a >= 0:
            anc.add(a)
            a = int(t.parents[a])
        assert set(np.nonzero(row)[0].tolist()) == anc             # ancestor closure
        assert row.sum() == t.depths[s] + 1
    sib = {}
    for s in range(1, n):
        key = (int(t.parents[s]), int(t.tokens[s]))
        assert key not in sib
        sib[key] = s
    for s in range(n, N):                                          # dead leaves (A10)
        assert (t.tokens[s], t.parents[s], t.depths[s]) == (0, 0, 1) and t.scores[s] == -np.inf
    assert np.all(t.res_score <= t.scores[n - 1] + 1e-15) or n - 1 < cfg.B


@pytest.mark.parametrize("regime", ["flat", "peaked"])
@pytest.mark.parametrize("T", [0.0, 0.6, 1.0])
def test_invariants_tiny(regime, T):
    cfg = wl.CONFIGS["tiny"].replace(T=T, B=16)
    cfg, w, x, ow = _setup(cfg, regime=regime, embed_std=1.0)
    t = _tree(cfg, ow, x)
    _check_invariants(t, cfg, int(x["root_tokens"][0]), int(x["root_positions"][0]))


def test_temperature_zero_equals_one():
    """A7: T=0 is scored with T_eff=1, so T=0 and T=1 give the same tree."""
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"].replace(B=16), embed_std=1.0)
    a, b = _tree(cfg, ow, x, temperature=0.0), _tree(cfg, ow, x, temperature=1.0)
    assert np.array_equal(a.tokens, b.tokens) and np.array_equal(a.scores, b.scores)


def test_exhausted_candidate_tree_pads_dead_leaves():
    cfg = wl.CONFIGS["tiny"].replace(k=1, M=4, B=8)      # k=1, L=4 => only 4 nodes exist
    cfg, w, x, ow = _setup(cfg)
    t = _tree(cfg, ow, x)
    assert t.n_nodes == cfg.L + 1
    _check_invariants(t, cfg, int(x["root_tokens"][0]), int(x["root_positions"][0]))


def test_eager_state_advance_is_bit_identical_to_lazy():
    """PAPER.md:144 advances the GRU per child at expansion; evaluating at pop is the same function."""
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"].replace(B=12), embed_std=1.0)
    a = _tree(cfg, ow, x, eager_states=False)
    b = _tree(cfg, ow, x, eager_states=True)
    for f in ("tokens", "parents", "depths", "scores", "mask"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f


def test_score_path_agrees_with_tree_scores():
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"].replace(B=16), embed_std=1.0)
    t = _tree(cfg, ow, x)
    for s in range(1, t.n_nodes):
        lp, rk, kth = oracle.score_path(ow, x["hidden"][0], int(x["root_tokens"][0]), t.cand_ids, t.cand_vals,
                                        cfg.k, cfg.T, t.path(s))
        assert abs(lp.sum() - t.scores[s]) < 1e-12
        assert np.all(rk < cfg.k) and np.all(lp >= kth - 1e-15)


def test_vocabulary_permutation_equivariance():
    """Relabelling tokens (E, W2 rows, logits columns, root) relabels the tree and nothing else.
    Token ids only break exact ties, and the inputs here are tie-free in the scores that matter."""
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"].replace(B=16), embed_std=1.0)
    t = _tree(cfg, ow, x)
    perm = torch.randperm(cfg.V, generator=torch.Generator().manual_seed(3))   # new id -> old id
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(cfg.V)
    w2 = dict(w)
    w2["embed"] = w["embed"][perm].contiguous()
    w2["corr_w2"] = w["corr_w2"][perm].contiguous()
    x2 = dict(x)
    x2["logits"] = x["logits"][:, :, perm].contiguous()
    x2["root_tokens"] = inv[x["root_tokens"].long()].to(torch.int32)
    t2 = _tree(cfg, oracle.Weights.from_dict(w2), x2)
    assert np.array_equal(perm[torch.from_numpy(t2.tokens[1:]).long()].numpy(), t.tokens[1:])
    assert np.array_equal(t2.parents, t.parents)
    np.testing.assert_allclose(t2.scores, t.scores, atol=1e-12)


def test_path_dependence_is_exercised_in_stress_config():
    """Two same-depth nodes with different paths get different menus (Fact B);
    zeroing only the state half of W1 (a path-independent correction) builds a different tree."""
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"].replace(B=32), embed_std=1.0)
    t = _tree(cfg, ow, x)
    by_depth = {}
    for s in range(1, t.n_nodes):
        by_depth.setdefault(int(t.depths[s]), []).append(s)
    pair = next(v for d, v in sorted(by_depth.items()) if len(v) >= 2 and d < cfg.L)
    d = int(t.depths[pair[0]])
    menus = []
    for s in pair[:2]:
        S = np.zeros(cfg.g)
        S = oracle.gru_cell(ow, S, int(x["root_tokens"][0]))
        for tok in t.path(s):
            S = oracle.gru_cell(ow, S, tok)
        menus.append(oracle.children(ow, x["hidden"][0, d], S, t.cand_ids[d], t.cand_vals[d], cfg.k)[2])
    assert np.abs(menus[0] - menus[1]).max() > 1e-3
    w_static = dict(w)
    w_static["corr_w1"] = w["corr_w1"].clone()
    w_static["corr_w1"][:, cfg.d:] = 0
    t_static = _tree(cfg, oracle.Weights.from_dict(w_static), x)
    assert not (np.array_equal(t_static.tokens, t.tokens) and np.array_equal(t_static.parents, t.parents))


def test_batch_is_independent_requests():
    cfg, w, x, ow = _setup(wl.CONFIGS["tiny"], batch=3, embed_std=1.0)
    trees = oracle.build_trees(ow, x["logits"], x["hidden"], x["root_tokens"], x["root_positions"],
                               cfg.M, cfg.B, cfg.k, cfg.T, threads=3)
    for b, t in enumerate(trees):
        solo = _tree(cfg, ow, x, b=b)
        assert np.array_equal(t.tokens, solo.tokens) and np.array_equal(t.scores, solo.scores)


# ----------------------------------------------------------------------------- golden fixture
def test_golden_hand_worked_factorized_example():
    """tests/golden/ddtree_2x3.txt: a 2-depth, 3-token factorized example worked by hand."""
    import os
    rows, expect = [], []
    with open(os.path.join(os.path.dirname(__file__), "golden", "ddtree_2x3.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            kind, *vals = line.split()
            if kind == "logits":
                rows.append([float(v) for v in vals])
            elif kind == "node":
                expect.append((int(vals[0]), int(vals[1]), int(vals[2]), float(vals[3])))
    V, L = len(rows[0]), len(rows)
    cfg = wl.CONFIGS["tiny"].replace(V=V, L=L, M=V, k=V, B=len(expect))
    w = wl.make_weights(cfg)
    w["corr_w2"].zero_()
    ow = oracle.Weights.from_dict(w)
    logits = torch.tensor(rows, dtype=torch.float32)
    hidden = torch.zeros((L, cfg.d), dtype=torch.float32)
    t = oracle.build_tree(ow, logits, hidden, 0, 0, M=V, B=len(expect), k=V, temperature=0.0)
    for s, (tok, par, dep, g) in enumerate(expect, start=1):
        assert (int(t.tokens[s]), int(t.parents[s]), int(t.depths[s])) == (tok, par, dep)
        assert abs(t.scores[s] - g) < 5e-7
