"""Longest-accepted-path commit: oracle pins (CPU) and GPU parity."""
import itertools
import os
import sys

import numpy as np
import pytest
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from oracle.commit import commit_path  # noqa: E402


def _random_tree(rng, n, L, k):
    """A prefix-closed tree in pop order: parents precede children, sibling tokens distinct, scores decreasing."""
    tokens, parents, depths, scores = [int(rng.integers(0, 50))], [-1], [0], [0.0]
    for _ in range(40 * n):                                  # bounded: a full tree (k^L nodes) cannot grow further
        if len(tokens) >= n:
            break
        par = int(rng.integers(0, len(tokens)))
        if depths[par] >= L:
            continue
        sib = {tokens[i] for i in range(len(tokens)) if parents[i] == par}
        if len(sib) >= k:
            continue
        tok = int(rng.integers(0, 50))
        if tok in sib:
            continue
        tokens.append(tok); parents.append(par); depths.append(depths[par] + 1)
        scores.append(scores[par] - float(rng.random()) - 1e-3)
    return tokens, parents, depths, scores


def _dfs_longest(tokens, parents, depths, scores, n, accepted):
    """Independent formulation: top-down DFS over the children lists, only through accepted edges."""
    kids = {i: [] for i in range(n)}
    for i in range(1, n):
        kids[parents[i]].append(i)
    best = [0]

    def go(u):
        if (depths[u], scores[u], -u) > (depths[best[0]], scores[best[0]], -best[0]):
            best[0] = u
        for c in kids[u]:
            if accepted(c):
                go(c)
    go(0)
    return best[0]


def test_oracle_chain_accepts_exactly_the_matching_prefix():
    # a pure chain 0 -> 1 -> ... -> 6 (PAPER.md:82 Domino's chain): the target agrees with the first j drafts
    L = 6
    tokens = [7, 11, 12, 13, 14, 15, 16]
    parents = [-1, 0, 1, 2, 3, 4, 5]
    depths = list(range(L + 1))
    scores = [-0.1 * i for i in range(L + 1)]
    for j in range(L + 1):
        nxt = [tokens[i + 1] if i < j and i + 1 <= L else 999 for i in range(L + 1)]
        ln, path, bonus = commit_path(tokens, parents, depths, scores, L + 1, target_next=nxt)
        assert ln == j and path == list(range(j + 1)) and bonus == nxt[j]


def test_oracle_hand_worked_tree():
    # root(0) -> a(1: tok 5), b(2: tok 6); a -> c(3: tok 8), d(4: tok 9); b -> e(5: tok 8)
    tokens, parents, depths = [1, 5, 6, 8, 9, 8], [-1, 0, 0, 1, 1, 2], [0, 1, 1, 2, 2, 2]
    scores = [0.0, -0.2, -0.5, -0.3, -0.9, -0.6]
    # target: after root says 5 (accept a), after a says 9 (accept d), after d says 3
    ln, path, bonus = commit_path(tokens, parents, depths, scores, 6, target_next=[5, 9, 8, 0, 3, 0])
    assert (ln, path, bonus) == (2, [0, 1, 4], 3)
    # target: after root says 6 (accept b), after b says 7 (no child): e is NOT reached although tok 8 == next[a]
    ln, path, bonus = commit_path(tokens, parents, depths, scores, 6, target_next=[6, 8, 7, 0, 0, 0])
    assert (ln, path, bonus) == (1, [0, 2], 7)
    # nothing accepted
    assert commit_path(tokens, parents, depths, scores, 6, target_next=[4, 0, 0, 0, 0, 0]) == (0, [0], 4)
    # edge flags: c and e both reachable at depth 2 -> higher draft score (c) wins
    ln, path, _ = commit_path(tokens, parents, depths, scores, 6, edge_ok=[0, 1, 1, 1, 0, 1])
    assert (ln, path) == (2, [0, 1, 3])
    # a padding slot (index >= n_nodes) is never reachable
    ln, path, _ = commit_path(tokens, parents, depths, scores, 5, edge_ok=[0, 0, 1, 1, 1, 1])
    assert (ln, path) == (1, [0, 2])


@pytest.mark.parametrize("seed", range(6))
def test_oracle_matches_independent_dfs_and_invariants(seed):
    rng = np.random.default_rng(100 + seed)
    for _ in range(40):
        n, L, k = int(rng.integers(1, 40)), int(rng.integers(1, 7)), int(rng.integers(1, 5))
        tokens, parents, depths, scores = _random_tree(rng, n, L, k)
        n = len(tokens)
        # greedy mode: the target mostly agrees with one child
        nxt = []
        for u in range(n):
            kids = [i for i in range(n) if parents[i] == u]
            nxt.append(tokens[int(rng.choice(kids))] if kids and rng.random() < 0.7 else int(rng.integers(50, 60)))
        ln, path, bonus = commit_path(tokens, parents, depths, scores, n, target_next=nxt)
        end = _dfs_longest(tokens, parents, depths, scores, n, lambda c: tokens[c] == nxt[parents[c]])
        assert path[-1] == end and ln == depths[end] == len(path) - 1 and path[0] == 0 and bonus == nxt[end]
        assert all(parents[path[i + 1]] == path[i] and tokens[path[i + 1]] == nxt[path[i]] for i in range(ln))
        assert all(tokens[c] != nxt[end] for c in range(n) if parents[c] == end)      # cannot be extended
        # flag mode
        ok = [0] + [int(rng.random() < 0.6) for _ in range(n - 1)]
        ln, path, bonus = commit_path(tokens, parents, depths, scores, n, edge_ok=ok)
        end = _dfs_longest(tokens, parents, depths, scores, n, lambda c: ok[c])
        assert path[-1] == end and ln == depths[end] and bonus == -1


def test_oracle_brute_force_over_all_flag_patterns():
    # every acceptance pattern of a 6-node tree: the result is the deepest node whose whole root path is accepted
    tokens, parents, depths = [1, 5, 6, 8, 9, 8], [-1, 0, 0, 1, 1, 2], [0, 1, 1, 2, 2, 2]
    scores = [0.0, -0.2, -0.5, -0.3, -0.9, -0.6]
    for bits in itertools.product([0, 1], repeat=5):
        ok = [0] + list(bits)
        reach = [True] + [False] * 5
        for i in range(1, 6):
            reach[i] = bool(ok[i]) and reach[parents[i]]
        cand = [i for i in range(6) if reach[i]]
        want = max(cand, key=lambda i: (depths[i], scores[i], -i))
        ln, path, _ = commit_path(tokens, parents, depths, scores, 6, edge_ok=ok)
        assert path[-1] == want and ln == depths[want]


@pytest.mark.gpu
@pytest.mark.parametrize("mode", ["target_next", "edge_ok"])
def test_gpu_commit_matches_oracle_on_built_trees(mode):
    """Trees built by the CUDA path (tiny config, several budgets), acceptance drawn at random around the tree."""
    import gpu_util as gu
    from paper_2607_08642_b200 import workloads as wl
    case = gu.tiny_case()
    rng = np.random.default_rng(7)
    for B, batch in ((8, 5), (31, 32), (64, 3)):
        inp = wl.make_inputs(case.cfg, batch=batch, seed=4000 + B)
        out = case.run_gpu(inp, 8, B, 0.0)
        torch.cuda.synchronize()
        tok, par = out.tokens.cpu().numpy(), out.parents.cpu().numpy()
        dep, sco, nn = out.depths.cpu().numpy(), out.scores.cpu().numpy(), out.n_nodes.cpu().numpy()
        N = B + 1
        if mode == "target_next":
            nxt = np.zeros((batch, N), dtype=np.int32)
            for b in range(batch):
                for u in range(N):
                    kids = [i for i in range(int(nn[b])) if par[b, i] == u and i != 0]
                    nxt[b, u] = tok[b, int(rng.choice(kids))] if kids and rng.random() < 0.75 else -5
            acc, path, bonus = case.builder.commit_paths(out, B, target_next=torch.from_numpy(nxt).cuda())
        else:
            ok = (rng.random((batch, N)) < 0.6).astype(np.uint8)
            acc, path, bonus = case.builder.commit_paths(out, B, edge_ok=torch.from_numpy(ok).cuda())
        torch.cuda.synchronize()
        acc, path, bonus = acc.cpu().numpy(), path.cpu().numpy(), bonus.cpu().numpy()
        L = case.cfg.L
        for b in range(batch):
            kw = dict(target_next=nxt[b].tolist()) if mode == "target_next" else dict(edge_ok=ok[b].tolist())
            ln, p, bo = commit_path(tok[b].tolist(), par[b].tolist(), dep[b].tolist(), sco[b].tolist(), int(nn[b]), **kw)
            assert int(acc[b]) == ln and path[b, :ln + 1].tolist() == p and (path[b, ln + 1:] == -1).all()
            assert path.shape[1] == L + 1 and int(bonus[b]) == bo


@pytest.mark.gpu
def test_gpu_commit_argument_validation():
    import gpu_util as gu
    from paper_2607_08642_b200 import workloads as wl
    import paper_2607_08642_b200 as dtb
    case = gu.tiny_case()
    inp = wl.make_inputs(case.cfg, batch=2)
    out = case.run_gpu(inp, 8, 8, 0.0)
    with pytest.raises(dtb.DominoTreeError):
        case.builder.commit_paths(out, 8)                       # neither acceptance input
    z = torch.zeros((2, 9), dtype=torch.int32, device="cuda")
    with pytest.raises(dtb.DominoTreeError):
        case.builder.commit_paths(out, 8, target_next=z, edge_ok=z.to(torch.uint8))
