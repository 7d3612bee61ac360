"""Factorized scorer arms of the paper's conditioning ladder -- TEST INFRASTRUCTURE ONLY (rules of oracle/__init__.py).

PAPER.md:553-555 (Appendix D, "The three arms"): all arms build the same best-first tree (Alg. 1 heap,
PAPER.md:145-149); they differ only in the children function.
  * Marg: scores from the base logits alone, the correction ignored; the menu at depth d is
    computed once and shared by every node at that depth.
  * Cond-static: the correction is applied once per depth, along the single greedy trajectory that
    Domino's own decoder walks; the corrected menu is then shared by every node at that depth.
Both are "factorized": g(u) = sum_d menu[d][rank_d].  Written step by step in float64 on top of the C oracle's
select / GRU cell / CHILDREN primitives and a linear-scan heap; no code is shared with the CUDA path.

Readings where the paper is silent (same as DESIGN.md section 2): log-probabilities are the log-softmax over the
depth's top-M slice of (logit [+ correction]) / T_eff (A1); the greedy trajectory takes the top-1 entry of the corrected
slice under (logp desc, token asc) -- with M = V that is Domino's full-vocabulary argmax; heap order (g desc, token
asc, parent slot asc) (A8); output conventions A10.
"""
from __future__ import annotations

from typing import List, Tuple

import numpy as np

import oracle

Menu = List[Tuple[np.ndarray, np.ndarray]]          # per depth: (tokens[k] int, logp[k] float64)


def _top_k(tokens: np.ndarray, lp: np.ndarray, k: int):
    order = sorted(range(len(tokens)), key=lambda m: (-lp[m], int(tokens[m])))[:k]
    return np.asarray([tokens[m] for m in order], np.int64), np.asarray([lp[m] for m in order], np.float64)


def marg_menus(logits, M: int, k: int, temperature: float) -> Menu:
    """per depth, log-softmax over the top-M slice of the base logits / T_eff, top-k."""
    logits = oracle.to_numpy(logits)
    T_eff = 1.0 if temperature == 0 else float(temperature)
    out = []
    for i in range(logits.shape[0]):
        cand, base = oracle.select_topm(logits[i], M)
        z = base / T_eff
        zmax = z.max()
        lp = (z - zmax) - np.log(np.exp(z - zmax).sum())
        out.append(_top_k(cand, lp, k))
    return out


def cond_static_menus(w: "oracle.Weights", logits, hidden, root_token: int, M: int, k: int, temperature: float) -> Menu:
    """CHILDREN along Domino's greedy chain: S_0 = GRU(0, E[root]); menu_d = CHILDREN(S_{d-1}, d);
    S_d = GRU(S_{d-1}, E[top-1 of menu_d])."""
    logits = oracle.to_numpy(logits); hidden = oracle.to_numpy(hidden)
    T_eff = 1.0 if temperature == 0 else float(temperature)
    S = oracle.gru_cell(w, np.zeros(w.g), int(root_token))
    out = []
    for i in range(logits.shape[0]):
        cand, base = oracle.select_topm(logits[i], M)
        tok, lp, _ = oracle.children(w, hidden[i], S, cand, base, k, T_eff)
        out.append((np.asarray(tok, np.int64), np.asarray(lp, np.float64)))
        S = oracle.gru_cell(w, S, int(tok[0]))
    return out


def factorized_tree(menus: Menu, root_token: int, root_pos: int, B: int):
    """Alg. 1 with a path-independent children function: linear-scan max heap, pop order =
    slot order; returns (tokens, parents, depths, positions, scores, mask, n_nodes) with the A10 conventions."""
    L = len(menus)
    N = B + 1
    tokens = np.zeros(N, np.int64); parents = np.zeros(N, np.int64); depths = np.ones(N, np.int64)
    scores = np.full(N, -np.inf); mask = np.zeros((N, N), np.uint8)
    tokens[0], parents[0], depths[0], scores[0] = root_token, -1, 0, 0.0
    heap = []                                                    # (g, token, parent slot, depth)
    def push_children(slot):
        d = int(depths[slot])
        if d < L:
            tk, lp = menus[d]
            for j in range(len(tk)):
                heap.append((scores[slot] + lp[j], int(tk[j]), slot, d + 1))
    push_children(0)
    n = 0
    while n < B and heap:
        bi = max(range(len(heap)), key=lambda i: (heap[i][0], -heap[i][1], -heap[i][2]))
        g, tok, par, dep = heap.pop(bi)
        n += 1
        tokens[n], parents[n], depths[n], scores[n] = tok, par, dep, g
        push_children(n)
    for i in range(N):
        if i > n:
            parents[i], tokens[i] = 0, 0
            mask[i, 0] = mask[i, i] = 1
            continue
        a = i
        while a >= 0:
            mask[i, a] = 1
            a = int(parents[a])
    positions = root_pos + depths
    return tokens, parents, depths, positions, scores, mask, n + 1
