"""Tolerant comparator: CUDA tree vs oracle tree (BASELINE.json north_star).

Bar: tokens / parents / depths / mask must match the oracle exactly, except where two oracle
scores differ by < 1e-4 (either order accepted); node log-scores within `score_tol` absolute.
When the trees are not bit-equal, every GPU node is re-scored along its own path by the ORACLE
(`oracle.score_path`) and the set / order conditions are checked against those float64 scores.
Test infrastructure only: imports the oracle, never the CUDA binding.
"""
from __future__ import annotations

import numpy as np

import oracle

MARGIN = 1e-4


def structure_errors(tokens, parents, depths, positions, mask, n_nodes, root_token, root_pos, L, B):
    """Invariants every output must satisfy (reading A10)."""
    errs = []
    N = B + 1
    if not (1 <= n_nodes <= N):
        return [f"n_nodes {n_nodes} out of range"]
    if tokens[0] != root_token or parents[0] != -1 or depths[0] != 0:
        errs.append("bad root slot")
    for i in range(1, N):
        if i < n_nodes:
            p = parents[i]
            if not (0 <= p < i):
                errs.append(f"slot {i}: parent {p} not earlier in pop order")
                continue
            if depths[i] != depths[p] + 1 or not (1 <= depths[i] <= L):
                errs.append(f"slot {i}: depth {depths[i]} vs parent depth {depths[p]}")
        else:  # dead leaf
            if tokens[i] != 0 or parents[i] != 0 or depths[i] != 1:
                errs.append(f"slot {i}: dead leaf malformed")
    if not np.array_equal(positions, root_pos + depths):
        errs.append("positions != root_pos + depth")
    want = np.zeros((N, N), np.uint8)
    for i in range(N):
        a = i
        while a >= 0:
            want[i, a] = 1
            a = parents[a] if a > 0 else -1
    if not np.array_equal(mask, want):
        errs.append("mask is not the ancestor-or-self closure")
    return errs


def _path(tokens, parents, slot):
    out = []
    while slot > 0:
        out.append(int(tokens[slot]))
        slot = int(parents[slot])
    return tuple(out[::-1])


def compare_tree(gpu: dict, orc: "oracle.Tree", w: "oracle.Weights", hidden, root_token: int, root_pos: int,
                 L: int, B: int, k: int, temperature: float, score_tol: float) -> str:
    """Returns "exact" or "tolerant"; raises AssertionError otherwise.  `gpu` holds numpy arrays of
    ONE request: tokens, parents, depths, positions, scores, mask, n_nodes."""
    tk, pa, de, po, sc, mk = (np.asarray(gpu[x]) for x in
                              ("tokens", "parents", "depths", "positions", "scores", "mask"))
    nn = int(gpu["n_nodes"])
    errs = structure_errors(tk, pa, de, po, mk, nn, root_token, root_pos, L, B)
    assert not errs, errs
    exact = (nn == orc.n_nodes and np.array_equal(tk, orc.tokens) and np.array_equal(pa, orc.parents)
             and np.array_equal(de, orc.depths) and np.array_equal(mk, orc.mask)
             and np.array_equal(po, orc.positions))
    if exact:
        diff = np.abs(sc[:nn].astype(np.float64) - orc.scores[:nn])
        diff = diff[np.isfinite(orc.scores[:nn])]
        assert diff.size == 0 or diff.max() <= score_tol, f"score error {diff.max():.3e} > {score_tol}"
        assert np.all(np.isneginf(sc[nn:]))
        return "exact"

    # ---- tolerant path -------------------------------------------------------------------------
    assert nn == orc.n_nodes, f"n_nodes {nn} vs oracle {orc.n_nodes}"
    gstar = np.zeros(nn)
    gpu_paths = {}
    for s in range(1, nn):
        path = _path(tk, pa, s)
        lp, rank, kth = oracle.score_path(w, hidden, root_token, orc.cand_ids, orc.cand_vals, k, temperature, path)
        assert not np.any(np.isnan(lp)), f"slot {s}: token outside its depth's candidate set"
        assert np.all(lp >= kth - MARGIN), f"slot {s}: token not within {MARGIN} of its parent's k-th best child"
        gstar[s] = lp.sum()
        gpu_paths[path] = s
    assert len(gpu_paths) == nn - 1, "duplicate node in GPU tree"
    g_last = orc.scores[orc.n_nodes - 1]
    assert np.all(gstar[1:] >= g_last - MARGIN), "GPU node scores below the oracle's B-th score by more than margin"
    for s in range(1, orc.n_nodes):
        if orc.scores[s] > g_last + MARGIN:
            assert tuple(orc.path(s)) in gpu_paths, f"oracle node {s} (score {orc.scores[s]:.6f}) missing from GPU tree"
    d = np.diff(gstar[1:])
    assert np.all(d <= MARGIN), "GPU pop order not non-increasing in oracle score (beyond margin)"
    err = np.abs(sc[1:nn].astype(np.float64) - gstar[1:])
    assert err.size == 0 or err.max() <= score_tol, f"score error {err.max():.3e} > {score_tol}"
    return "tolerant"


def tree_to_numpy(tb, b: int) -> dict:
    """Slice request b out of a binding TreeBatch (torch tensors, any device) as numpy arrays."""
    return {n: getattr(tb, n)[b].detach().cpu().numpy() for n in
            ("tokens", "parents", "depths", "positions", "scores", "mask", "n_nodes")}
