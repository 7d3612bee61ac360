"""Longest-accepted-path commit over a draft tree -- TEST INFRASTRUCTURE ONLY (same rules as oracle/__init__.py).

PAPER.md:167-169 (Sec. 3.5): after one target forward pass with the ancestor-only mask has scored every tree
position, "we commit the highest-scoring root-to-leaf path along which every edge is accepted
(longest-accepted-path)".  Plain definition, written out node by node with pure-Python loops (trees have at
most 256 slots):

  * an edge (parent u -> node i) is accepted, in greedy verification, iff tokens[i] == target_next[u], the token
    the target model predicts after u; for any other acceptance rule the caller passes the
    per-edge flags edge_ok[i] directly;
  * a node is reachable iff every edge on its root path is accepted (the root always is);
  * the committed path ends at the reachable node of greatest depth; ties (possible only with edge flags:
    sibling tokens are distinct, so greedy verification accepts at most one child per node) go to the higher
    draft score ("highest-scoring"), then to the lower slot.

Readings where the paper is silent: slot 0 is the root and is always on the path; dead-leaf padding slots
(index >= n_nodes, A10) are never reachable; the bonus token is target_next at the end node.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple


def commit_path(tokens: Sequence[int], parents: Sequence[int], depths: Sequence[int], scores: Sequence[float],
                n_nodes: int, target_next: Optional[Sequence[int]] = None,
                edge_ok: Optional[Sequence[int]] = None) -> Tuple[int, List[int], int]:
    """Returns (accept_len, path slots root..end, bonus token or -1)."""
    assert (target_next is None) != (edge_ok is None)
    best = 0
    for i in range(1, n_nodes):
        # walk the root path of node i, checking every edge on it
        ok, u = True, i
        while u != 0:
            par = parents[u]
            acc = (tokens[u] == target_next[par]) if target_next is not None else bool(edge_ok[u])
            if not acc:
                ok = False
                break
            u = par
        if not ok:
            continue
        if (depths[i], scores[i], -i) > (depths[best], scores[best], -best):
            best = i
    path = []
    u = best
    while u != -1:
        path.append(u)
        u = parents[u] if u != 0 else -1
    path.reverse()
    bonus = int(target_next[best]) if target_next is not None else -1
    return int(depths[best]), path, bonus
