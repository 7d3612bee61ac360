"""ORACLE (test infrastructure, not the product): first-child / next-sibling link arrays of an emitted draft tree.

PAPER.md:169 (section 3.5) verifies "all n nodes ... in one forward pass under an ancestor-only attention mask" and
PAPER.md:187 runs the serving build on SGLang's EAGLE tree-verify kernel, which walks the tree through two arrays
instead of the mask: the first child of every node and its next sibling.  Definition written out (slots in pop order,
slot 0 = root, n_nodes valid slots, parents[i] < i):

    first_child[i]  = the smallest slot j > i with parents[j] == i, else -1
    next_sibling[i] = the smallest slot j > i with parents[j] == parents[i], else -1   (-1 for the root)

so siblings are chained in pop order (best first) and dead-leaf padding slots (reading A10) are linked nowhere (-1, -1).
Plain Python loops; shares nothing with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def tree_links(parents, n_nodes: int):
    parents = np.asarray(parents)
    N = parents.shape[0]
    first_child = np.full(N, -1, np.int32)
    next_sibling = np.full(N, -1, np.int32)
    for i in range(n_nodes):
        for j in range(i + 1, n_nodes):
            if parents[j] == i:
                first_child[i] = j
                break
        if i > 0:
            for j in range(i + 1, n_nodes):
                if parents[j] == parents[i]:
                    next_sibling[i] = j
                    break
    return first_child, next_sibling
