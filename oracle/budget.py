"""Cost-aware adaptive budget (CaDDTree's stopping rule inlined in the pop loop) -- TEST INFRASTRUCTURE ONLY.

PAPER.md:97-101 (Sec. 2.5) and 161-165 (Sec. 3.4): with pi_s = exp(cumulative log-score of the s-th popped node),
Phi(n) = sum_{s <= n} pi_s and theta(n) = (1 + Phi(n)) / (C_d + C_v(n)); "grow the tree node by node in best-first
order and stop the first time theta stops improving" / "run Algorithm 1 to a generous cap, accumulate Phi(n) as nodes
pop, and stop when theta(n) stops improving".  Plain float64 loop.

Readings where the paper is silent: the root is not a draft node (s counts slots 1..); theta(0) = 1 / (C_d + C_v(0));
"stops improving" means theta(n + 1) <= theta(n); C_v is a caller-supplied table cv[0..B]; dead-leaf slots
(>= n_nodes) are never counted.
"""
from __future__ import annotations

import math
from typing import Sequence, Tuple


def adaptive_budget(scores: Sequence[float], n_nodes: int, C_d: float, cv: Sequence[float]) -> Tuple[int, float]:
    """Returns (n_star, Phi(n_star)): the number of draft nodes (slots 1..n_star) the rule keeps."""
    n, phi = 0, 0.0
    theta = (1.0 + phi) / (C_d + cv[0])
    while n + 1 < n_nodes:
        phi_next = phi + math.exp(scores[n + 1])
        theta_next = (1.0 + phi_next) / (C_d + cv[n + 1])
        if theta_next <= theta:
            break
        n, phi, theta = n + 1, phi_next, theta_next
    return n, phi
