"""Cost-aware adaptive budget: oracle pins (CPU) and GPU parity."""
import math
import os
import sys

import numpy as np
import pytest
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from oracle.budget import adaptive_budget  # noqa: E402


def _theta(scores, n, C_d, cv):
    return (1.0 + sum(math.exp(scores[s]) for s in range(1, n + 1))) / (C_d + cv[n])


def test_free_verification_runs_to_the_cap():
    # C_v constant: one more node can only add acceptance mass, theta keeps improving (the paper's observed failure
    # mode on the over-credited corrected tree: "n* runs to the cap")
    scores = [0.0] + [-0.3 * s for s in range(1, 17)]
    n, phi = adaptive_budget(scores, 17, 3.5, [18.7] * 17)
    assert n == 16 and abs(phi - sum(math.exp(x) for x in scores[1:])) < 1e-12


def test_expensive_first_node_keeps_nothing():
    scores = [0.0, -5.0, -5.1, -5.2]
    n, phi = adaptive_budget(scores, 4, 1.0, [1.0, 5.0, 9.0, 13.0])
    assert (n, phi) == (0, 0.0)


def test_hand_worked_example():
    # pi = 0.5, 0.25, 0.125; C_d = 1, C_v(n) = 0.2 n^2: theta = 1/1, 1.5/1.2 = 1.25, 1.75/1.8 = 0.972 -> stop at n = 1
    scores = [0.0, math.log(0.5), math.log(0.25), math.log(0.125)]
    cv = [0.2 * n * n for n in range(4)]
    n, phi = adaptive_budget(scores, 4, 1.0, cv)
    assert n == 1 and abs(phi - 0.5) < 1e-15


@pytest.mark.parametrize("seed", range(8))
def test_greedy_stop_is_the_global_optimum_under_convex_cost(seed):
    # CaDDTree's theorem: convex C_v and pop-order (non-increasing) masses make theta unimodal, so the
    # greedy stop equals the brute-force argmax of theta over all budgets
    rng = np.random.default_rng(seed)
    for _ in range(50):
        B = int(rng.integers(1, 64))
        scores = [0.0] + sorted((-float(x) for x in rng.exponential(1.5, B)), reverse=True)
        a, b2, c = rng.uniform(0.0, 2.0), rng.uniform(0.0, 0.3), rng.uniform(0.0, 0.02)
        cv = [a + b2 * n + c * n * n for n in range(B + 1)]
        C_d = float(rng.uniform(0.1, 4.0))
        n_valid = int(rng.integers(1, B + 2))
        n, phi = adaptive_budget(scores, n_valid, C_d, cv)
        thetas = [_theta(scores, m, C_d, cv) for m in range(n_valid)]
        best = max(thetas)
        assert thetas[n] >= best - 1e-12 * abs(best)
        assert abs(phi - sum(math.exp(scores[s]) for s in range(1, n + 1))) < 1e-12
        assert all(thetas[m + 1] > thetas[m] for m in range(n))                  # improved at every kept node


@pytest.mark.gpu
def test_gpu_adaptive_budget_matches_oracle():
    import gpu_util as gu
    from paper_2607_08642_b200 import workloads as wl
    case = gu.tiny_case()
    rng = np.random.default_rng(3)
    for B, batch in ((8, 5), (31, 32), (64, 3)):
        inp = wl.make_inputs(case.cfg, batch=batch, seed=5000 + B)
        out = case.run_gpu(inp, 8, B, 0.0)
        sco, nn = out.scores.cpu().numpy().astype(np.float64), out.n_nodes.cpu().numpy()
        for trial in range(3):
            a, b2, c = rng.uniform(0.0, 2.0), rng.uniform(0.0, 0.3), rng.uniform(0.0, 0.02)
            cv = np.asarray([a + b2 * n + c * n * n for n in range(B + 1)], np.float32)
            C_d = float(rng.uniform(0.1, 4.0))
            n_star, phi = case.builder.adaptive_budget(out, B, C_d, torch.from_numpy(cv).cuda())
            torch.cuda.synchronize()
            n_star, phi = n_star.cpu().numpy(), phi.cpu().numpy()
            for b in range(batch):
                n, ph = adaptive_budget(sco[b].tolist(), int(nn[b]), C_d, cv.astype(np.float64).tolist())
                assert int(n_star[b]) == n and abs(float(phi[b]) - ph) < 1e-5 * max(1.0, ph)
