"""First-child / next-sibling link arrays (second half).

CPU: pins of the plain-Python oracle (oracle/links.py): a hand-worked tree, the chain and the star, the walk property
(a first-child / next-sibling traversal from the root visits every valid node exactly once, in an order in which every
sibling group appears in pop order), agreement with children lists built independently, dead leaves unlinked.
GPU: dt_tree_links against the oracle on trees built by the CUDA path."""
import numpy as np
import pytest

from oracle import links


def _walk(fc, ns):
    """Pre-order traversal through the two arrays only."""
    out, stack = [], [0]
    while stack:
        i = stack.pop()
        out.append(i)
        if ns[i] >= 0:
            stack.append(int(ns[i]))
        if fc[i] >= 0:
            stack.append(int(fc[i]))
    return out


def test_hand_worked_tree():
    #            0
    #        1       2
    #      3   5     4
    #      6
    parents = np.array([-1, 0, 0, 1, 2, 1, 3, 0, 0], np.int32)      # slots 7, 8: dead-leaf padding (parent 0, reading A10)
    fc, ns = links.tree_links(parents, 7)
    assert fc.tolist() == [1, 3, 4, 6, -1, -1, -1, -1, -1]
    assert ns.tolist() == [-1, 2, -1, 5, -1, -1, -1, -1, -1]
    assert _walk(fc, ns) == [0, 1, 3, 6, 5, 2, 4]


def test_chain_and_star():
    fc, ns = links.tree_links(np.array([-1, 0, 1, 2, 3], np.int32), 5)
    assert fc.tolist() == [1, 2, 3, 4, -1] and ns.tolist() == [-1] * 5
    fc, ns = links.tree_links(np.array([-1, 0, 0, 0, 0], np.int32), 5)
    assert fc.tolist() == [1, -1, -1, -1, -1] and ns.tolist() == [-1, 2, 3, 4, -1]


@pytest.mark.parametrize("seed", range(20))
def test_walk_visits_every_node_once_and_siblings_in_pop_order(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 40))
    N = n + int(rng.integers(0, 4))
    parents = np.zeros(N, np.int32)
    parents[0] = -1
    for i in range(1, n):
        parents[i] = rng.integers(0, i)
    fc, ns = links.tree_links(parents, n)
    order = _walk(fc, ns)
    assert sorted(order) == list(range(n))
    kids = {i: [j for j in range(1, n) if parents[j] == i] for i in range(n)}      # independent: children lists
    for i in range(n):
        chain, j = [], int(fc[i])
        while j >= 0:
            chain.append(j)
            j = int(ns[j])
        assert chain == kids[i]
    assert np.all(fc[n:] == -1) and np.all(ns[n:] == -1)


@pytest.mark.gpu
def test_gpu_tree_links_match_oracle():
    import torch
    import gpu_util as gu
    from paper_2607_08642_b200 import workloads as wl
    cfg = wl.CONFIGS["tiny"].replace(dtype="bf16", g=128, r=40, d=96, V=2000, L=5, embed_std=1.0)
    for k, M, B, batch in ((8, 24, 40, 9), (1, 8, 12, 3), (3, 20, 17, 5)):
        case = gu.get_case(f"links-{k}", cfg, max_batch=16, max_M=32, max_B=48, k=k)
        inp = wl.make_inputs(cfg, batch=batch, seed=6100 + k)
        out = case.run_gpu(inp, M, B, 0.6)
        fc, ns = case.builder.tree_links(out, B)
        torch.cuda.synchronize()
        for b in range(batch):
            rfc, rns = links.tree_links(out.parents[b].cpu().numpy(), int(out.n_nodes[b]))
            assert np.array_equal(fc[b].cpu().numpy(), rfc), (k, b)
            assert np.array_equal(ns[b].cpu().numpy(), rns), (k, b)
