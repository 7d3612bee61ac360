"""Shared fixtures for the -m gpu parity tests: seeded workloads -> CUDA builder + oracle weights.

The CUDA path is reached only through the C-ABI binding (paper_2607_08642_b200.DominoTreeBuilder);
the oracle only through the `oracle` package.  The two share nothing but the seeded input
generator (paper_2607_08642_b200.workloads, which holds none of the method's arithmetic).
"""
from __future__ import annotations

import os

import numpy as np
import torch

import oracle
from paper_2607_08642_b200 import workloads as wl

_CACHE = {}


def host_threads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


class Case:
    """Weights of one shape on both sides: CPU tensors -> oracle.Weights, CUDA copies -> builder."""

    def __init__(self, cfg: wl.Config, max_batch: int, max_M: int, max_B: int, k: int, weight_seed=None,
                 weights=None):
        import paper_2607_08642_b200 as dtb
        self.cfg = cfg
        self.k = k
        self.w_cpu = weights if weights is not None else wl.make_weights(cfg, seed=weight_seed)
        self.w_orc = oracle.Weights.from_dict(self.w_cpu)
        self.w_gpu = {n: t.cuda() for n, t in self.w_cpu.items()}
        self.builder = dtb.DominoTreeBuilder(self.w_gpu, max_batch=max_batch, L=cfg.L, max_M=max_M,
                                             max_B=max_B, k=k)

    def run_gpu(self, inp, M, B, T, use_root_pos=True):
        lg = inp["logits"].cuda(); hd = inp["hidden"].cuda()
        rt = inp["root_tokens"].cuda()
        rp = inp["root_positions"].cuda() if use_root_pos else None
        out = self.builder.build_trees(lg, hd, rt, rp, M, B, T)
        torch.cuda.synchronize()
        return out

    def run_oracle(self, inp, M, B, T, use_root_pos=True, threads=None):
        return oracle.build_trees(self.w_orc, inp["logits"], inp["hidden"], inp["root_tokens"],
                                  inp["root_positions"] if use_root_pos else None, M, B, self.k, T,
                                  threads=threads or host_threads())


def get_case(key: str, cfg: wl.Config, **kw) -> Case:
    if key not in _CACHE:
        _CACHE[key] = Case(cfg, **kw)
    return _CACHE[key]


def qwen8b_case() -> Case:
    """One Qwen3-8B-shaped weight set (configs[2] seed) shared by configs[2], [3] and [4]."""
    cfg = wl.CONFIGS["qwen8b"]
    return get_case("qwen8b", cfg, max_batch=32, max_M=128, max_B=128, k=8)


def qwen4b_case() -> Case:
    cfg = wl.CONFIGS["qwen4b"]
    return get_case("qwen4b", cfg, max_batch=4, max_M=128, max_B=64, k=8)


def tiny_case(k=8, max_M=64, max_B=64, name="tiny", **cfg_kw) -> Case:
    cfg = wl.CONFIGS[name].replace(**cfg_kw) if cfg_kw else wl.CONFIGS[name]
    key = f"{name}-{k}-{max_M}-{max_B}-{sorted(cfg_kw.items())}"
    return get_case(key, cfg, max_batch=32, max_M=max_M, max_B=max_B, k=k)


def check_batch(case: Case, inp, M, B, T, score_tol, use_root_pos=True, out=None, trees=None):
    """Compare every request of a batch; returns (#exact, #tolerant)."""
    from compare import compare_tree, tree_to_numpy
    if out is None:
        out = case.run_gpu(inp, M, B, T, use_root_pos)
    if trees is None:
        trees = case.run_oracle(inp, M, B, T, use_root_pos)
    n_exact = n_tol = 0
    hid = oracle.to_numpy(inp["hidden"])
    for b, tr in enumerate(trees):
        res = compare_tree(tree_to_numpy(out, b), tr, case.w_orc, hid[b], int(inp["root_tokens"][b]),
                           int(inp["root_positions"][b]) if use_root_pos else 0,
                           case.cfg.L, B, case.k, T, score_tol)
        n_exact += res == "exact"
        n_tol += res == "tolerant"
    return n_exact, n_tol
