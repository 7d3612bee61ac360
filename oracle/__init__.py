"""CPU float64 oracle for the DominoTree draft-tree builder -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper over ``oracle/dominotree_oracle.c`` (plain C, gcc -O2, no BLAS).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
leg may import this package; the product (``paper_2607_08642_b200``) never does, and this
package never imports the product's CUDA binding.  Inputs are numpy arrays: bf16 tensors are
passed as ``uint16`` bit patterns (widened exactly to double inside the C code), fp32/fp64 as is.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dominotree_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

BF16, F32, F64 = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the C oracle (gcc -O2).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _W(ctypes.Structure):
    _fields_ = [("embed", ctypes.c_void_p), ("w_ih", ctypes.c_void_p), ("w_hh", ctypes.c_void_p),
                ("w1", ctypes.c_void_p), ("w2", ctypes.c_void_p),
                ("V", ctypes.c_int32), ("d", ctypes.c_int32), ("g", ctypes.c_int32),
                ("r", ctypes.c_int32), ("dtype", ctypes.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        for name in ("orc_select_topm", "orc_gru_cell", "orc_slice_logprobs", "orc_children",
                     "orc_build_tree", "orc_score_path", "orc_version"):
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def _dtype_code(a: np.ndarray) -> int:
    if a.dtype == np.uint16:
        return BF16
    if a.dtype == np.float32:
        return F32
    if a.dtype == np.float64:
        return F64
    raise TypeError(f"unsupported dtype {a.dtype} (bf16 must be passed as uint16 bits)")


def _p(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return ctypes.c_void_p(a.ctypes.data)


def to_numpy(t) -> np.ndarray:
    """torch CPU tensor (bf16/f32/f64/int) -> numpy; bf16 becomes its uint16 bit pattern."""
    import torch
    if isinstance(t, np.ndarray):
        return np.ascontiguousarray(t)
    t = t.detach().cpu().contiguous()
    if t.dtype == torch.bfloat16:
        return t.view(torch.uint16).numpy()
    return t.numpy()


def widen(a: np.ndarray) -> np.ndarray:
    """Exact float64 view of a bf16-bits / fp32 / fp64 numpy array."""
    if a.dtype == np.uint16:
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


class Weights:
    """Frozen drafter weights held as numpy arrays (kept alive for the C struct)."""

    def __init__(self, embed, gru_w_ih, gru_w_hh, corr_w1, corr_w2):
        self.embed, self.w_ih, self.w_hh, self.w1, self.w2 = (
            to_numpy(x) for x in (embed, gru_w_ih, gru_w_hh, corr_w1, corr_w2))
        dts = {_dtype_code(x) for x in (self.embed, self.w_ih, self.w_hh, self.w1, self.w2)}
        assert len(dts) == 1, "all weights must share one dtype"
        self.dtype = dts.pop()
        self.V, self.d = self.embed.shape
        self.g = self.w_hh.shape[1]
        self.r = self.w1.shape[0]
        assert self.w_ih.shape == (3 * self.g, self.d)
        assert self.w_hh.shape == (3 * self.g, self.g)
        assert self.w1.shape == (self.r, self.d + self.g)
        assert self.w2.shape == (self.V, self.r)
        self.c = _W(self.embed.ctypes.data, self.w_ih.ctypes.data, self.w_hh.ctypes.data,
                    self.w1.ctypes.data, self.w2.ctypes.data, self.V, self.d, self.g, self.r, self.dtype)

    @classmethod
    def from_dict(cls, w: dict) -> "Weights":
        return cls(w["embed"], w["gru_w_ih"], w["gru_w_hh"], w["corr_w1"], w["corr_w2"])


# ----------------------------------------------------------------------------- primitives
def select_topm(row, M: int):
    """(ids[M] int32, vals[M] float64) of the M largest entries, order (value desc, token asc)."""
    row = to_numpy(row)
    V = row.shape[0]
    ids = np.empty(M, np.int32)
    vals = np.empty(M, np.float64)
    rc = _load().orc_select_topm(_p(row), _dtype_code(row), V, M, _p(ids), _p(vals))
    if rc:
        raise ValueError(f"orc_select_topm failed rc={rc}")
    return ids, vals


def gru_cell(w: Weights, h: np.ndarray, token: int) -> np.ndarray:
    h = np.ascontiguousarray(h, np.float64)
    out = np.empty(w.g, np.float64)
    rc = _load().orc_gru_cell(ctypes.byref(w.c), _p(h), int(token), _p(out))
    if rc:
        raise ValueError(f"orc_gru_cell failed rc={rc}")
    return out


def children(w: Weights, H_i, S: np.ndarray, cand: np.ndarray, base: np.ndarray, k: int,
             T_eff: float = 1.0):
    """CHILDREN(S, i): (tokens[k], logp[k], all_logp[M])."""
    H_i = to_numpy(H_i)
    assert _dtype_code(H_i) == w.dtype
    S = np.ascontiguousarray(S, np.float64)
    cand = np.ascontiguousarray(cand, np.int32)
    base = np.ascontiguousarray(base, np.float64)
    M = cand.shape[0]
    tok = np.empty(k, np.int32)
    lp = np.empty(k, np.float64)
    allp = np.empty(M, np.float64)
    rc = _load().orc_children(ctypes.byref(w.c), _p(H_i), _p(S), _p(cand), _p(base), M, k,
                              ctypes.c_double(T_eff), _p(tok), _p(lp), _p(allp))
    if rc:
        raise ValueError(f"orc_children failed rc={rc}")
    return tok, lp, allp


# ----------------------------------------------------------------------------- Algorithm 1
@dataclass
class Tree:
    tokens: np.ndarray      # [N] int32, slot 0 = root
    parents: np.ndarray     # [N] int32, -1 for root
    depths: np.ndarray      # [N] int32
    positions: np.ndarray   # [N] int32
    scores: np.ndarray      # [N] float64 cumulative log-score
    mask: np.ndarray        # [N, N] uint8 ancestor-or-self
    n_nodes: int
    cand_ids: np.ndarray    # [L, M] int32
    cand_vals: np.ndarray   # [L, M] float64
    res_token: np.ndarray   # residual heap (never popped)
    res_parent: np.ndarray
    res_depth: np.ndarray
    res_score: np.ndarray

    def path(self, slot: int) -> List[int]:
        out = []
        while slot > 0:
            out.append(int(self.tokens[slot]))
            slot = int(self.parents[slot])
        return out[::-1]


def build_tree(w: Weights, logits, hidden, root_token: int, root_pos: int, M: int, B: int, k: int,
               temperature: float, eager_states: bool = False) -> Tree:
    logits = to_numpy(logits)
    hidden = to_numpy(hidden)
    assert _dtype_code(logits) == w.dtype and _dtype_code(hidden) == w.dtype
    L, V = logits.shape
    assert V == w.V and hidden.shape == (L, w.d)
    N = B + 1
    cap = (B + 1) * k
    tokens = np.zeros(N, np.int32); parents = np.zeros(N, np.int32); depths = np.zeros(N, np.int32)
    positions = np.zeros(N, np.int32); scores = np.zeros(N, np.float64)
    mask = np.zeros((N, N), np.uint8); n_nodes = np.zeros(1, np.int32)
    cand_ids = np.zeros((L, M), np.int32); cand_vals = np.zeros((L, M), np.float64)
    rt = np.zeros(cap, np.int32); rp = np.zeros(cap, np.int32); rd = np.zeros(cap, np.int32)
    rs = np.zeros(cap, np.float64); nres = np.zeros(1, np.int32)
    rc = _load().orc_build_tree(ctypes.byref(w.c), _p(logits), _p(hidden), L, int(root_token), int(root_pos),
                                M, B, k, ctypes.c_double(temperature), int(bool(eager_states)),
                                _p(tokens), _p(parents), _p(depths), _p(positions), _p(scores), _p(mask),
                                _p(n_nodes), _p(cand_ids), _p(cand_vals), _p(rt), _p(rp), _p(rd), _p(rs), _p(nres))
    if rc:
        raise ValueError(f"orc_build_tree failed rc={rc}")
    n = int(nres[0])
    return Tree(tokens, parents, depths, positions, scores, mask, int(n_nodes[0]), cand_ids, cand_vals,
                rt[:n].copy(), rp[:n].copy(), rd[:n].copy(), rs[:n].copy())


def build_trees(w: Weights, logits, hidden, root_tokens, root_positions, M: int, B: int, k: int,
                temperature: float, threads: int = 1) -> List[Tree]:
    """A batch of independent requests; optionally one request per host thread."""
    logits = to_numpy(logits); hidden = to_numpy(hidden)
    roots = to_numpy(root_tokens); rpos = to_numpy(root_positions) if root_positions is not None else None
    batch = logits.shape[0]

    def one(b):
        return build_tree(w, logits[b], hidden[b], int(roots[b]), int(rpos[b]) if rpos is not None else 0,
                          M, B, k, temperature)
    if threads <= 1 or batch == 1:
        return [one(b) for b in range(batch)]
    with ThreadPoolExecutor(max_workers=threads) as ex:
        return list(ex.map(one, range(batch)))


def score_path(w: Weights, hidden, root_token: int, cand_ids: np.ndarray, cand_vals: np.ndarray, k: int,
               temperature: float, path: Sequence[int]):
    """Per-level (logp, rank, kth_logp) of a token path under its own prefix (g(u) = cumsum(logp))."""
    hidden = to_numpy(hidden)
    L, M = cand_ids.shape
    path = np.ascontiguousarray(np.asarray(path, np.int32))
    n = path.shape[0]
    lp = np.zeros(max(n, 1), np.float64); rk = np.zeros(max(n, 1), np.int32); kth = np.zeros(max(n, 1), np.float64)
    ci = np.ascontiguousarray(cand_ids, np.int32); cv = np.ascontiguousarray(cand_vals, np.float64)
    rc = _load().orc_score_path(ctypes.byref(w.c), _p(hidden), L, int(root_token), _p(ci), _p(cv), M, k,
                                ctypes.c_double(temperature), _p(path), n, _p(lp), _p(rk), _p(kth))
    if rc:
        raise ValueError(f"orc_score_path failed rc={rc}")
    return lp[:n], rk[:n], kth[:n]


def version() -> int:
    return _load().orc_version()
