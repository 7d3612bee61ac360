"""paper_2607_08642_b200 -- B200-native DominoTree per-round draft-tree builder.

Thin Python binding over the C-ABI library ``libdominotree.so`` (``include/dominotree.h``):
argument marshalling only -- every step of the path (top-M select, per-round precompute, GRU
step, correction + slice log-softmax, heap, emitter) runs in the library's CUDA kernels.
PyTorch is used for device memory and streams.  There is no CPU fallback: if the library cannot
be loaded, or a call returns an error, a ``DominoTreeError`` is raised.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Dict, Optional

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libdominotree.so")

DT_BF16, DT_F32 = 0, 1
EXPORTS = ("dt_create", "dt_build_trees", "dt_select_topm", "dt_select_topm_static", "dt_static_init", "dt_build_trees_host", "dt_commit_paths", "dt_tree_links", "dt_adaptive_budget", "dt_set_option", "dt_get_option",
           "dt_kernel_launches", "dt_destroy", "dt_error_string", "dt_version", "dt_workspace_bytes",
           "dt_last_cuda_error", "dt_phase_timing", "dt_phase_slot", "dt_phase_elapsed_ms")
PHASES = ("select", "precompute", "expand", "emit")


class DominoTreeError(RuntimeError):
    pass


class _Weights(ctypes.Structure):
    _fields_ = [("embed", ctypes.c_void_p), ("gru_w_ih", ctypes.c_void_p), ("gru_w_hh", ctypes.c_void_p),
                ("corr_w1", ctypes.c_void_p), ("corr_w2", ctypes.c_void_p),
                ("V", ctypes.c_int32), ("d", ctypes.c_int32), ("g", ctypes.c_int32), ("r", ctypes.c_int32),
                ("dtype", ctypes.c_int32)]


class _Outputs(ctypes.Structure):
    _fields_ = [("tokens", ctypes.c_void_p), ("parents", ctypes.c_void_p), ("depths", ctypes.c_void_p),
                ("positions", ctypes.c_void_p), ("scores", ctypes.c_void_p), ("mask", ctypes.c_void_p),
                ("n_nodes", ctypes.c_void_p)]


_lib = None


def load_library(path: Optional[str] = None) -> ctypes.CDLL:
    """dlopen libdominotree.so and declare the prototypes of include/dominotree.h."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise DominoTreeError(f"{p} not found: run `python -m paper_2607_08642_b200.build` "
                              "(there is no CPU fallback)")
    lib = ctypes.CDLL(p)
    vp, i32, i64, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
    lib.dt_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(_Weights), i32, i32, i32, i32, i32]
    lib.dt_create.restype = ctypes.c_int
    lib.dt_build_trees.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, f32, ctypes.POINTER(_Outputs), vp]
    lib.dt_build_trees.restype = ctypes.c_int
    lib.dt_build_trees_host.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, f32, ctypes.POINTER(_Outputs), vp]
    lib.dt_build_trees_host.restype = ctypes.c_int
    lib.dt_adaptive_budget.argtypes = [vp, ctypes.POINTER(_Outputs), i32, i32, ctypes.c_double, vp, vp, vp, vp]
    lib.dt_adaptive_budget.restype = ctypes.c_int
    lib.dt_commit_paths.argtypes = [vp, ctypes.POINTER(_Outputs), i32, i32, vp, vp, vp, vp, vp, vp]
    lib.dt_commit_paths.restype = ctypes.c_int
    lib.dt_tree_links.argtypes = [vp, ctypes.POINTER(_Outputs), i32, i32, vp, vp, vp]
    lib.dt_tree_links.restype = ctypes.c_int
    lib.dt_select_topm.argtypes = [vp, vp, i32, i32, vp, vp, vp]
    lib.dt_select_topm_static.argtypes = [vp, i32, i32, i32, i32, vp, vp, vp]
    lib.dt_select_topm_static.restype = ctypes.c_int
    lib.dt_static_init.argtypes = []
    lib.dt_static_init.restype = ctypes.c_int
    lib.dt_select_topm.restype = ctypes.c_int
    lib.dt_set_option.argtypes = [vp, ctypes.c_char_p, i64]
    lib.dt_set_option.restype = ctypes.c_int
    lib.dt_get_option.argtypes = [vp, ctypes.c_char_p, ctypes.POINTER(i64)]
    lib.dt_get_option.restype = ctypes.c_int
    lib.dt_kernel_launches.argtypes = [vp]
    lib.dt_kernel_launches.restype = i64
    lib.dt_destroy.argtypes = [vp]
    lib.dt_destroy.restype = ctypes.c_int
    lib.dt_error_string.argtypes = [ctypes.c_int]
    lib.dt_error_string.restype = ctypes.c_char_p
    lib.dt_version.argtypes = []
    lib.dt_version.restype = ctypes.c_int
    lib.dt_workspace_bytes.argtypes = [vp]
    lib.dt_workspace_bytes.restype = ctypes.c_size_t
    lib.dt_last_cuda_error.argtypes = [vp]
    lib.dt_last_cuda_error.restype = ctypes.c_int
    lib.dt_phase_timing.argtypes = [vp, i32]
    lib.dt_phase_timing.restype = ctypes.c_int
    lib.dt_phase_slot.argtypes = [vp, i32]
    lib.dt_phase_slot.restype = ctypes.c_int
    lib.dt_phase_elapsed_ms.argtypes = [vp, i32, i32, ctypes.POINTER(f32)]
    lib.dt_phase_elapsed_ms.restype = ctypes.c_int
    if path is None:
        _lib = lib
    return lib


def _check(lib, rc: int, what: str, handle=None):
    if rc != 0:
        msg = lib.dt_error_string(rc).decode()
        extra = f" (cudaError {lib.dt_last_cuda_error(handle)})" if handle and rc == -3 else ""
        raise DominoTreeError(f"{what} failed: {msg}{extra}")


STATIC_MAX_ROWS = 1024          # DT_STATIC_MAX_ROWS of include/dominotree.h


def select_topm_static(logits, M: int, ids, vals, stream=None):
    """dt_select_topm_static: top-M select of [rows, V] (or [batch, L, V]) bf16 / fp32 device logits into the caller's
    `ids` (int32 [rows, M]) and `vals` (float32 [rows, M]) without a handle and without any device allocation (the
    scratch is a static device array of the library: rows <= 1024, M <= 256; calls that overlap on the GPU race)."""
    import torch
    lib = load_library()
    lg = logits.reshape(-1, logits.shape[-1])
    if not (lg.is_cuda and lg.is_contiguous()) or lg.dtype not in (torch.bfloat16, torch.float32):
        raise DominoTreeError("select_topm_static: logits must be a contiguous CUDA tensor of bfloat16 or float32")
    rows, V = lg.shape
    for t, dt_ in ((ids, torch.int32), (vals, torch.float32)):
        if not (t.is_cuda and t.is_contiguous()) or t.dtype != dt_ or tuple(t.shape) != (rows, M) or t.device != lg.device:
            raise DominoTreeError(f"select_topm_static: outputs must be contiguous [{rows}, {M}] int32 / float32 on {lg.device}")
    st = stream if stream is not None else torch.cuda.current_stream(lg.device)
    with torch.cuda.device(lg.device):
        rc = lib.dt_select_topm_static(lg.data_ptr(), DT_BF16 if lg.dtype == torch.bfloat16 else DT_F32, rows, V, M,
                                       ids.data_ptr(), vals.data_ptr(), st.cuda_stream)
    _check(lib, rc, "dt_select_topm_static")
    return ids, vals


@dataclass
class TreeBatch:
    """Device (or host, for build_trees_host) outputs of one round; N = B+1 slots, slot 0 = root."""
    tokens: "object"     # [batch, N] int32
    parents: "object"    # [batch, N] int32
    depths: "object"     # [batch, N] int32
    positions: "object"  # [batch, N] int32
    scores: "object"     # [batch, N] float32
    mask: "object"       # [batch, N, N] uint8
    n_nodes: "object"    # [batch] int32

    def _struct(self) -> _Outputs:
        return _Outputs(*(t.data_ptr() for t in (self.tokens, self.parents, self.depths, self.positions,
                                                  self.scores, self.mask, self.n_nodes)))


def alloc_outputs(batch: int, B: int, device="cuda", pin: bool = False) -> TreeBatch:
    import torch
    N = B + 1
    kw = dict(device=device)
    if pin and str(device) == "cpu":
        kw["pin_memory"] = True
    i32 = lambda *s: torch.empty(s, dtype=torch.int32, **kw)
    return TreeBatch(i32(batch, N), i32(batch, N), i32(batch, N), i32(batch, N),
                     torch.empty((batch, N), dtype=torch.float32, **kw),
                     torch.empty((batch, N, N), dtype=torch.uint8, **kw), i32(batch))


class DominoTreeBuilder:
    """Handle around dt_create / dt_build_trees / dt_destroy.  `weights` maps embed, gru_w_ih,
    gru_w_hh, corr_w1, corr_w2 to contiguous CUDA tensors of one dtype (bf16 or fp32); they are
    borrowed for the lifetime of the builder."""

    def __init__(self, weights: Dict[str, "object"], max_batch: int, L: int, max_M: int, max_B: int, k: int = 8,
                 lib_path: Optional[str] = None):
        import torch
        self.lib = load_library(lib_path)
        self._h = ctypes.c_void_p()
        ws = [weights[n] for n in ("embed", "gru_w_ih", "gru_w_hh", "corr_w1", "corr_w2")]
        for t in ws:
            if not (t.is_cuda and t.is_contiguous()):
                raise DominoTreeError("weights must be contiguous CUDA tensors")
        dts = {t.dtype for t in ws}
        if dts == {torch.bfloat16}:
            self.dtype, self.torch_dtype = DT_BF16, torch.bfloat16
        elif dts == {torch.float32}:
            self.dtype, self.torch_dtype = DT_F32, torch.float32
        else:
            raise DominoTreeError(f"weights must all be bf16 or all fp32, got {dts}")
        E, Wih, Whh, W1, W2 = ws
        self.V, self.d = E.shape
        self.g = Whh.shape[1]
        self.r = W1.shape[0]
        if Wih.shape != (3 * self.g, self.d) or Whh.shape != (3 * self.g, self.g) \
                or W1.shape != (self.r, self.d + self.g) or W2.shape != (self.V, self.r):
            raise DominoTreeError("inconsistent weight shapes")
        self._keep = ws
        self.max_batch, self.L, self.max_M, self.max_B, self.k = max_batch, L, max_M, max_B, k
        cw = _Weights(E.data_ptr(), Wih.data_ptr(), Whh.data_ptr(), W1.data_ptr(), W2.data_ptr(),
                      self.V, self.d, self.g, self.r, self.dtype)
        rc = self.lib.dt_create(ctypes.byref(self._h), ctypes.byref(cw), max_batch, L, max_M, max_B, k)
        _check(self.lib, rc, "dt_create")

    # -- the hot path ---------------------------------------------------------------------------
    def build_trees(self, marginal_logits, backbone_hidden, root_tokens, root_positions, M: int, B: int,
                    temperature: float, out: Optional[TreeBatch] = None, stream=None) -> TreeBatch:
        """dt_build_trees: asynchronous on `stream` (default: torch's current stream), capture-safe."""
        import torch
        batch = marginal_logits.shape[0]
        self._check_in(marginal_logits, (batch, self.L, self.V), self.torch_dtype, True)
        self._check_in(backbone_hidden, (batch, self.L, self.d), self.torch_dtype, True)
        self._check_in(root_tokens, (batch,), torch.int32, True)
        if root_positions is not None:
            self._check_in(root_positions, (batch,), torch.int32, True)
        if out is None:
            out = alloc_outputs(batch, B, marginal_logits.device)
        else:
            self._check_out(out, batch, B, True)
        st = stream if stream is not None else torch.cuda.current_stream()
        os_ = out._struct()
        rc = self.lib.dt_build_trees(self._h, marginal_logits.data_ptr(), backbone_hidden.data_ptr(),
                                     root_tokens.data_ptr(),
                                     root_positions.data_ptr() if root_positions is not None else None,
                                     batch, M, B, float(temperature), ctypes.byref(os_), st.cuda_stream)
        _check(self.lib, rc, "dt_build_trees", self._h)
        return out

    def select_topm(self, logits, M: int, stream=None):
        """dt_select_topm on [rows, V] (or [batch, L, V]) logits -> (cand_id int32, cand_val fp32)."""
        import torch
        lg = logits.reshape(-1, logits.shape[-1])
        self._check_in(lg, (lg.shape[0], self.V), self.torch_dtype, True)
        rows = lg.shape[0]
        ids = torch.empty((rows, M), dtype=torch.int32, device=lg.device)
        vals = torch.empty((rows, M), dtype=torch.float32, device=lg.device)
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = self.lib.dt_select_topm(self._h, lg.data_ptr(), rows, M, ids.data_ptr(), vals.data_ptr(), st.cuda_stream)
        _check(self.lib, rc, "dt_select_topm", self._h)
        return ids, vals

    def select_topm_into(self, logits, M: int, ids, vals, stream=None):
        import torch
        lg = logits.reshape(-1, logits.shape[-1])
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = self.lib.dt_select_topm(self._h, lg.data_ptr(), lg.shape[0], M, ids.data_ptr(), vals.data_ptr(), st.cuda_stream)
        _check(self.lib, rc, "dt_select_topm", self._h)

    def adaptive_budget(self, tree: TreeBatch, B: int, C_d: float, cv, stream=None):
        """dt_adaptive_budget: (n_star [batch] int32, phi [batch] float32) on the device; cv = float32 [B+1] costs."""
        import torch
        batch = tree.tokens.shape[0]
        self._check_in(cv, (B + 1,), torch.float32, True)
        n_star = torch.empty((batch,), dtype=torch.int32, device=cv.device)
        phi = torch.empty((batch,), dtype=torch.float32, device=cv.device)
        st = stream if stream is not None else torch.cuda.current_stream()
        os_ = tree._struct()
        rc = self.lib.dt_adaptive_budget(self._h, ctypes.byref(os_), batch, B, float(C_d), cv.data_ptr(),
                                         n_star.data_ptr(), phi.data_ptr(), st.cuda_stream)
        _check(self.lib, rc, "dt_adaptive_budget", self._h)
        return n_star, phi

    def commit_paths(self, tree: TreeBatch, B: int, target_next=None, edge_ok=None, stream=None):
        """dt_commit_paths: longest accepted path of every tree -> (accept_len [batch], path_slots [batch, L+1],
        bonus_token [batch]) on the device.  Pass target_next (int32 [batch, B+1], greedy verification) or
        edge_ok (uint8 [batch, B+1])."""
        import torch
        batch = tree.tokens.shape[0]
        if target_next is not None:
            self._check_in(target_next, (batch, B + 1), torch.int32, True)
        if edge_ok is not None:
            self._check_in(edge_ok, (batch, B + 1), torch.uint8, True)
        dev = tree.tokens.device
        acc = torch.empty((batch,), dtype=torch.int32, device=dev)
        path = torch.empty((batch, self.L + 1), dtype=torch.int32, device=dev)
        bonus = torch.empty((batch,), dtype=torch.int32, device=dev)
        st = stream if stream is not None else torch.cuda.current_stream()
        os_ = tree._struct()
        rc = self.lib.dt_commit_paths(self._h, ctypes.byref(os_), batch, B,
                                      target_next.data_ptr() if target_next is not None else None,
                                      edge_ok.data_ptr() if edge_ok is not None else None,
                                      acc.data_ptr(), path.data_ptr(), bonus.data_ptr(), st.cuda_stream)
        _check(self.lib, rc, "dt_commit_paths", self._h)
        return acc, path, bonus

    def tree_links(self, tree: TreeBatch, B: int, stream=None):
        """dt_tree_links: (first_child, next_sibling), int32 [batch, B+1] on the device."""
        import torch
        batch = tree.tokens.shape[0]
        dev = tree.tokens.device
        fc = torch.empty((batch, B + 1), dtype=torch.int32, device=dev)
        ns = torch.empty((batch, B + 1), dtype=torch.int32, device=dev)
        st = stream if stream is not None else torch.cuda.current_stream()
        os_ = tree._struct()
        rc = self.lib.dt_tree_links(self._h, ctypes.byref(os_), batch, B, fc.data_ptr(), ns.data_ptr(), st.cuda_stream)
        _check(self.lib, rc, "dt_tree_links", self._h)
        return fc, ns

    def build_trees_host(self, marginal_logits, backbone_hidden, root_tokens, root_positions, M: int, B: int,
                         temperature: float, out: Optional[TreeBatch] = None, stream=None) -> TreeBatch:
        """dt_build_trees_host: HOST tensors in, HOST tensors out; copies both ways and synchronises."""
        import torch
        batch = marginal_logits.shape[0]
        self._check_in(marginal_logits, (batch, self.L, self.V), self.torch_dtype, False)
        self._check_in(backbone_hidden, (batch, self.L, self.d), self.torch_dtype, False)
        self._check_in(root_tokens, (batch,), torch.int32, False)
        if root_positions is not None:
            self._check_in(root_positions, (batch,), torch.int32, False)
        if out is None:
            out = alloc_outputs(batch, B, "cpu", pin=True)
        else:
            self._check_out(out, batch, B, False)
        st = stream if stream is not None else torch.cuda.current_stream()
        os_ = out._struct()
        rc = self.lib.dt_build_trees_host(self._h, marginal_logits.data_ptr(), backbone_hidden.data_ptr(),
                                          root_tokens.data_ptr(),
                                          root_positions.data_ptr() if root_positions is not None else None,
                                          batch, M, B, float(temperature), ctypes.byref(os_), st.cuda_stream)
        _check(self.lib, rc, "dt_build_trees_host", self._h)
        return out

    # -- misc -------------------------------------------------------------------------------------
    def set_option(self, name: str, value: int):
        _check(self.lib, self.lib.dt_set_option(self._h, name.encode(), int(value)), f"dt_set_option({name})")

    def get_option(self, name: str) -> int:
        v = ctypes.c_int64()
        _check(self.lib, self.lib.dt_get_option(self._h, name.encode(), ctypes.byref(v)), f"dt_get_option({name})", self._h)
        return int(v.value)

    def phase_timing(self, n_slots: int):
        """dt_phase_timing: create (or with 0 free) n_slots sets of phase-boundary CUDA events."""
        _check(self.lib, self.lib.dt_phase_timing(self._h, int(n_slots)), "dt_phase_timing", self._h)

    def phase_slot(self, slot: int):
        _check(self.lib, self.lib.dt_phase_slot(self._h, int(slot)), "dt_phase_slot", self._h)

    def phase_ms(self, slot: int) -> Dict[str, float]:
        """Device milliseconds of each phase of the last completed round recorded into `slot`."""
        out = {}
        for i, name in enumerate(PHASES):
            ms = ctypes.c_float()
            _check(self.lib, self.lib.dt_phase_elapsed_ms(self._h, int(slot), i, ctypes.byref(ms)),
                   "dt_phase_elapsed_ms", self._h)
            out[name] = float(ms.value)
        return out

    @property
    def kernel_launches(self) -> int:
        return int(self.lib.dt_kernel_launches(self._h))

    @property
    def workspace_bytes(self) -> int:
        return int(self.lib.dt_workspace_bytes(self._h))

    def _check_in(self, t, shape, dtype, cuda: bool):
        if tuple(t.shape) != tuple(shape) or t.dtype != dtype or not t.is_contiguous() or t.is_cuda != cuda:
            raise DominoTreeError(f"expected contiguous {'cuda' if cuda else 'cpu'} tensor {shape} {dtype}, "
                                  f"got {tuple(t.shape)} {t.dtype} cuda={t.is_cuda}")

    def _check_out(self, out: TreeBatch, batch: int, B: int, cuda: bool):
        """A caller-supplied TreeBatch must have exactly the shapes the kernels write: [batch, B+1] (mask [batch, B+1, B+1])."""
        import torch
        N = B + 1
        for name in ("tokens", "parents", "depths", "positions"):
            self._check_in(getattr(out, name), (batch, N), torch.int32, cuda)
        self._check_in(out.scores, (batch, N), torch.float32, cuda)
        self._check_in(out.mask, (batch, N, N), torch.uint8, cuda)
        self._check_in(out.n_nodes, (batch,), torch.int32, cuda)

    def close(self):
        if self._h:
            self.lib.dt_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def version() -> int:
    return int(load_library().dt_version())
