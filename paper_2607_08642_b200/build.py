"""Build libdominotree.so (the C-ABI library of include/dominotree.h) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
repo snapshot.  Usage:  python -m paper_2607_08642_b200.build  [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libdominotree.so")
LIB_TRACE = os.path.join(PKG, "libdominotree_trace.so")   # measurement build (-DDT_TRACE): in-kernel timeline for bench.py --trace
SOURCES = ["dt_api.cu"]
HEADERS = ["dt_common.cuh", "dt_select.cuh", "dt_precompute.cuh", "dt_expand.cuh", "dt_fused.cuh", "dt_gemm_mma.cuh",
           "dt_tcgen05.cuh", "dt_commit.cuh", "dt_scorers.cuh", "dt_budget.cuh", "dt_gemm_tc.cuh", "dt_frontier.cuh", "dt_wave.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps():
    out = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    out.append(os.path.join(ROOT, "include", "dominotree.h"))
    out.append(os.path.abspath(__file__))
    return out


def needs_build(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in _deps() if os.path.exists(d))


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    """Compile the product library, or with trace=True the measurement build libdominotree_trace.so (same sources,
    -DDT_TRACE: the wavefront kernel stamps %globaltimer into a device buffer read by dt_trace_read)."""
    lib = LIB_TRACE if trace else LIB
    if not force and not needs_build(lib):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [_nvcc()] + NVCC_FLAGS + (["-DDT_TRACE"] if trace else []) + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd, cwd=CSRC)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
