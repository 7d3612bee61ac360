"""CPU-only checks of the boundary: libdominotree.so loads, exports every symbol that
include/dominotree.h declares, argument validation returns error codes without touching a GPU,
and the N>1 host logic (request sharding, max-over-ranks timing) works over gloo, world_size 2."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_08642_b200 import build, load_library
    build.build()
    return load_library()


def test_library_exports_every_declared_symbol(lib):
    import paper_2607_08642_b200 as dtb
    hdr = open(os.path.join(ROOT, "include", "dominotree.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(dt_[a-z_]+)\s*\(", hdr))
    assert declared == set(dtb.EXPORTS), declared ^ set(dtb.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_version_and_error_strings(lib):
    assert lib.dt_version() == 1
    assert lib.dt_error_string(0) == b"ok"
    seen = {lib.dt_error_string(c) for c in (-1, -2, -3, -4)}
    assert len(seen) == 4 and b"unknown error" not in seen
    assert lib.dt_error_string(-99) == b"unknown error"


def test_argument_validation_needs_no_gpu(lib):
    import paper_2607_08642_b200 as dtb
    h = ctypes.c_void_p()
    assert lib.dt_create(ctypes.byref(h), None, 1, 4, 8, 8, 8) == -1          # null weights
    w = dtb._Weights(1, 1, 1, 1, 1, 1024, 64, 32, 32, dtb.DT_F32)
    assert lib.dt_create(None, ctypes.byref(w), 1, 4, 8, 8, 8) == -1
    assert lib.dt_create(ctypes.byref(h), ctypes.byref(w), 1, 4, 4, 8, 8) == -1   # max_M < k
    assert lib.dt_create(ctypes.byref(h), ctypes.byref(w), 1, 4, 2000, 8, 8) == -1  # max_M > V
    assert lib.dt_create(ctypes.byref(h), ctypes.byref(w), 1, 4, 512, 8, 8) == -2  # > DT_MAX_M
    assert lib.dt_create(ctypes.byref(h), ctypes.byref(w), 1, 4, 8, 300, 8) == -2  # > DT_MAX_B
    w.dtype = 7
    assert lib.dt_create(ctypes.byref(h), ctypes.byref(w), 1, 4, 8, 8, 8) == -1
    assert lib.dt_build_trees(None, None, None, None, None, 1, 8, 8, 0.0, None, None) == -1
    assert lib.dt_select_topm(None, None, 1, 8, None, None, None) == -1
    assert lib.dt_destroy(None) == 0
    assert lib.dt_workspace_bytes(None) == 0


def test_product_fails_loudly_without_library(tmp_path):
    import paper_2607_08642_b200 as dtb
    with pytest.raises(dtb.DominoTreeError):
        dtb.load_library(str(tmp_path / "missing.so"))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2607_08642_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "liboracle" not in src and "dominotree_oracle" not in src, f


def test_shard_range_partitions():
    from paper_2607_08642_b200.dist import shard_range
    for n in (0, 1, 5, 32, 33):
        for world in (1, 2, 3, 8):
            parts = [shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _gloo_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    from paper_2607_08642_b200 import dist as d
    dist = d.init_process_group("gloo")
    lo, hi = d.shard_range(33, rank, world)
    dist.barrier()
    t_max = d.max_over_ranks(10.0 + rank)
    n_sum = d.sum_over_ranks(hi - lo)
    q.put((rank, lo, hi, t_max, n_sum))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_sharding_and_timing_reduction():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + os.getpid() % 300
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, m0, s0), (r1, lo1, hi1, m1, s1) = res
    assert (lo0, hi0, lo1, hi1) == (0, 17, 17, 33)
    assert m0 == m1 == 11.0          # max over ranks
    assert s0 == s1 == 33.0          # every request counted exactly once
