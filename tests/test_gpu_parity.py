"""-m gpu parity tests: the CUDA path (through the C-ABI binding) vs the float64 oracle, element by
element on the same seeded inputs.  Bar (BASELINE.json north_star): select bit-exact; trees exact
except where two oracle scores differ by < 1e-4; scores within 2e-3 (bf16 configs) / 1e-5 (tiny fp32).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_08642_b200 import workloads as wl

pytestmark = pytest.mark.gpu

BF16_TOL = 2e-3
F32_TOL = 1e-5


def _gu():
    import gpu_util
    return gpu_util


# ------------------------------------------------------------------------------------ select (a1)
def _check_select(builder, logits_cpu, M, rows_to_check=None):
    ids, vals = builder.select_topm(logits_cpu.cuda(), M)
    torch.cuda.synchronize()
    ids = ids.cpu().numpy(); vals = vals.cpu().numpy()
    lg = logits_cpu.reshape(-1, logits_cpu.shape[-1])
    rows = range(lg.shape[0]) if rows_to_check is None else rows_to_check
    for r in rows:
        oi, ov = oracle.select_topm(lg[r], M)
        assert np.array_equal(ids[r], oi), f"row {r}: ids differ at {np.nonzero(ids[r] != oi)[0][:5]}"
        assert np.array_equal(vals[r].astype(np.float64), ov), f"row {r}: values differ"
    return ids, vals


@pytest.mark.parametrize("M", [1, 8, 64])
def test_select_tiny_fp32_exact(M):
    case = _gu().tiny_case()
    inp = wl.make_inputs(case.cfg, batch=8)
    _check_select(case.builder, inp["logits"], M)


@pytest.mark.parametrize("chunks", [0, 1, 2, 5, 32])
@pytest.mark.parametrize("M", [32, 64, 128])
def test_select_qwen_rows_exact_all_chunkings(M, chunks):
    case = _gu().qwen8b_case()
    inp = wl.make_inputs(case.cfg, batch=1, regime="peaked" if M == 64 else "flat")
    case.builder.set_option("select_chunks", chunks)
    try:
        _check_select(case.builder, inp["logits"], M)
    finally:
        case.builder.set_option("select_chunks", 0)


@pytest.mark.parametrize("chunks", [1, 4])
def test_select_register_tile_kernel_on_aligned_rows(chunks):
    """The register-tile kernel (select_kernel = 1; the default for aligned rows is the bulk-copy kernel) on
    Qwen-sized rows and on the adversarial rows, M = 64 and M = 256 (largest supported)."""
    gu = _gu()
    case = gu.get_case("qwen8b-m256", wl.CONFIGS["qwen8b"], max_batch=1, max_M=256, max_B=16, k=8)
    inp = wl.make_inputs(case.cfg, batch=1, regime="peaked")
    rows = wl.adversarial_select_rows(case.cfg.V, case.cfg.torch_dtype)
    adv = torch.stack(list(rows.values()))
    case.builder.set_option("select_chunks", chunks)
    try:
        for kern in (1, 0):
            case.builder.set_option("select_kernel", kern)
            _check_select(case.builder, inp["logits"], 256)
            _check_select(case.builder, inp["logits"], 64)
            _check_select(case.builder, adv, 256)
    finally:
        case.builder.set_option("select_kernel", 0)
        case.builder.set_option("select_chunks", 0)


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("chunks", [1, 3])
def test_select_adversarial_rows(dtype, chunks):
    """all-equal, ascending, descending, many ties at the M-th value, -inf entries, signed zeros:
    exercises the candidate-buffer overflow path and the (value desc, token asc) rule with -0 == +0."""
    gu = _gu()
    if dtype == "bf16":
        case = gu.qwen8b_case()
    else:
        case = gu.tiny_case(name="tiny", V=8192 + 64)      # several tiles + a ragged tail
    rows = wl.adversarial_select_rows(case.cfg.V, case.cfg.torch_dtype)
    lg = torch.stack(list(rows.values()))
    case.builder.set_option("select_chunks", chunks)
    try:
        for M in (8, 64):
            _check_select(case.builder, lg, M)
    finally:
        case.builder.set_option("select_chunks", 0)


@pytest.mark.parametrize("V", [1001, 4099, 33])
def test_select_unaligned_vocab(V):
    """V not a multiple of the vector width -> scalar-load kernel variant; ragged last vector."""
    case = _gu().tiny_case(name="tiny", V=V, dtype="bf16", max_M=8)
    inp = wl.make_inputs(case.cfg, batch=3)
    _check_select(case.builder, inp["logits"], 8)


def test_select_full_size_batch32():
    """BASELINE configs[4] select at full size, in the launch configuration bench.py times:
    512 rows x 151,936 bf16.  Oracle on sampled rows; every row against library top-k values and
    the ordering rule."""
    case = _gu().qwen8b_case()
    cfg = wl.CONFIGS["concurrent8b"]
    inp = wl.make_inputs(cfg, batch=32)
    lg = inp["logits"]
    sample = list(range(0, 512, 37)) + [511]
    ids, vals = _check_select(case.builder, lg, 64, rows_to_check=sample)
    lgc = lg.reshape(512, -1).cuda().float()
    tv = torch.topk(lgc, 64, dim=1).values.cpu().numpy()
    assert np.array_equal(vals, tv)
    gathered = torch.gather(lgc, 1, torch.from_numpy(ids).cuda().long()).cpu().numpy()
    assert np.array_equal(gathered, vals)
    same = vals[:, 1:] == vals[:, :-1]
    assert np.all(ids[:, 1:][same] > ids[:, :-1][same]), "ties must be ordered by token id ascending"


# ------------------------------------------------------------------------------------ trees
@pytest.mark.parametrize("regime", ["flat", "peaked"])
@pytest.mark.parametrize("T", [0.0, 0.6, 1.0])
def test_tree_tiny_fp32(regime, T):
    """BASELINE configs[0]."""
    gu = _gu()
    case = gu.tiny_case()
    cfg = case.cfg
    inp = wl.make_inputs(cfg, batch=4, regime=regime)
    ne, nt = gu.check_batch(case, inp, cfg.M, cfg.B, T, F32_TOL)
    assert ne + nt == 4


def test_tree_tiny_bruteforce_shape():
    """V=16, M=16, k=16 variant of configs[0] (the oracle itself is brute-force pinned at this size)."""
    gu = _gu()
    case = gu.tiny_case(k=16, max_M=16, max_B=64, name="brute")
    inp = wl.make_inputs(case.cfg, batch=8)
    for B in (1, 8, 40):
        ne, nt = gu.check_batch(case, inp, 16, B, 0.0, F32_TOL)
        assert ne + nt == 8


@pytest.mark.parametrize("k,M,B", [(1, 8, 8), (1, 1, 4), (8, 8, 64), (3, 5, 17)])
def test_tree_tiny_edge_shapes(k, M, B):
    """k=1 chain incl. exhausted candidate tree (dead leaves), M=k, M=1 degenerate ties, odd sizes."""
    gu = _gu()
    case = gu.tiny_case(k=k)
    inp = wl.make_inputs(case.cfg, batch=5, regime="peaked")
    ne, nt = gu.check_batch(case, inp, M, B, 0.0, F32_TOL)
    assert ne + nt == 5


def test_tree_tiny_no_root_positions_and_batch_sizes():
    gu = _gu()
    case = gu.tiny_case()
    for batch in (1, 2, 7, 32):
        inp = wl.make_inputs(case.cfg, batch=batch, seed=500 + batch)
        ne, nt = gu.check_batch(case, inp, 8, 8, 0.0, F32_TOL, use_root_pos=False)
        assert ne + nt == batch


def test_tree_stress_path_dependence():
    """E ~ N(0,1): sibling paths get visibly different corrections (SURVEY.md 8(c) stress config)."""
    gu = _gu()
    case = gu.tiny_case(embed_std=1.0)
    inp = wl.make_inputs(case.cfg, batch=8)
    ne, nt = gu.check_batch(case, inp, 8, 32, 0.0, 5e-5)
    assert ne + nt == 8


def _small_bf16_case(gu, g, r, k, max_M, max_B):
    """Small bf16 shapes that take the fused persistent expansion kernel (dt_fused.cuh)."""
    cfg = wl.CONFIGS["tiny"].replace(dtype="bf16", g=g, r=r, d=96, V=2000, L=5, embed_std=1.0)
    key = f"smallbf16-{g}-{r}-{k}-{max_M}-{max_B}"
    return gu.get_case(key, cfg, max_batch=40, max_M=max_M, max_B=max_B, k=k)


@pytest.mark.parametrize("path", [0, 1, 2, 3])
@pytest.mark.parametrize("batch,M,B,k", [(1, 8, 8, 8), (5, 20, 17, 3), (33, 24, 40, 8), (40, 9, 6, 1)])
def test_tree_small_bf16_all_expand_paths(path, batch, M, B, k):
    """Ragged small shapes (batch > one 32-request MMA pass, M and r not powers of two, short trees
    with k = 1) through every expansion path: auto, per-step kernels, fused upc=8, fused upc=16."""
    gu = _gu()
    case = _small_bf16_case(gu, 64, 40, k, 32, 48)
    inp = wl.make_inputs(case.cfg, batch=batch, seed=900 + batch, regime="flat" if batch % 2 else "peaked")
    case.builder.set_option("expand_path", path)
    try:
        ne, nt = gu.check_batch(case, inp, M, B, 0.6, BF16_TOL)
        launches = case.builder.kernel_launches
    finally:
        case.builder.set_option("expand_path", 0)
    assert ne + nt == batch
    if path != 1:
        assert launches <= 5, launches            # select, GEMM, init, fused kernel: no per-pop launches


@pytest.mark.parametrize("batch,M,B,k", [(1, 8, 8, 8), (5, 20, 17, 3), (33, 24, 40, 8), (40, 9, 6, 1)])
def test_tree_small_bf16_tcgen05_path(batch, M, B, k):
    """The tcgen05 + TMEM GRU role (expand_path 4) on a small shape it accepts (g a multiple of 256, r <= 256 and
    not a multiple of 16), ragged batch / M / B, against the oracle."""
    gu = _gu()
    case = _small_bf16_case(gu, 256, 40, k, 32, 48)
    inp = wl.make_inputs(case.cfg, batch=batch, seed=700 + batch, regime="flat" if batch % 2 else "peaked")
    case.builder.set_option("expand_path", 4)
    try:
        ne, nt = gu.check_batch(case, inp, M, B, 0.6, BF16_TOL)
        launches = case.builder.kernel_launches
    finally:
        case.builder.set_option("expand_path", 0)
    assert ne + nt == batch
    assert launches <= 5, launches


def test_tree_fused_short_tree_and_leaf_pops():
    """k = 1 chain longer than L (tree exhausted: n_nodes < B+1, dead-leaf padding) and B large
    enough that depth-L leaves are popped (nodes that are never expanded) on the fused path."""
    gu = _gu()
    case = _small_bf16_case(gu, 32, 16, 1, 32, 48)
    inp = wl.make_inputs(case.cfg, batch=3, seed=31)
    ne, nt = gu.check_batch(case, inp, 4, 12, 0.0, BF16_TOL)
    assert ne + nt == 3
    out = case.run_gpu(inp, 4, 12, 0.0)
    assert out.n_nodes.tolist() == [6, 6, 6]          # root + L = 5 chain nodes
    case2 = _small_bf16_case(gu, 32, 16, 2, 32, 48)
    ne, nt = gu.check_batch(case2, inp, 6, 48, 1.0, BF16_TOL)
    assert ne + nt == 3


@pytest.mark.parametrize("regime", ["flat", "peaked"])
def test_tree_qwen4b(regime):
    """BASELINE configs[1]."""
    gu = _gu()
    case = gu.qwen4b_case()
    cfg = case.cfg
    inp = wl.make_inputs(cfg, batch=1, regime=regime)
    ne, nt = gu.check_batch(case, inp, cfg.M, cfg.B, cfg.T, BF16_TOL)
    assert ne + nt == 1


@pytest.mark.parametrize("regime", ["flat", "peaked"])
@pytest.mark.parametrize("T", [0.0, 0.6, 1.0])
def test_tree_qwen8b_temperatures(regime, T):
    """BASELINE configs[2]."""
    gu = _gu()
    case = gu.qwen8b_case()
    cfg = wl.CONFIGS["qwen8b"]
    inp = wl.make_inputs(cfg, batch=1, regime=regime)
    ne, nt = gu.check_batch(case, inp, cfg.M, cfg.B, T, BF16_TOL)
    assert ne + nt == 1


@pytest.mark.parametrize("B", [16, 32, 64, 128])
@pytest.mark.parametrize("M", [32, 64, 128])
def test_tree_qwen8b_sweep(B, M):
    """BASELINE configs[3]."""
    gu = _gu()
    case = gu.qwen8b_case()
    cfg = wl.CONFIGS["sweep8b"]
    inp = wl.make_inputs(cfg, batch=1, regime="flat" if (B // 16 + M // 32) % 2 else "peaked")
    ne, nt = gu.check_batch(case, inp, M, B, 0.0, BF16_TOL)
    assert ne + nt == 1


@pytest.mark.parametrize("regime", ["flat", "peaked"])
def test_tree_concurrent_batch32_cuda_graph(regime):
    """BASELINE configs[4] at full size, replayed from ONE CUDA graph as bench.py times it, and
    batch invariance: the batch-32 result equals 32 batch-1 results."""
    gu = _gu()
    case = gu.qwen8b_case()
    cfg = wl.CONFIGS["concurrent8b"]
    inp = wl.make_inputs(cfg, batch=32, regime=regime)
    import paper_2607_08642_b200 as dtb
    lg, hd = inp["logits"].cuda(), inp["hidden"].cuda()
    rt, rp = inp["root_tokens"].cuda(), inp["root_positions"].cuda()
    out = dtb.alloc_outputs(32, cfg.B)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        case.builder.build_trees(lg, hd, rt, rp, cfg.M, cfg.B, cfg.T, out=out, stream=st)   # warm-up
        st.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=st):
            case.builder.build_trees(lg, hd, rt, rp, cfg.M, cfg.B, cfg.T, out=out, stream=st)
    for t in (out.tokens, out.parents, out.depths, out.positions, out.scores, out.mask, out.n_nodes):
        t.zero_()
    graph.replay(); graph.replay()
    torch.cuda.synchronize()
    ne, nt = gu.check_batch(case, inp, cfg.M, cfg.B, cfg.T, BF16_TOL, out=out)
    assert ne + nt == 32
    # batch invariance (bitwise, GPU vs GPU)
    for b in (0, 13, 31):
        one = {k_: v[b:b + 1] for k_, v in inp.items()}
        o1 = case.run_gpu(one, cfg.M, cfg.B, cfg.T)
        for name in ("tokens", "parents", "depths", "positions", "scores", "mask", "n_nodes"):
            assert torch.equal(getattr(o1, name)[0], getattr(out, name)[b]), (b, name)


def test_host_entry_point_matches_device_entry_point():
    gu = _gu()
    case = gu.tiny_case()
    cfg = case.cfg
    inp = wl.make_inputs(cfg, batch=6, seed=77)
    dev = case.run_gpu(inp, 8, 8, 0.6)
    host = case.builder.build_trees_host(inp["logits"], inp["hidden"], inp["root_tokens"],
                                         inp["root_positions"], 8, 8, 0.6)
    for name in ("tokens", "parents", "depths", "positions", "scores", "mask", "n_nodes"):
        assert torch.equal(getattr(dev, name).cpu(), getattr(host, name)), name


def test_error_codes_and_empty_batch():
    import paper_2607_08642_b200 as dtb
    gu = _gu()
    case = gu.tiny_case()
    cfg = case.cfg
    inp = wl.make_inputs(cfg, batch=2)
    with pytest.raises(dtb.DominoTreeError):
        case.run_gpu(inp, 4, 8, 0.0)            # M < k
    with pytest.raises(dtb.DominoTreeError):
        case.run_gpu(inp, 8, 1000, 0.0)         # B > max_B
    with pytest.raises(dtb.DominoTreeError):
        case.run_gpu(inp, 8, 8, -1.0)           # negative temperature
    with pytest.raises(dtb.DominoTreeError):
        case.run_gpu(inp, 8, 8, float("nan"))
    empty = {k_: v[:0] for k_, v in inp.items()}
    out = case.run_gpu(empty, 8, 8, 0.0)
    assert out.tokens.shape == (0, 9)
    assert case.builder.kernel_launches == 0
    case.run_gpu(inp, 8, 8, 0.0)
    assert case.builder.kernel_launches > 0
