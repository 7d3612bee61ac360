"""Speculation in the lock-step expansion kernel (dt_fused.cuh, fused_gru_role_tc), -m gpu, through the C-ABI.

The GRU CTAs run the pass of the node a chain would pop next (parent = the node just confirmed, token = the marginal
top-1 of the next depth) while the request CTA still scores that parent; a hit is served by that pass, a miss by a
second one.  It changes WHEN a node's state is computed, never what is computed, so:
* with the speculation forced on (option 2) the trees match the float64 oracle on small bf16 shapes, flat inputs (mostly
  misses) and peaked ones (mostly hits), ragged batches, several request groups, short trees, leaf pops (B > what L allows
  along a chain), k = 1;
* at full size the forced-on and the off kernel return bit-identical outputs, scores included;
* the Cond-static arm (greedy chain) gives the same menus / trees with it;
* the adaptive schedule uses it on peaked rounds by default.
"""
import pytest
import torch

from paper_2607_08642_b200 import workloads as wl

pytestmark = pytest.mark.gpu
BF16_TOL = 2e-3
FIELDS = ("tokens", "parents", "depths", "positions", "scores", "mask", "n_nodes")


def _gu():
    import gpu_util
    return gpu_util


class _Opts:
    """Set handle options for a block; put the defaults back afterwards."""
    DEFAULTS = {"adaptive_schedule": 1, "lockstep_speculation": 1}

    def __init__(self, case, **opts):
        self.case, self.opts = case, opts

    def __enter__(self):
        for n, v in self.opts.items():
            self.case.builder.set_option(n, v)

    def __exit__(self, *exc):
        for n in self.opts:
            self.case.builder.set_option(n, self.DEFAULTS.get(n, 0))


def _small(gu, k, max_batch=40):
    cfg = wl.CONFIGS["tiny"].replace(dtype="bf16", g=256, r=40, d=96, V=2000, L=5, embed_std=1.0)
    return gu.get_case(f"wave-256-40-{k}-{max_batch}", cfg, max_batch=max_batch, max_M=32, max_B=48, k=k)


@pytest.mark.parametrize("group", [0, 16])
@pytest.mark.parametrize("batch,M,B,k,regime", [(1, 8, 8, 8, "peaked"), (5, 20, 17, 3, "flat"), (33, 24, 40, 8, "peaked"),
                                                (40, 9, 6, 1, "peaked"), (7, 32, 48, 4, "flat"), (32, 16, 2, 8, "peaked")])
def test_speculation_small_bf16_vs_oracle(batch, M, B, k, regime, group):
    gu = _gu()
    case = _small(gu, k)
    inp = wl.make_inputs(case.cfg, batch=batch, seed=4100 + batch + B, regime=regime)
    with _Opts(case, expand_path=4, lockstep_speculation=2, lockstep_group=group):
        ne, nt = gu.check_batch(case, inp, M, B, 0.6, BF16_TOL)
        assert case.builder.get_option("expand_path_taken") == 4
        assert case.builder.get_option("lockstep_speculation_used") == 1
        assert case.builder.get_option("device_error") == 0
    print(f"exact {ne} tolerant {nt}")
    assert ne + nt == batch


def _stress_case(gu):
    cfg = wl.CONFIGS["qwen8b"].replace(embed_std=1.0)
    return gu.get_case("qwen8b-stress", cfg, max_batch=40, max_M=128, max_B=128, k=8)


@pytest.mark.parametrize("batch,M,B,regime", [(32, 64, 32, "peaked"), (32, 64, 32, "flat"), (1, 64, 16, "peaked"), (40, 128, 128, "peaked"),
                                              (9, 64, 100, "flat")])
def test_speculation_full_size_bitwise_equal_to_plain_lockstep(batch, M, B, regime):
    """Full-size shapes with real path dependence (the stress weights of test_wave.py): forced speculation == none, bit for
    bit, through one CUDA graph each (as bench.py times them); three requests also against the oracle."""
    import paper_2607_08642_b200 as dtb
    gu = _gu()
    case = _stress_case(gu)
    T = 0.6
    inp = wl.make_inputs(case.cfg, batch=batch, seed=5100 + B, regime=regime)
    dev = [inp[n].cuda() for n in ("logits", "hidden", "root_tokens", "root_positions")]
    outs = {}
    for spec in (0, 2):
        with _Opts(case, expand_path=4, lockstep_speculation=spec):
            out = dtb.alloc_outputs(batch, B)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                case.builder.build_trees(*dev, M, B, T, out=out, stream=st)
                st.synchronize()
                assert case.builder.get_option("expand_path_taken") == 4
                assert case.builder.get_option("lockstep_speculation_used") == (1 if spec else 0)
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=st):
                    case.builder.build_trees(*dev, M, B, T, out=out, stream=st)
            for t in (out.tokens, out.parents, out.scores, out.mask):
                t.zero_()
            graph.replay()
            graph.replay()                       # round counter, flags and both partial buffers carry over
            torch.cuda.synchronize()
            assert case.builder.get_option("device_error") == 0
            outs[spec] = out
    for name in FIELDS:
        assert torch.equal(getattr(outs[0], name), getattr(outs[2], name)), name
    sub = {k_: v[:3] for k_, v in inp.items()}
    with _Opts(case, expand_path=4, lockstep_speculation=2):
        ne, nt = gu.check_batch(case, sub, M, B, T, BF16_TOL)
    assert ne + nt == min(batch, 3)


def test_many_rounds_alternating_modes_on_one_handle():
    """The hand-over words carry an 8-bit round tag and are never cleared: 600 rounds on one handle (past two wraps of the
    tag), alternating speculation on / off, batch sizes, budgets and regimes, must reproduce each configuration's first
    output bit for bit and never raise the device error word."""
    gu = _gu()
    case = _small(gu, 8)
    confs = [(2, 33, 24, 40, "peaked"), (0, 7, 32, 48, "flat"), (2, 1, 8, 8, "peaked"), (0, 33, 24, 12, "peaked"), (2, 12, 16, 3, "flat")]
    inputs = [wl.make_inputs(case.cfg, batch=c[1], seed=4300 + i, regime=c[4]) for i, c in enumerate(confs)]
    first = {}
    try:
        case.builder.set_option("expand_path", 4)
        for rnd in range(600):
            i = (rnd * 7 + rnd // 5) % len(confs)
            spec, batch, M, B, _ = confs[i]
            case.builder.set_option("lockstep_speculation", spec)
            out = case.run_gpu(inputs[i], M, B, 0.6)
            if i not in first:
                first[i] = out
                continue
            for name in FIELDS:
                assert torch.equal(getattr(first[i], name), getattr(out, name)), (rnd, i, name)
        assert case.builder.get_option("device_error") == 0
    finally:
        case.builder.set_option("expand_path", 0)
        case.builder.set_option("lockstep_speculation", 1)


def test_widest_candidate_set_uses_one_staging_buffer():
    """M = 256 (DT_MAX_M): two staging buffers of W2 rows do not fit a request CTA's shared memory, so the kernel keeps one
    and does not prefetch; the tree still matches the oracle, with and without speculation."""
    gu = _gu()
    case = gu.get_case("qwen8b-m256", wl.CONFIGS["qwen8b"], max_batch=1, max_M=256, max_B=16, k=8)
    inp = wl.make_inputs(case.cfg, batch=1, seed=5500, regime="peaked")
    for spec in (2, 0):
        with _Opts(case, expand_path=4, lockstep_speculation=spec):
            ne, nt = gu.check_batch(case, inp, 256, 16, 0.6, BF16_TOL)
            assert case.builder.get_option("expand_path_taken") == 4
            assert case.builder.get_option("device_error") == 0
        assert ne + nt == 1


def test_speculation_cond_static_arm_unchanged():
    """The Cond-static arm walks the greedy chain with the same kernel (static mode): same trees with and without."""
    gu = _gu()
    case = _stress_case(gu)
    inp = wl.make_inputs(case.cfg, batch=4, seed=5300, regime="peaked")
    outs = {}
    for spec in (0, 2):
        with _Opts(case, scorer=2, lockstep_speculation=spec):
            outs[spec] = case.run_gpu(inp, 64, 16, 0.6)
            assert case.builder.get_option("device_error") == 0
    for name in FIELDS:
        assert torch.equal(getattr(outs[0], name), getattr(outs[2], name)), name


def test_adaptive_round_speculates_on_peaked_inputs_by_default():
    gu = _gu()
    case = _stress_case(gu)
    inp = wl.make_inputs(case.cfg, batch=32, seed=5400, regime="peaked")
    ref = None
    with _Opts(case, expand_path=4, lockstep_speculation=0):
        ref = case.run_gpu(inp, 64, 32, 0.6)
    out = case.run_gpu(inp, 64, 32, 0.6)                     # defaults: adaptive schedule
    assert case.builder.get_option("expand_path_taken") == 6
    assert case.builder.get_option("schedule_chosen") == 0   # 0 = lock-step (peaked round)
    assert case.builder.get_option("lockstep_speculation_used") == 1
    assert case.builder.get_option("device_error") == 0
    for name in FIELDS:
        assert torch.equal(getattr(ref, name), getattr(out, name)), name
