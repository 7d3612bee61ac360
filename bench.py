#!/usr/bin/env python
"""bench.py -- throughput of the DominoTree per-round draft-tree builder on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one whole tree-build round (Algorithm 1: top-M select, per-round
precompute, best-first expansion with the GRU correction, emitter) over one batch of synthetic
requests.  Default workload: BASELINE.json configs[4] / north_star target ("concurrent8b":
Qwen3-8B-shaped, batch 32, V=151936, L=16, d=4096, g=1024, r=256, M=64, B=32, k=8, T=0.6), the
whole round replayed from ONE CUDA graph.  Rank 0 prints one JSON line (see README / DESIGN.md).

Timing: CUDA events on the launching stream around exactly K graph replays after W >= 3 warm-up
replays; R distinct input sets (R x 155.6 MB of logits > the 126 MB L2) are rotated so every
replay reads its logits from HBM; clocks are sampled through NVML during the timed region.
N > 1 (torchrun): requests are independent, every rank builds its own batch with
replicated weights, there is no data-path collective; value = total trees / max-over-ranks time.

--impl reference: no reference implementation exists for this paper, so the reference arm is the
float64 CPU oracle (oracle/) as it stands, timed on the box's host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tree_build_throughput"
UNIT = "trees/s"
FP32_FMA_LANES_PER_SM = 128          # B200 SM: 4 sub-partitions x 32 fp32 lanes (blackwell guide)


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def host_cores() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


def load_peaks():
    """MEASURED_PEAKS.json (driver-written) or the profiling guide's stated fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "bf16_tflops": float(d.get("bf16_tflops", 1590.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "bf16_tflops": 1590.0, "source": "fallback"}


def pctl(xs, q):
    xs = sorted(xs)
    if not xs:
        return None
    i = q * (len(xs) - 1)
    lo = int(i)
    hi = min(lo + 1, len(xs) - 1)
    return xs[lo] + (xs[hi] - xs[lo]) * (i - lo)


# ----------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock / throttle reasons of one GPU through NVML while the timed region runs."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, device_index: int, period_s: float = 0.01):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period, self._stop, self._thr, self._h = period_s, threading.Event(), None, None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            h = None
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(device_index).uuid)
                h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if hasattr(uuid, "encode") else uuid)
            except Exception:
                h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self._h = h
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # pragma: no cover
            log(f"[bench] NVML unavailable ({e}); clocks not sampled")

    def _run(self):
        nv, h = self.nv, self._h
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                bits = int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
                for b, name in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self._h is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------------- workload math
def algorithmic_counts(cfg, batch: int):
    """Algorithmic bytes / flops of one round."""
    esz = 2 if cfg.dtype == "bf16" else 4
    select_bytes = batch * cfg.L * cfg.V * esz + batch * cfg.L * cfg.M * 8
    g, r, M, B = cfg.g, cfg.r, cfg.M, cfg.B
    per_exp = 2 * r * g + 2 * M * r                    # W1s S  +  W2 slice . a
    per_gru = 2 * 3 * g * g                            # W_hh S_parent
    expand_flops = batch * (B * per_exp + (B - 1) * per_gru)
    precompute_flops = 2 * batch * cfg.L * r * cfg.d
    return select_bytes, expand_flops, precompute_flops


# ----------------------------------------------------------------------------------- oracle legs
def oracle_trees(w_cpu, inp, lo, hi, cfg, threads):
    """Run the float64 oracle (as it stands) on requests [lo, hi) of `inp`; returns (trees, seconds)."""
    import oracle
    w_orc = oracle.Weights.from_dict(w_cpu)
    sl = slice(lo, hi)
    t0 = time.perf_counter()
    trees = oracle.build_trees(w_orc, inp["logits"][sl], inp["hidden"][sl], inp["root_tokens"][sl],
                               inp["root_positions"][sl], cfg.M, cfg.B, cfg.k, cfg.T, threads=threads)
    return trees, time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores; each step = `cores` requests of the
    workload (one per thread).  Under torchrun only rank 0 works."""
    from paper_2607_08642_b200 import workloads as wl
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    cfg = wl.CONFIGS[args.workload]
    cores = host_cores()
    n_req = min(cfg.batch, cores)
    log(f"[bench/reference] generating weights for {cfg.name} ...")
    w_cpu = wl.make_weights(cfg)
    inp = wl.make_inputs(cfg, batch=n_req, regime="flat")
    inp2 = wl.make_inputs(cfg, batch=n_req, regime="peaked", seed=cfg.seed + 64)
    sets = [inp, inp2]
    # bound the run: if K steps of `cores` concurrent requests would exceed ~150 s, one request per step
    _, t_par = oracle_trees(w_cpu, sets[0], 0, n_req, cfg, cores)
    if t_par * (args.steps + args.warmup) > 150.0:
        n_req = 1
    for i in range(args.warmup):
        oracle_trees(w_cpu, sets[i % 2], 0, n_req, cfg, cores)
    total = 0.0
    for i in range(args.steps):
        _, dt_s = oracle_trees(w_cpu, sets[i % 2], 0, n_req, cfg, cores)
        total += dt_s
    ms_per_step = 1e3 * total / max(args.steps, 1)
    value = n_req / (ms_per_step / 1e3)
    sample = f"{n_req} requests per step (one per host thread) of {cfg.name}, flat/peaked alternating"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "batch": n_req, "V": cfg.V, "L": cfg.L, "d": cfg.d, "g": cfg.g, "r": cfg.r,
                   "M": cfg.M, "B": cfg.B, "k": cfg.k, "T": cfg.T, "note": "CPU float64 oracle, bounded sample"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------- CUDA arm
def run_ours(args):
    import torch
    import paper_2607_08642_b200 as dtb
    from paper_2607_08642_b200 import build as dtbuild
    from paper_2607_08642_b200 import dist as dtdist
    from paper_2607_08642_b200 import workloads as wl

    rank, local_rank, world = dtdist.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path (use --impl reference "
                         "for the CPU oracle)")
    dev = local_rank % torch.cuda.device_count()
    torch.cuda.set_device(dev)
    if world > 1:
        dtdist.init_process_group("nccl")
    if rank == 0:
        dtbuild.build()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    peaks = load_peaks()
    cfg = wl.CONFIGS[args.workload]
    batch, M, B, T = cfg.batch, cfg.M, cfg.B, cfg.T
    R = args.rotate
    t0 = time.perf_counter()
    w_cpu = wl.make_weights(cfg)
    w_gpu = {n: t.cuda() for n, t in w_cpu.items()}
    log(f"[bench r{rank}] weights for {cfg.name} generated in {time.perf_counter() - t0:.1f}s")
    t0 = time.perf_counter()
    builder = dtb.DominoTreeBuilder(w_gpu, max_batch=batch, L=cfg.L, max_M=M, max_B=B, k=cfg.k)
    torch.cuda.synchronize()
    create_s = time.perf_counter() - t0
    log(f"[bench r{rank}] dt_create {create_s:.2f}s, workspace {builder.workspace_bytes / 2**20:.1f} MiB")

    # R distinct input sets, flat / peaked alternating; per-rank seeds
    sets_cpu, sets = [], []
    for i in range(R):
        inp = wl.make_inputs(cfg, batch=batch, seed=cfg.seed + 64 * (rank * R + i),
                             regime="flat" if i % 2 == 0 else "peaked")
        sets_cpu.append(inp)
        sets.append({k_: inp[k_].cuda() for k_ in ("logits", "hidden", "root_tokens", "root_positions")})
    outs = [dtb.alloc_outputs(batch, B) for _ in range(R)]
    st = torch.cuda.Stream()

    def enqueue(i):
        s = sets[i]
        builder.build_trees(s["logits"], s["hidden"], s["root_tokens"], s["root_positions"], M, B, T,
                            out=outs[i], stream=st)

    def capture(i):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            enqueue(i)
        return g

    with torch.cuda.stream(st):
        for i in range(R):
            enqueue(i)
        st.synchronize()
        launches_per_round = builder.kernel_launches
        graphs = [capture(i) for i in range(R)]             # clean graphs: the timed region
        builder.phase_timing(R)
        ph_graphs = []
        for i in range(R):                                  # same round + phase-boundary event nodes
            builder.phase_slot(i)
            ph_graphs.append(capture(i))
        builder.phase_slot(0)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    W, K = max(args.warmup, 3), args.steps
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(st):
        for i in range(W):
            graphs[i % R].replay()
        barrier()
        with ClockSampler(dev) as clk:
            ev0.record(st)
            for i in range(K):
                graphs[i % R].replay()
            ev1.record(st)
            barrier()
        ms_total = ev0.elapsed_time(ev1)
    ms_total = dtdist.max_over_ranks(ms_total, device="cuda" if world > 1 else "cpu")
    ms_per_step = ms_total / K
    value = batch * world / (ms_per_step / 1e3)

    # per-phase device times: K replays of the event-carrying graphs, read after each replay
    phase_sum = {n: 0.0 for n in dtb.PHASES}
    Kp = min(K, 100)
    with torch.cuda.stream(st):
        ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tot_ph = 0.0
        for i in range(Kp):
            ev2.record(st)
            ph_graphs[i % R].replay()
            ev3.record(st)
            st.synchronize()
            tot_ph += ev2.elapsed_time(ev3)
            for n, v in builder.phase_ms(i % R).items():
                phase_sum[n] += v
    phases_us = {n: 1e3 * v / Kp for n, v in phase_sum.items()}
    phase_round_us = 1e3 * tot_ph / Kp

    # distribution over the replays: one event between consecutive replays (a separate pass: the timed region above is
    # bracketed by exactly two events), and the split by input regime (even sets flat, odd sets peaked)
    with torch.cuda.stream(st):
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
        evs[0].record(st)
        for i in range(K):
            graphs[i % R].replay()
            evs[i + 1].record(st)
        st.synchronize()
    per = [1e3 * evs[i].elapsed_time(evs[i + 1]) for i in range(K)]
    by_regime = {"flat": [per[i] for i in range(K) if (i % R) % 2 == 0], "peaked": [per[i] for i in range(K) if (i % R) % 2 == 1]}
    dist_us = {"p10": pctl(per, 0.1), "p50": pctl(per, 0.5), "p90": pctl(per, 0.9),
               "by_regime_p50": {n: pctl(v, 0.5) for n, v in by_regime.items() if v}}
    schedule = {}
    with torch.cuda.stream(st):
        for i in range(R):
            graphs[i].replay()
            st.synchronize()
            if builder.get_option("expand_path_taken") == 6:
                schedule["flat" if i % 2 == 0 else "peaked"] = "wavefront" if (builder.get_option("schedule_chosen") or B >= 48) else "lock-step"
                if builder.get_option("schedule_chosen"):
                    schedule["wavefront_steps_request0"] = builder.get_option("wave_steps")

    # the select kernel's own duration inside the round: device-side span (first CTA start .. last CTA end, %globaltimer),
    # free of the launch / event latency a CUDA-event pair around ONE kernel of a graph includes
    span_us = None
    try:
        builder.set_option("select_span", 1)
        with torch.cuda.stream(st):
            sg = [capture(i) for i in range(R)]
            tot_ns = 0
            for i in range(4 * R):
                sg[i % R].replay()
                st.synchronize()
                tot_ns += builder.get_option("select_span_ns")
        span_us = tot_ns / (4 * R) / 1e3
    finally:
        builder.set_option("select_span", 0)

    # select alone, back to back on the rotating buffers (dt_select_topm)
    ids = torch.empty((batch * cfg.L, M), dtype=torch.int32, device="cuda")
    vals = torch.empty((batch * cfg.L, M), dtype=torch.float32, device="cuda")
    with torch.cuda.stream(st):
        for i in range(R):
            builder.select_topm_into(sets[i]["logits"], M, ids, vals, stream=st)
        ev2.record(st)
        for i in range(40):
            builder.select_topm_into(sets[i % R]["logits"], M, ids, vals, stream=st)
        ev3.record(st)
        st.synchronize()
    select_alone_us = 1e3 * ev2.elapsed_time(ev3) / 40
    # L2-warm: the same 4 requests (64 rows, 19.4 MB) over and over
    warm_rows = min(batch, 4) * cfg.L
    with torch.cuda.stream(st):
        wl_ = sets[0]["logits"][:min(batch, 4)]
        for i in range(5):
            builder.select_topm_into(wl_, M, ids[:warm_rows], vals[:warm_rows], stream=st)
        ev2.record(st)
        for i in range(40):
            builder.select_topm_into(wl_, M, ids[:warm_rows], vals[:warm_rows], stream=st)
        ev3.record(st)
        st.synchronize()
    select_warm_us = 1e3 * ev2.elapsed_time(ev3) / 40

    return dict(torch=torch, dtb=dtb, wl=wl, cfg=cfg, rank=rank, world=world, dev=dev, peaks=peaks, builder=builder,
                w_cpu=w_cpu, sets_cpu=sets_cpu, sets=sets, outs=outs, graphs=graphs, st=st, R=R, W=W, K=K,
                ms_per_step=ms_per_step, value=value, clocks=clk.summary(), phases_us=phases_us,
                phase_round_us=phase_round_us, select_alone_us=select_alone_us, select_warm_us=select_warm_us,
                select_warm_rows=warm_rows, select_span_us=span_us, dist_us=dist_us, schedule=schedule,
                launches_per_round=launches_per_round, create_s=create_s, barrier=barrier)


def measure_e2e(ctx, steps: int):
    """Same metric through the public host-buffer API (dt_build_trees_host): pinned host inputs are
    copied host->device, the round runs, the outputs are copied back, every step, inside the timed
    region (wall clock around synchronous calls, max over ranks)."""
    torch, dtb, cfg, builder, st = ctx["torch"], ctx["dtb"], ctx["cfg"], ctx["builder"], ctx["st"]
    from paper_2607_08642_b200 import dist as dtdist
    batch, M, B, T, R = cfg.batch, cfg.M, cfg.B, cfg.T, ctx["R"]
    pinned = []
    for inp in ctx["sets_cpu"]:
        pinned.append({k_: inp[k_].pin_memory() for k_ in ("logits", "hidden", "root_tokens", "root_positions")})
    out_h = dtb.alloc_outputs(batch, B, "cpu", pin=True)

    def one(i):
        s = pinned[i % R]
        builder.build_trees_host(s["logits"], s["hidden"], s["root_tokens"], s["root_positions"], M, B, T,
                                 out=out_h, stream=st)
    for i in range(3):
        one(i)
    ctx["barrier"]()
    t0 = time.perf_counter()
    for i in range(steps):
        one(i)
    ctx["barrier"]()
    sec = time.perf_counter() - t0
    sec = dtdist.max_over_ranks(sec, device="cuda" if ctx["world"] > 1 else "cpu")
    s0 = pinned[0]
    h2d = sum(s0[k_].numel() * s0[k_].element_size() for k_ in s0)
    d2h = sum(t.numel() * t.element_size() for t in (out_h.tokens, out_h.parents, out_h.depths, out_h.positions,
                                                     out_h.scores, out_h.mask, out_h.n_nodes))
    return {"value": batch * ctx["world"] * steps / sec, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
            "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * sec / steps, "steps": steps}


def measure_cpu_baseline(ctx):
    """The oracle, as it stands, on the host cores: the first n requests of input set 0 (one request
    per thread); its trees are also compared with what the CUDA path produced for the same requests."""
    import numpy as np
    cfg, torch = ctx["cfg"], ctx["torch"]
    cores = host_cores()
    n = min(cfg.batch, max(cores, 8))
    trees, sec = oracle_trees(ctx["w_cpu"], ctx["sets_cpu"][0], 0, n, cfg, cores)
    with torch.cuda.stream(ctx["st"]):
        ctx["graphs"][0].replay()
        ctx["st"].synchronize()
    out = ctx["outs"][0]
    tok, par, sc = out.tokens.cpu().numpy(), out.parents.cpu().numpy(), out.scores.cpu().numpy()
    exact, max_dscore = 0, 0.0
    for b, tr in enumerate(trees):
        same = np.array_equal(tok[b], tr.tokens) and np.array_equal(par[b], tr.parents)
        exact += bool(same)
        if same:
            max_dscore = max(max_dscore, float(np.max(np.abs(sc[b][:tr.n_nodes] - tr.scores[:tr.n_nodes]))))
    _, sec1 = oracle_trees(ctx["w_cpu"], ctx["sets_cpu"][0], 0, 1, cfg, 1)
    base = {"value": n / sec, "unit": UNIT, "cores": cores, "kind": "oracle", "single_thread_value": 1.0 / sec1,
            "single_thread_s_per_tree": sec1,
            "sample": f"requests 0..{n - 1} of input set 0 of {cfg.name} (flat regime), one request per thread, "
                      f"{sec:.2f}s wall"}
    parity = {"requests": n, "tokens_parents_exact": exact, "max_abs_score_diff_on_exact": max_dscore,
              "note": "near-tie reorderings (< 1e-4) are accepted by tests/compare.py, not counted here"}
    return base, parity


def measure_batch1(ctx):
    """Context numbers for BASELINE.json configs[2]/[3]: batch 1, M=64, B in {16, 32}, same weights;
    one CUDA graph per (B, input), 64 rotating inputs (311 MB of logits > L2)."""
    torch, dtb, wl, cfg, st = ctx["torch"], ctx["dtb"], ctx["wl"], ctx["cfg"], ctx["st"]
    builder = ctx["builder"]
    out = {}
    n_in = 64
    lg = torch.cat([s["logits"] for s in ctx["sets"]])[:n_in]
    hd = torch.cat([s["hidden"] for s in ctx["sets"]])[:n_in]
    rt = torch.cat([s["root_tokens"] for s in ctx["sets"]])[:n_in]
    rp = torch.cat([s["root_positions"] for s in ctx["sets"]])[:n_in]
    n_in = lg.shape[0]
    for B in (16, 32):
        if B > builder.max_B:
            continue
        o = dtb.alloc_outputs(1, B)
        graphs = []
        with torch.cuda.stream(st):
            builder.build_trees(lg[0:1], hd[0:1], rt[0:1], rp[0:1], cfg.M, B, 0.0, out=o, stream=st)
            st.synchronize()
            for i in range(n_in):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=st):
                    builder.build_trees(lg[i:i + 1], hd[i:i + 1], rt[i:i + 1], rp[i:i + 1], cfg.M, B, 0.0, out=o, stream=st)
                graphs.append(g)
            for i in range(n_in):
                graphs[i].replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for i in range(2 * n_in):
                graphs[i % n_in].replay()
            e1.record(st)
            st.synchronize()
        us = 1e3 * e0.elapsed_time(e1) / (2 * n_in)
        out[f"B{B}"] = {"us_per_round": us, "trees_per_s": 1e6 / us}
    return out


def _time_graphs(torch, dtb, builder, st, lg, hd, rt, rp, M, B, T):
    """us per round of batch-1 rounds, one CUDA graph per input, inputs rotated (working set > L2)."""
    n_in = lg.shape[0]
    o = dtb.alloc_outputs(1, B)
    graphs = []
    with torch.cuda.stream(st):
        builder.build_trees(lg[0:1], hd[0:1], rt[0:1], rp[0:1], M, B, T, out=o, stream=st)
        st.synchronize()
        for i in range(n_in):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                builder.build_trees(lg[i:i + 1], hd[i:i + 1], rt[i:i + 1], rp[i:i + 1], M, B, T, out=o, stream=st)
            graphs.append(g)
        for g in graphs:
            g.replay()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for i in range(2 * n_in):
            graphs[i % n_in].replay()
        e1.record(st)
        st.synchronize()
    return 1e3 * e0.elapsed_time(e1) / (2 * n_in)


def measure_sweep_and_arms(ctx):
    """--sweep: BASELINE configs[3] (batch 1, B in {16,32,64,128} x M in {32,64,128}, T = 0) and the three scorer
    arms of PAPER.md:553-555 at batch 1, B = 16, M = 64, on the bench's weights; 64 rotating inputs per point."""
    torch, dtb, wl, cfg, st = ctx["torch"], ctx["dtb"], ctx["wl"], ctx["cfg"], ctx["st"]
    w_gpu = {n: t.cuda() for n, t in ctx["w_cpu"].items()}
    builder = dtb.DominoTreeBuilder(w_gpu, max_batch=1, L=cfg.L, max_M=128, max_B=128, k=cfg.k)
    n_in = 64
    lg = torch.cat([s["logits"] for s in ctx["sets"]])[:n_in]
    hd = torch.cat([s["hidden"] for s in ctx["sets"]])[:n_in]
    rt = torch.cat([s["root_tokens"] for s in ctx["sets"]])[:n_in]
    rp = torch.cat([s["root_positions"] for s in ctx["sets"]])[:n_in]
    sweep = {}
    for M in (32, 64, 128):
        for B in (16, 32, 64, 128):
            sweep[f"M{M}_B{B}"] = _time_graphs(torch, dtb, builder, st, lg, hd, rt, rp, M, B, 0.0)
    arms = {}
    for scorer, name in ((0, "dominotree"), (1, "marg"), (2, "cond_static")):
        builder.set_option("scorer", scorer)
        arms[name] = _time_graphs(torch, dtb, builder, st, lg, hd, rt, rp, 64, 16, 0.0)
    builder.set_option("scorer", 0)
    builder.close()
    # the frontier schedule (dt_set_option "schedule" 1: the wavefront kernel at its maximal width) beside the adaptive heap
    # schedule at the bench workload, and the select kernel over chunk counts and candidate widths
    big = ctx["builder"]
    s0 = ctx["sets"][0]
    sched = {}
    for name, val in (("adaptive", 0), ("frontier", 1)):
        big.set_option("schedule", val)
        o = dtb.alloc_outputs(cfg.batch, cfg.B)
        with torch.cuda.stream(st):
            big.build_trees(s0["logits"], s0["hidden"], s0["root_tokens"], s0["root_positions"], cfg.M, cfg.B, cfg.T, out=o, stream=st)
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                big.build_trees(s0["logits"], s0["hidden"], s0["root_tokens"], s0["root_positions"], cfg.M, cfg.B, cfg.T, out=o, stream=st)
            for _ in range(3):
                g.replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for _ in range(20):
                g.replay()
            e1.record(st)
            st.synchronize()
        sched[name] = 1e3 * e0.elapsed_time(e1) / 20
    big.set_option("schedule", 0)
    sel = {}
    ids = torch.empty((cfg.batch * cfg.L, cfg.M), dtype=torch.int32, device="cuda")
    vals = torch.empty((cfg.batch * cfg.L, cfg.M), dtype=torch.float32, device="cuda")
    for S in (1, 2, 4):
        big.set_option("select_chunks", S)
        with torch.cuda.stream(st):
            for i in range(ctx["R"]):
                big.select_topm_into(ctx["sets"][i]["logits"], cfg.M, ids, vals, stream=st)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for i in range(20):
                big.select_topm_into(ctx["sets"][i % ctx["R"]]["logits"], cfg.M, ids, vals, stream=st)
            e1.record(st)
            st.synchronize()
        sel[f"chunks_per_row_{S}"] = 1e3 * e0.elapsed_time(e1) / 20
    big.set_option("select_chunks", 0)
    sweep["schedules_at_bench_workload_flat_set"] = sched
    sweep["select_us_by_chunks"] = sel
    return {"us_per_round": sweep, "note": "batch 1, flat / peaked inputs mixed, one CUDA graph per round"}, \
           {"us_per_round_batch1_B16_M64": arms}



# ----------------------------------------------------------------------------------- in-kernel timeline
# (stamp index, what has happened by then), in program order, for GRU CTA 0 / request CTA 0 (dt_wave.cuh WV_TR)
GRU_STAMPS = ((0, "items polled + compacted"), (1, "pass begins"), (2, "P / previous-state loads issued"), (14, "producer thread 128: sources computed"), (15, "producer thread 128: first group issued"),
              (8, "issuer 0: first K chunk landed"), (9, "issuer 0: all tcgen05.mma + commit issued"), (3, "D1 complete (mbarrier)"),
              (10, "TMEM loads, hi + lo shuffles, gates"), (11, "global + DSMEM state stores issued"), (12, "cluster barrier"),
              (4, "proxy fence + CTA barrier"), (13, "thread 0: D2 tcgen05.mma + commit issued"), (5, "D2 complete (mbarrier)"),
              (6, "partials stored + CTA barrier"), (7, "gpu fence + flag store"))
REQ_STAMPS = ((0, "flags seen"), (1, "a = SiLU(C + partials)"), (2, "W2 slice dots"), (10, "top-k: threshold from the lane maxima (warp 0)"),
              (11, "top-k: ranks among the keys above it, log-softmax (warp 0)"), (3, "CTA barrier after the top-k"),
              (6, "merge into the sorted frontier"), (9, "nominate + publish (warp 0)"), (4, "CTA barrier"),
              (5, "slices staged (issue)"))


FUSED_GRU_STAMPS = ((0, "descriptors seen + CTA barrier"), (1, "state copies, P / previous-state loads issued"), (3, "D1 complete (copies landed, tcgen05.mma, mbarrier)"),
                    (10, "TMEM -> shared + CTA barrier"), (11, "gates, state stores, W1 operand + CTA barrier"), (5, "D2 issued and complete"),
                    (6, "partials stored + CTA barrier"), (7, "gpu fence + flag store"))
FUSED_REQ_STAMPS = ((0, "flags seen"), (1, "a = SiLU(C + partials)"), (2, "W2 slice dots + online softmax statistics"), (3, "top-k + CTA barrier"),
                    (9, "pop: next descriptor published (thread 0)"), (4, "CTA barrier, then warp 0: next flags seen (warps 1-7 merge + stage meanwhile)"))


def run_trace(args):
    """--trace: the measurement build libdominotree_trace.so (-DDT_TRACE) stamps %globaltimer inside the wavefront
    kernel (GRU CTA 0, request CTA 0); prints the median time between consecutive stamps per regime as one JSON line.
    Never a bench value: the stamps perturb the kernel slightly."""
    import ctypes
    import numpy as np
    import torch
    import paper_2607_08642_b200 as dtb
    from paper_2607_08642_b200 import build as dtbuild
    from paper_2607_08642_b200 import workloads as wl
    lib_path = dtbuild.build(trace=True)
    cfg = wl.CONFIGS[args.workload]
    batch = args.trace_batch or cfg.batch
    w_gpu = {n: t.cuda() for n, t in wl.make_weights(cfg).items()}
    builder = dtb.DominoTreeBuilder(w_gpu, max_batch=batch, L=cfg.L, max_M=cfg.M, max_B=cfg.B, k=cfg.k, lib_path=lib_path)
    fused = (args.trace_path == 4)
    builder.set_option("expand_path", args.trace_path)   # the timeline of ONE kernel, whatever the adaptive schedule would pick
    if not fused:
        builder.set_option("wave_groups", 1)      # one request group: GRU step i and request step i are the same step
    else:
        # speculation (the default) makes GRU pass i and request step i different things: the plain chain (one pass per
        # step, two request groups) unless --trace-spec; with it only the per-role segments and the periods are meaningful
        builder.set_option("lockstep_speculation", 2 if args.trace_spec else 0)
    gru_stamps, req_stamps = (FUSED_GRU_STAMPS, FUSED_REQ_STAMPS) if fused else (GRU_STAMPS, REQ_STAMPS)
    if args.wave_width:
        builder.set_option("wave_width", args.wave_width)
    lib = builder.lib
    lib.dt_trace_read.argtypes = [ctypes.c_void_p]
    lib.dt_trace_read.restype = ctypes.c_int
    S, K = 64, 16
    buf = np.zeros((2, S, K), dtype=np.uint64)
    out = {"workload": cfg.name, "batch": batch, "kernel": ("fused_expand_kernel<0> (lock-step, speculation, one request group)" if args.trace_spec else "fused_expand_kernel<0> (lock-step, no speculation, two request groups)") if fused else "wave_expand_kernel (one request group)",
           "wave_width": args.wave_width or "auto", "unit": "ns (median over steps)"}
    for regime in ("flat", "peaked"):
        inp = wl.make_inputs(cfg, batch=batch, regime=regime)
        dev = {k_: inp[k_].cuda() for k_ in ("logits", "hidden", "root_tokens", "root_positions")}
        o = dtb.alloc_outputs(batch, cfg.B)
        for _ in range(3):
            builder.build_trees(dev["logits"], dev["hidden"], dev["root_tokens"], dev["root_positions"], cfg.M, cfg.B, cfg.T, out=o)
        torch.cuda.synchronize()
        assert lib.dt_trace_read(buf.ctypes.data) == 0
        builder.build_trees(dev["logits"], dev["hidden"], dev["root_tokens"], dev["root_positions"], cfg.M, cfg.B, cfg.T, out=o)
        torch.cuda.synchronize()
        assert lib.dt_trace_read(buf.ctypes.data) == 0
        t = buf.astype(np.int64)
        steps = int((t[0, :S - 1, 0] > 0).sum())
        rows = {}
        g = t[0, 1:max(steps - 1, 2)]          # skip step 0 (weight load) and the last
        q = t[1, 1:max(steps - 1, 2)]
        for role, arr, stamps in (("gru", g, gru_stamps), ("req", q, req_stamps)):
            for (i0, _), (i1, name) in zip(stamps[:-1], stamps[1:]):
                ok = (arr[:, i1] > 0) & (arr[:, i0] > 0)
                rows[f"{role}: {name}"] = float(np.median((arr[:, i1] - arr[:, i0])[ok])) if ok.any() else None
        ok = (q[:, 0] > 0) & (g[:, 7] > 0)
        rows["hop: flag released -> request sees flags"] = float(np.median((q[:, 0] - g[:, 7])[ok])) if ok.any() else None
        spec_on = fused and args.trace_spec
        if spec_on:
            rows["hop: flag released -> request sees flags"] = None
        gn = t[0, 2:max(steps, 3)]
        ok = (gn[:, 0] > 0) & (q[:len(gn), 9] > 0)
        rows["hop: request published -> GRU sees headers"] = float(np.median((gn[:, 0] - q[:len(gn), 9])[ok])) if ok.any() and not spec_on else None
        if spec_on:
            rq = t[1, 1:min(cfg.B, S - 1), 0]
            rq = rq[rq > 0]
            rows["request step period"] = float(np.median(np.diff(rq))) if len(rq) > 1 else None
            rows["gru_passes_request0"] = builder.get_option("wave_steps")
            t00 = int(t[0, 0, 0])                                  # absolute timeline of the first passes / steps (ns)
            rows["timeline_gru_pass_begins"] = [int(x - t00) for x in t[0, :14, 0] if x > 0]
            rows["timeline_gru_flag_stored"] = [int(x - t00) for x in t[0, :14, 7] if x > 0]
            rows["timeline_req_flags_seen"] = [int(x - t00) for x in t[1, :14, 0] if x > 0]
            rows["timeline_req_published"] = [int(x - t00) for x in t[1, :14, 9] if x > 0]
            rows["gru_passes_max"] = builder.get_option("wave_expansions")
        kt = t[:, S - 1, :]                      # kernel-level stamps: entry, loop begins, loop ends, (request CTA) emitted
        def span(r0, i0, r1, i1):
            return float(kt[r1, i1] - kt[r0, i0]) if kt[r1, i1] > 0 and kt[r0, i0] > 0 else None
        rows["kernel: GRU CTA 0 entry -> weights resident, step loop begins"] = span(0, 0, 0, 1)
        rows["kernel: request CTA 0 entry -> root staged, step loop begins"] = span(1, 0, 1, 1)
        rows["kernel: GRU CTA 0 step loop"] = span(0, 1, 0, 2)
        rows["kernel: request CTA 0 step loop"] = span(1, 1, 1, 2)
        rows["kernel: request CTA 0 emitter (tokens .. mask)"] = span(1, 2, 1, 3)
        rows["kernel: GRU CTA 0 entry -> request CTA 0 done"] = span(0, 0, 1, 3)
        period = np.diff(t[0, 1:steps, 0])
        rows["step period"] = float(np.median(period)) if len(period) else None
        rows["steps"] = steps
        rows["expansions_request0"] = cfg.B if fused else builder.get_option("wave_expansions")
        out[regime] = rows
    print(json.dumps({"trace": out}), flush=True)
    builder.close()


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", default="concurrent8b")
    ap.add_argument("--rotate", type=int, default=4, help="distinct input sets rotated through the timed region")
    ap.add_argument("--no-extras", action="store_true", help="skip the e2e / cpu_baseline / batch-1 legs")
    ap.add_argument("--sweep", action="store_true", help="also time the batch-1 B x M sweep and the three scorer arms")
    ap.add_argument("--trace", action="store_true", help="in-kernel timeline of the wavefront kernel (measurement build, not a bench value)")
    ap.add_argument("--trace-batch", type=int, default=0, help="batch of the --trace leg (default: the workload's)")
    ap.add_argument("--trace-spec", action="store_true", help="--trace --trace-path 4 with the speculation on (one request group)")
    ap.add_argument("--trace-path", type=int, default=5, choices=(4, 5), help="kernel of the --trace leg: 5 = wavefront (default), 4 = lock-step fused")
    ap.add_argument("--wave-width", type=int, default=0, help="nodes a request may expand per step (0 = auto)")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.steps == 200 and args.warmup == 20:      # defaults: keep the CPU run within minutes
            args.steps, args.warmup = 10, 3
        return run_reference(args)
    if args.trace:
        return run_trace(args)

    ctx = run_ours(args)
    cfg, peaks, world, rank = ctx["cfg"], ctx["peaks"], ctx["world"], ctx["rank"]
    batch = cfg.batch
    sel_bytes, exp_flops, pre_flops = algorithmic_counts(cfg, batch)
    ph = ctx["phases_us"]
    round_us = 1e3 * ctx["ms_per_step"]
    # select: the kernel's duration inside the round = its device-side span; the CUDA-event phase (which also holds the launch
    # and event latency of the graph's first node) and the back-to-back figure are reported beside it
    sel_us = ctx["select_span_us"] or ph["select"]
    sel_gbs = sel_bytes / (sel_us * 1e-6) / 1e9
    # `traffic`: dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full captures summarised under
    # profiles/ (C5 workload only; None for any other workload): a constant of that capture, not measured by this run
    c5 = (cfg.name == "concurrent8b")
    roof_select = {"kernel": "select_topm_bulk_kernel", "bound": "hbm", "achieved": sel_gbs, "peak": peaks["hbm_gbs"],
                   "unit": "GB/s", "frac": sel_gbs / peaks["hbm_gbs"], "traffic": 161.90e6 if c5 else None,
                   "traffic_source": "profiles/r2_select_ncu.md (ncu --set full, one launch)" if c5 else None,
                   "peak_source": peaks["source"], "algorithmic_bytes": sel_bytes, "us_per_launch": sel_us,
                   "how": "device-side span of the kernel inside the round (L2 defeated by rotating inputs)",
                   "us_event_phase": ph["select"], "gbs_event_phase": sel_bytes / (ph["select"] * 1e-6) / 1e9,
                   "share_of_step": sel_us / ctx["phase_round_us"],
                   "alone_back_to_back_gbs": sel_bytes / (ctx["select_alone_us"] * 1e-6) / 1e9,
                   "alone_back_to_back_frac": sel_bytes / (ctx["select_alone_us"] * 1e-6) / 1e9 / peaks["hbm_gbs"],
                   "l2_warm": {"rows": ctx["select_warm_rows"], "us": ctx["select_warm_us"],
                               "gbs": ctx["select_warm_rows"] * cfg.V * 2 / (ctx["select_warm_us"] * 1e-6) / 1e9}}
    fma_peak_tflops = 148 * FP32_FMA_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    exp_tflops = exp_flops / (ph["expand"] * 1e-6) / 1e12
    # the expansion is a chain of dependent steps: neither fraction is a target, the microseconds per step are
    roof_expand = {"kernel": "expansion phase (wave_expand_kernel or fused_expand_kernel<0>, chosen per round on the device)",
                   "bound": "latency", "achieved": exp_tflops, "unit": "TFLOP/s",
                   "peak": fma_peak_tflops, "frac": exp_tflops / fma_peak_tflops,
                   "peak_source": "148 SMs x 128 fp32 FMA lanes x 2 x sm_max_mhz (DESIGN.md)",
                   "frac_of_bf16_tensor_peak": exp_tflops / peaks["bf16_tflops"],
                   "bf16_tensor_peak": peaks["bf16_tflops"],
                   "traffic": 30.6e6, "traffic_source": "profiles/r2_fused_ncu.md (ncu --set full of the lock-step kernel on a peaked round: "
                                                        "dram read 30.0 MB + write 0.6 MB; the wavefront kernel cannot be replayed by ncu)",
                   "algorithmic_flops": exp_flops, "us_per_round": ph["expand"],
                   "share_of_step": ph["expand"] / ctx["phase_round_us"], "schedule": ctx["schedule"],
                   "us_per_round_by_regime_p50": ctx["dist_us"]["by_regime_p50"],
                   "note": "a chain of dependent GRU -> correction -> pop steps (lock-step: ~34 GRU passes for 32 nodes, the pass of "
                           "the likely next node speculated while its parent is scored; wavefront: ~9 steps of ~4 nodes per "
                           "request): latency-bound; 92 % of the flops run as bf16 hi/lo pairs on tcgen05"}
    dominant = roof_expand if ph["expand"] > sel_us else roof_select

    line = {
        "metric": METRIC, "value": ctx["value"], "unit": UNIT, "n_gpus": world, "steps": ctx["K"], "warmup": ctx["W"],
        "ms_per_step": ctx["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "batch_per_gpu": batch, "V": cfg.V, "L": cfg.L, "d": cfg.d, "g": cfg.g,
                   "r": cfg.r, "M": cfg.M, "B": cfg.B, "k": cfg.k, "T": cfg.T, "input_dtype": cfg.dtype,
                   "launch": "one CUDA graph per round", "parallelism": f"dp{world} (independent requests, no collective)",
                   "l2": f"{ctx['R']} distinct input sets rotated ({ctx['R']} x {sel_bytes / 1e6:.1f} MB logits > 126 MB L2)",
                   "regimes": "flat / peaked alternating"},
        "us_per_round": round_us, "us_per_round_dist": ctx["dist_us"],
        "phases_us": ph, "phase_pass_us_per_round": ctx["phase_round_us"],
        "select_hbm_gbs": sel_gbs,
        "roofline": dominant, "roofline_select": roof_select, "roofline_expand": roof_expand,
        "clocks": ctx["clocks"], "gpu_launches": int(ctx["launches_per_round"] * ctx["K"]),
        "launches_per_round": int(ctx["launches_per_round"]), "create_s": ctx["create_s"],
    }
    if not args.no_extras:
        line["e2e"] = measure_e2e(ctx, min(ctx["K"], 20))
        if rank == 0 and world == 1:
            line["cpu_baseline"], line["parity_sample"] = measure_cpu_baseline(ctx)
            line["batch1"] = measure_batch1(ctx)
            if args.sweep:
                line["sweep"], line["arms"] = measure_sweep_and_arms(ctx)
    if rank == 0:
        print(json.dumps(line), flush=True)
    ctx["builder"].close()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
