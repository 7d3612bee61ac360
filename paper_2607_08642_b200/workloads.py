"""Seeded synthetic workloads for the DominoTree tree builder.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path: it draws random tensors and nothing else.  It contains none of the
method's arithmetic (no GRU, no correction, no softmax, no selection), imports
neither the oracle nor the CUDA binding, and always draws on the CPU with a
seeded ``torch.Generator`` so that the same bits are produced on every machine;
the CUDA path receives copies of exactly these bits.

The inputs stand in for the paper's Qwen3-4B / Qwen3-8B workloads (PAPER.md:175,
185: block size 16, budget 16, M=64, branching 8, |V|=151,936 PAPER.md:133), whose
checkpoints and datasets are not available: only shapes, dtypes and rough
peakedness are imitated.  Recipe (BASELINE.json ``configs``; DESIGN.md "Input
recipe"; second parameter of N(.,.) is a standard deviation):

* token embeddings  E      [V, d]    ~ N(0, 0.02)
* GRU               W_ih   [3g, d]   ~ N(0, 1/sqrt(d)),  W_hh [3g, g] ~ N(0, 1/sqrt(g))
* correction head   W1     [r, d+g]  ~ N(0, 1/sqrt(d+g)), W2  [V, r]  ~ N(0, 1/sqrt(r))
* backbone hidden   H      [batch, L, d] ~ N(0, 1)
* marginal logits          [batch, L, V] ~ N(0, 3) plus one planted token per
  position of height h (h = 8 for the tiny config, h = clip(6 + 1.5*Gumbel, 4, 10)
  for the Qwen shapes).  Two regimes: ``flat``  x[t] += h   (literal text) and
  ``peaked`` x[t] = row_max + h  (a real peak, Domino-like sharp rows).
* root tokens uniform in [0, V).

Everything is rounded to the config dtype (bf16 or fp32) once, here.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict

import torch

MASTER_SEED = 8642


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    idx: int            # config index c -> seed MASTER_SEED + 1000*c
    batch: int
    V: int
    L: int
    d: int
    g: int
    r: int
    M: int
    B: int
    k: int
    T: float
    dtype: str          # "bf16" | "f32"
    regime: str = "flat"
    embed_std: float = 0.02
    planted: str = "gumbel"   # "gumbel" | "fixed8"

    @property
    def seed(self) -> int:
        return MASTER_SEED + 1000 * self.idx

    def replace(self, **kw) -> "Config":
        return dataclasses.replace(self, **kw)

    @property
    def torch_dtype(self):
        return torch.bfloat16 if self.dtype == "bf16" else torch.float32


QWEN_V = 151936

CONFIGS: Dict[str, Config] = {
    # BASELINE.json configs[0]
    "tiny": Config("tiny", 0, batch=1, V=1024, L=4, d=64, g=32, r=32, M=8, B=8, k=8,
                   T=0.0, dtype="f32", planted="fixed8"),
    # brute-force variant of configs[0] (V<=16, L<=4)
    "brute": Config("brute", 0, batch=1, V=16, L=4, d=64, g=32, r=32, M=16, B=8, k=16,
                    T=0.0, dtype="f32", planted="fixed8"),
    # BASELINE.json configs[1]
    "qwen4b": Config("qwen4b", 1, batch=1, V=QWEN_V, L=16, d=2560, g=1024, r=256, M=64,
                     B=16, k=8, T=0.0, dtype="bf16"),
    # BASELINE.json configs[2]
    "qwen8b": Config("qwen8b", 2, batch=1, V=QWEN_V, L=16, d=4096, g=1024, r=256, M=64,
                     B=16, k=8, T=0.0, dtype="bf16"),
    # BASELINE.json configs[3] (B and M are swept by the caller)
    "sweep8b": Config("sweep8b", 3, batch=1, V=QWEN_V, L=16, d=4096, g=1024, r=256, M=64,
                      B=16, k=8, T=0.0, dtype="bf16"),
    # BASELINE.json configs[4]
    "concurrent8b": Config("concurrent8b", 4, batch=32, V=QWEN_V, L=16, d=4096, g=1024,
                           r=256, M=64, B=32, k=8, T=0.6, dtype="bf16"),
}


def _gen(seed: int) -> torch.Generator:
    g = torch.Generator(device="cpu")
    g.manual_seed(int(seed))
    return g


def _normal(shape, std: float, gen: torch.Generator, dtype, chunk_rows: int = 8192) -> torch.Tensor:
    """N(0, std) drawn in fp32 on the CPU, rounded once to `dtype` (chunked over rows)."""
    out = torch.empty(shape, dtype=dtype)
    if len(shape) == 1:
        out.copy_(torch.randn(shape, generator=gen, dtype=torch.float32).mul_(std))
        return out
    rows = shape[0]
    for r0 in range(0, rows, chunk_rows):
        r1 = min(rows, r0 + chunk_rows)
        blk = torch.randn((r1 - r0,) + tuple(shape[1:]), generator=gen, dtype=torch.float32)
        out[r0:r1].copy_(blk.mul_(std))
    return out


def make_weights(cfg: Config, seed: int | None = None) -> Dict[str, torch.Tensor]:
    """Frozen drafter weights: E, W_ih, W_hh, W1, W2 as CPU tensors."""
    gen = _gen((cfg.seed if seed is None else seed) * 7 + 1)
    dt = cfg.torch_dtype
    V, d, g, r = cfg.V, cfg.d, cfg.g, cfg.r
    w = {
        "embed": _normal((V, d), cfg.embed_std, gen, dt),
        "gru_w_ih": _normal((3 * g, d), 1.0 / math.sqrt(d), gen, dt),
        "gru_w_hh": _normal((3 * g, g), 1.0 / math.sqrt(g), gen, dt),
        "corr_w1": _normal((r, d + g), 1.0 / math.sqrt(d + g), gen, dt),
        "corr_w2": _normal((V, r), 1.0 / math.sqrt(r), gen, dt),
    }
    return w


def make_inputs(cfg: Config, batch: int | None = None, seed: int | None = None,
                regime: str | None = None) -> Dict[str, torch.Tensor]:
    """Per-round inputs: marginal logits, backbone hidden states, root tokens/positions.

    Request b uses seed  cfg.seed + b  (independent requests)."""
    batch = cfg.batch if batch is None else batch
    regime = cfg.regime if regime is None else regime
    base_seed = cfg.seed if seed is None else seed
    dt = cfg.torch_dtype
    V, L, d = cfg.V, cfg.L, cfg.d
    logits = torch.empty((batch, L, V), dtype=dt)
    hidden = torch.empty((batch, L, d), dtype=dt)
    roots = torch.empty((batch,), dtype=torch.int32)
    rpos = torch.empty((batch,), dtype=torch.int32)
    planted = torch.empty((batch, L), dtype=torch.int64)
    for b in range(batch):
        gen = _gen((base_seed + b) * 7 + 3)
        x = torch.randn((L, V), generator=gen, dtype=torch.float32).mul_(3.0)
        tok = torch.randint(0, V, (L,), generator=gen)
        if cfg.planted == "fixed8":
            h = torch.full((L,), 8.0)
        else:
            u = torch.rand((L,), generator=gen, dtype=torch.float64).clamp_(1e-12, 1 - 1e-12)
            gum = -torch.log(-torch.log(u))
            h = (6.0 + 1.5 * gum).clamp_(4.0, 10.0).to(torch.float32)
        rows = torch.arange(L)
        if regime == "flat":
            x[rows, tok] += h
        elif regime == "peaked":
            x[rows, tok] = x.max(dim=1).values + h
        else:
            raise ValueError(f"unknown regime {regime!r}")
        logits[b].copy_(x)
        hidden[b].copy_(torch.randn((L, d), generator=gen, dtype=torch.float32))
        roots[b] = int(torch.randint(0, V, (1,), generator=gen))
        rpos[b] = int(torch.randint(0, 4096, (1,), generator=gen))
        planted[b] = tok
    return {"logits": logits, "hidden": hidden, "root_tokens": roots,
            "root_positions": rpos, "planted": planted}


def adversarial_select_rows(V: int, dtype, seed: int = MASTER_SEED) -> Dict[str, torch.Tensor]:
    """Rows that stress the select's tie rule and threshold logic (SURVEY.md 8(d) extras)."""
    gen = _gen(seed * 7 + 5)
    rows = {}
    rows["all_equal"] = torch.full((V,), 1.5)
    rows["ascending"] = torch.linspace(-20.0, 20.0, V)
    rows["descending"] = torch.linspace(20.0, -20.0, V)
    coarse = torch.randint(-3, 4, (V,), generator=gen).to(torch.float32)   # 7 distinct values
    rows["many_ties"] = coarse
    x = torch.randn((V,), generator=gen).mul_(3.0)
    x[torch.randint(0, V, (max(1, V // 7),), generator=gen)] = float("-inf")
    rows["neg_inf"] = x
    z = torch.randn((V,), generator=gen)
    z[::3] = 0.0
    z[1::3] = -0.0
    rows["signed_zeros"] = z
    rows["all_neg_inf_but_few"] = torch.full((V,), float("-inf"))
    rows["all_neg_inf_but_few"][torch.randint(0, V, (5,), generator=gen)] = 1.0
    return {k: v.to(dtype) for k, v in rows.items()}
