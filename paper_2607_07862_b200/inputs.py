"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2607_07862_b200.binding`).  It holds none of the method's
arithmetic: it draws random numbers (numpy Philox, a counter-based generator
keyed by (seed, matrix id)), scales them as the config says, and hands them to
torch's own fp32->bf16 cast (a library routine) so that both sides receive the
*same bf16 bit patterns*.  It imports neither the oracle nor the binding.

Recipe (SURVEY.md section 8c readings c4, c7, c9):
  * the paper's workload is random dense matrices of a stated shape, no dataset
    (PAPER.md:139); the Llama-3 names in BASELINE.json are
    dimension triples only.
  * weights W_l are stored [N_l x K_l], K contiguous (the nn.Linear.weight
    layout); fan_in(W_l) = K_l, its contraction length.
  * "normal":  W ~ N(0, 1/fan_in); X ~ N(0, 1)       (x_scale="unit", default)
                                   X ~ N(0, 1/K)     (x_scale="fan_in", literal reading)
  * "uniform": W ~ U[-1,1]/sqrt(fan_in); X ~ U[-1,1] (or /sqrt(K))
  * "exact":   X, W i.i.d. integers uniform in {-2,-1,0,1,2}
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Sequence

import numpy as np
import torch

ACT_NONE, ACT_RELU, ACT_GELU_TANH = 0, 1, 2


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: a chain of `len(widths)-1` GEMMs on M tokens."""

    name: str
    M: int
    widths: Sequence[int]          # K -> N1 -> N2 [-> ...]
    act: int
    dist: str                      # "normal" | "uniform" | "exact"
    seed: int
    note: str = ""

    @property
    def n_layers(self) -> int:
        return len(self.widths) - 1

    @property
    def flops(self) -> int:
        return sum(2 * self.M * self.widths[i] * self.widths[i + 1] for i in range(self.n_layers))

    @property
    def algorithmic_bytes(self) -> int:
        """every weight once, X once, each hidden
        activation written once and read once, Y once (all bf16)."""
        w = sum(self.widths[i] * self.widths[i + 1] for i in range(self.n_layers))
        x = self.M * self.widths[0]
        h = sum(2 * self.M * self.widths[i] for i in range(1, self.n_layers))
        y = self.M * self.widths[-1]
        return 2 * (w + x + h + y)


# BASELINE.json:configs[0..4] (0-based).
CONFIGS: List[Config] = [
    Config("cfg0_tiny", 64, (512, 2048, 512), ACT_RELU, "uniform", 0,
           "tiny 2-layer GEMM; also run with dist='exact'"),
    Config("cfg1_8b_decode", 16, (4096, 14336, 4096), ACT_GELU_TANH, "normal", 1,
           "Llama-3-8B-shaped MLP, M=16 (weight-bandwidth-bound)"),
    Config("cfg2_8b_prefill", 256, (4096, 14336, 4096), ACT_GELU_TANH, "normal", 2,
           "Llama-3-8B-shaped MLP, M=256"),
    Config("cfg3_70b", 128, (8192, 28672, 8192), ACT_GELU_TANH, "normal", 3,
           "Llama-3-70B-shaped MLP, M=128"),
    Config("cfg4_chain", 128, (4096, 14336, 4096, 14336, 4096), ACT_GELU_TANH, "normal", 4,
           "4-layer GEMM chain, GeLU after layers 1..3"),
]


def get_config(i: int, dist: str | None = None) -> Config:
    c = CONFIGS[i]
    if dist is not None and dist != c.dist:
        c = Config(c.name + "_" + dist, c.M, c.widths, c.act, dist, c.seed, c.note)
    return c


def _draw(seed: int, matrix_id: int, shape, dist: str, scale: float) -> torch.Tensor:
    """bf16 CPU tensor of `shape`, drawn from Philox keyed by (seed, matrix_id)."""
    gen = np.random.Generator(np.random.Philox(key=[int(seed), int(matrix_id)]))
    n = int(np.prod(shape))
    if dist == "normal":
        a = gen.standard_normal(n, dtype=np.float32)
    elif dist == "uniform":
        a = gen.random(n, dtype=np.float32)
        a *= 2.0
        a -= 1.0
    elif dist == "exact":
        a = gen.integers(-2, 3, size=n).astype(np.float32)
        scale = 1.0
    else:
        raise ValueError(f"unknown dist {dist!r}")
    if scale != 1.0:
        a *= np.float32(scale)
    return torch.from_numpy(a).reshape(*shape).to(torch.bfloat16)


def make_inputs(cfg: Config, x_scale: str = "unit", M: int | None = None):
    """Return (X, [W_1..W_L]) as bf16 CPU tensors.

    X is [M x K]; W_l is [N_l x K_l] (K contiguous).  `M` overrides cfg.M
    (used to draw a bounded row sample of a workload; row m of X does not
    depend on M because rows are drawn in order from one stream).
    """
    M = cfg.M if M is None else M
    K = cfg.widths[0]
    if x_scale == "unit":
        xs = 1.0
    elif x_scale == "fan_in":
        xs = 1.0 / float(np.sqrt(K))
    else:
        raise ValueError(x_scale)
    X = _draw(cfg.seed, 0, (M, K), cfg.dist, xs)
    Ws = []
    for l in range(cfg.n_layers):
        k, n = cfg.widths[l], cfg.widths[l + 1]
        Ws.append(_draw(cfg.seed, 1 + l, (n, k), cfg.dist, 1.0 / float(np.sqrt(k))))
    return X, Ws


def as_u16(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> numpy uint16 bit patterns (what the oracle consumes)."""
    assert t.dtype == torch.bfloat16
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def from_u16(a: np.ndarray) -> torch.Tensor:
    """numpy uint16 bit patterns -> bf16 tensor."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).view(torch.bfloat16)
